// fstat_api.cu -- the C ABI declared in include/fstat.h: plan management, argument validation,
// segmentation of the frequency band into CTA work items, workspace, launches.  Host code only; the arithmetic
// of the hot path lives in the kernels (fstat_fast.cu, fstat_fastband.cu, fstat_kernels.cu, fstat_band.cu,
// fstat_pso.cu).  There is no CPU fallback.
#include "../../include/fstat.h"
#include "fstat_internal.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <string>
#include <vector>

using namespace fstat;

// Segment tables of one segment length (they depend on the partitions, the options and the segment length only):
// kept per plan in a small cache, so that batches of different sizes -- a ragged last batch, swarms that shrink --
// neither rebuild nor re-upload anything, and no evaluation has to wait for the device.
struct SegTables {
    int64_t seg_len = 0;
    int32_t n_seg = 0;
    int32_t *d_seg_edge = nullptr, *d_part_seg = nullptr, *d_seg_gbase = nullptr;
    SegCrit *d_seg_crit = nullptr;
    int8_t *d_seg_maxlvl = nullptr;
    std::vector<int32_t> seg_edge_h;
    std::vector<int32_t> part_seg_h;
};

struct fstat_plan {
    int device = 0;
    int n_sm = 0;
    int64_t n_bins = 0;
    double df = 0.0;
    fstat_options opt{};
    int32_t n_part = 0;
    std::vector<int64_t> edges;        // host copy [n_part+1]
    double f0 = 0.0;                   // freq[0]
    double *d_dwp = nullptr;           // [n_bins][2]       folded data (interpolating kernel)
    double *d_fw = nullptr;            // [n_bins][2]       (f, w' = 4 df f^(-7/3) |K_f|^2 / S_n): full-model kernels, Gram builders
    double *d_node = nullptr;          // [n_node_rows][kTabW]
    int64_t n_node_rows = 0;
    bool fast_ok = false;              // the node grid (2 kMaxStride bins below, 3 above the band) stays at f > 0
    int32_t min_level = 0;             // smallest stride level with per-sub-block tables (options.min_stride_level)
    // partition-dependent tables of the interpolating kernel
    int32_t *d_edges32 = nullptr; size_t edges32_cap = 0;
    int32_t *d_cnt = nullptr; size_t cnt_cap = 0;          // scratch [n_part]
    double *d_gram[kNLevels] = {}; size_t gram_cap[kNLevels] = {};
    std::vector<int32_t> cnt[kNLevels];                    // host copies (segment -> first sub-block)
    // segmentation (depends on the partitions and on the number of particle groups)
    int32_t seg_groups = -1;           // n_groups the current segmentation was made for
    int32_t n_seg = 0;
    int32_t seg_len = 0;               // bins per work segment of the current segmentation (aligned cuts)
    std::vector<SegTables> seg_cache;  // one entry per segment length seen since the partitions were set (<= 8)
    // the entry in use (aliases into seg_cache):
    int32_t *d_seg_edge = nullptr;     // [n_seg+1]
    int32_t *d_part_seg = nullptr;     // [n_part+1]
    std::vector<int32_t> seg_edge_h;   // host copy of d_seg_edge
    std::vector<int32_t> part_seg_h;   // host copy of d_part_seg
    int32_t *d_seg_gbase = nullptr;    // [n_seg][kNLevels]
    SegCrit *d_seg_crit = nullptr;     // [n_seg]
    int8_t *d_seg_maxlvl = nullptr;    // [n_seg]
    int8_t *d_level = nullptr; size_t level_cap = 0;       // [n_groups][n_seg] of the most recent evaluation
    int32_t *d_direct = nullptr; size_t direct_cap = 0;    // [1 + n_groups * n_seg]: count, then the work list
    int64_t n_launches = 0;                                 // kernels launched by evaluations so far
    double *d_fpart = nullptr; size_t fpart_cap = 0;       // [n_chunk][P_pad] per-chunk sums of F_k (epilogue)
    int32_t last_groups = 0;
    // workspace
    double *d_coef = nullptr;  size_t coef_cap = 0;      // doubles
    int32_t *d_valid = nullptr; size_t valid_cap = 0;    // ints
    int32_t *d_slot = nullptr; size_t slot_cap = 0;      // [P] particle -> slot (sorted by chirp mass)
    unsigned char *d_sort = nullptr; size_t sort_cap = 0; // scratch of the slot ranking (keys, radix sort buffers)
    int32_t *d_perm = nullptr; size_t perm_cap = 0;      // [P_pad] slot -> particle (-1: padding)
    double *d_partial = nullptr; size_t partial_cap = 0; // doubles
    // row f2 (fstat_eval_batch_bands)
    fstat_plan *bandplan = nullptr;     // internal plan whose one partition is the whole grid (work segments only); shares the tables
    bool shares_tables = false;         // d_dwp, d_fw, d_node belong to the parent plan
    double *d_pgram[kNLevels] = {};     // prefix Gram matrices [ceil(n_bins / 8)][kNGram] per stride level (first band call)
    bool pgram_built = false;
    int32_t *d_band = nullptr; size_t band_cap = 0;       // [2][P_pad] k_lo, k_hi per slot
    double *d_rec = nullptr; size_t rec_cap = 0;          // [n_seg][2][kNPartial][P_pad] head / tail fragments of the work segments
    uint32_t *d_err = nullptr;                            // device flag raised by an internal invariant, then [4] 64-bit work counters
    double *d_band_fk = nullptr; size_t band_fk_cap = 0;  // [P][n_seg] when the caller passes Fk = NULL
    int64_t *d_band_out = nullptr; size_t band_out_cap = 0; // [P][2] (host-buffer call)
    bool last_was_band = false;         // fstat_plan_level_bins reports the band plan's stride mix
    // host-buffer path
    double *d_params = nullptr, *d_F = nullptr, *d_Fk = nullptr;
    size_t params_cap = 0, F_cap = 0, Fk_cap = 0;
    // fstat_eval_batch_host: the interpolating kernel is launched as up to kPipe ranges of partitions on streams of
    // its own, so that the epilogue and the device-to-host copy of one range's F_k run under the next ranges' kernels
    static constexpr int kPipe = 8;
    int32_t pipe_ranges = 1;
    cudaStream_t pipe_main[kPipe] = {}, pipe_copy = nullptr;
    cudaEvent_t pipe_fork = nullptr, pipe_main_done[kPipe] = {}, pipe_copy_done = nullptr;
    OrbitCoef orb{};
    // ring of event pairs around the main kernel of the most recent evaluations (bench roofline)
    static constexpr int kRing = 128;
    cudaEvent_t ev0[kRing] = {}, ev1[kRing] = {};
    int64_t n_timed = 0;
    std::string err;
};

static thread_local std::string g_create_err;

static fstat_status fail(fstat_plan *pl, fstat_status s, const std::string &msg)
{
    if (pl) pl->err = msg; else g_create_err = msg;
    return s;
}

#define CU_TRY(pl, call)                                                                             \
    do {                                                                                             \
        cudaError_t e__ = (call);                                                                    \
        if (e__ != cudaSuccess) {                                                                    \
            const bool oom__ = (e__ == cudaErrorMemoryAllocation);                                   \
            cudaGetLastError();                                                                      \
            return fail(pl, oom__ ? FSTAT_ENOMEM : FSTAT_ECUDA,                                      \
                        std::string(#call) + ": " + cudaGetErrorString(e__));                        \
        }                                                                                            \
    } while (0)

namespace {

struct DeviceGuard {
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev) { ok = (cudaGetDevice(&prev) == cudaSuccess) && (cudaSetDevice(dev) == cudaSuccess); }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <class T>
cudaError_t grow(T **ptr, size_t *cap, size_t need)
{
    if (need <= *cap) return cudaSuccess;
    if (*ptr) { cudaFree(*ptr); *ptr = nullptr; *cap = 0; }
    cudaError_t e = cudaMalloc((void **)ptr, need * sizeof(T));
    if (e == cudaSuccess) *cap = need;
    return e;
}

bool edges_valid(int64_t n_bins, int32_t n_part, const int64_t *e, std::string *why)
{
    if (n_part < 1) { *why = "n_part < 1"; return false; }
    if (!e) { *why = "part_edges is NULL"; return false; }
    if (e[0] != 0) { *why = "part_edges[0] != 0"; return false; }
    if (e[n_part] != n_bins) { *why = "part_edges[n_part] != n_bins"; return false; }
    for (int32_t k = 0; k < n_part; ++k)
        if (!(e[k + 1] > e[k])) { *why = "part_edges not strictly increasing (empty partition)"; return false; }
    return true;
}

// Cut every partition into CTA work items ("segments").  A segment never crosses a partition edge, so
// the main kernels need no per-bin edge test and write plain partial sums.
//   aligned: the cuts inside a partition are the multiples of max_len (itself a multiple of kMaxStride),
//            so that node intervals of every stride and the 512-bin data tiles never straddle a segment
//            boundary other than a partition edge -- the layout the interpolating kernel needs;
//   else:    near-equal pieces of at most max_len bins (tuning / tests; direct kernel only).
void make_segments(const std::vector<int64_t> &edges, int64_t max_len, bool aligned,
                   std::vector<int32_t> *seg_edge, std::vector<int32_t> *part_seg)
{
    const size_t n_part = edges.size() - 1;
    seg_edge->clear();
    part_seg->assign(n_part + 1, 0);
    seg_edge->push_back(0);
    for (size_t k = 0; k < n_part; ++k) {
        const int64_t lo = edges[k], hi = edges[k + 1], len = hi - lo;
        (*part_seg)[k] = (int32_t)(seg_edge->size() - 1);
        if (aligned) {
            for (int64_t c = (lo / max_len + 1) * max_len; c < hi; c += max_len) seg_edge->push_back((int32_t)c);
            seg_edge->push_back((int32_t)hi);
        } else {
            const int64_t n = (len + max_len - 1) / max_len;
            for (int64_t s = 1; s <= n; ++s) seg_edge->push_back((int32_t)(lo + (len * s) / n));
        }
    }
    (*part_seg)[n_part] = (int32_t)(seg_edge->size() - 1);
}

// The band plan (row f2) always cuts at the multiples of its segment length: its stitch kernel finds the work segment
// of a bin by division.  Elsewhere a segment length that is not a multiple of 512 means near-equal pieces (tests).
bool segments_aligned(const fstat_plan *pl)
{
    return pl->shares_tables || pl->opt.max_segment_bins <= 0 || pl->opt.max_segment_bins % kMaxStride == 0;
}

// the interpolating kernel needs segments that start at multiples of 512 bins
bool segments_fast_capable(int64_t seg_len)
{
    return seg_len % kMaxStride == 0;
}

int64_t auto_segment_len(const fstat_plan *pl, int32_t n_groups)
{
    if (pl->opt.max_segment_bins > 0) return pl->opt.max_segment_bins;
    // Short grids (config 0: 2096 bins): with segments of >= 2048 bins a handful of CTAs would walk the whole band one bin
    // after the other.  Below 4096 bins the work items are single 64-bin tiles instead; such segments are not multiples
    // of 512 bins, so these items all go to the direct kernel (on so short a grid the interpolating kernel would pay its
    // five start-up nodes per partition anyway).
    if (pl->n_bins < 2 * 4 * kMaxStride) return kTileBins;
    // aim at >= 48 work items per SM so that the tail wave is short; multiples of kMaxStride
    const int64_t target_ctas = (int64_t)pl->n_sm * 48;
    int64_t want_seg = (target_ctas + n_groups - 1) / n_groups;
    if (want_seg < 1) want_seg = 1;
    int64_t len = (pl->n_bins + want_seg - 1) / want_seg;
    len = ((len + kMaxStride - 1) / kMaxStride) * kMaxStride;
    if (len < 4 * kMaxStride) len = 4 * kMaxStride;
    if (len > 64 * kMaxStride) len = 64 * kMaxStride;
    return len;
}

// short segments (narrow partitions): one CTA of the interpolating kernel walks ~4096 bins' worth of consecutive
// segments, so that the five start-up node evaluations are shared
int32_t segs_per_cta(int64_t n_bins, int64_t n_seg)
{
    const int64_t avg = n_bins / (n_seg > 0 ? n_seg : 1);
    const int64_t g = avg > 0 ? (4096 + avg / 2) / avg : 1;
    return (int32_t)(g < 1 ? 1 : (g > 8 ? 8 : g));
}

int64_t n_segments_for(const fstat_plan *pl, int32_t n_groups)
{
    std::vector<int32_t> seg_edge, part_seg;
    make_segments(pl->edges, auto_segment_len(pl, n_groups), segments_aligned(pl), &seg_edge, &part_seg);
    return (int64_t)seg_edge.size() - 1;
}

// Per-segment factors of the a-priori interpolation error bound (see schedule_kernel; DESIGN.md
// "Stride selection").  Psi_q = Psi in quarter turns = ... + c3 f^(-5/3) + c9 f^(-34/9); t_f = Psi_q'/4.
SegCrit make_seg_crit(double f_lo, double f_hi, double df, double part_len)
{
    const double Om = 2.0 * kPi / kYear;
    SegCrit q;
    q.p1 = 1.15 * Om * df * 0.25 * (40.0 / 9.0) * pow(f_lo, -11.0 / 3.0);
    q.p2 = 1.15 * Om * df * 0.25 * (1462.0 / 81.0) * pow(f_lo, -52.0 / 9.0);
    const double df4 = df * df * df * df;
    q.q1 = (3.0 / 128.0) * (6160.0 / 81.0) * pow(f_lo, -17.0 / 3.0) * df4;
    q.q2 = (3.0 / 128.0) * (4637464.0 / 6561.0) * pow(f_lo, -70.0 / 9.0) * df4;
    q.ad = (3.0 / 128.0) * 4.0 * f_hi * 1.01 * kAU / kC;
    q.r1 = (440.0 / 27.0) * pow(f_lo, -14.0 / 3.0) * df * df * df;
    q.r2 = (76024.0 / 729.0) * pow(f_lo, -61.0 / 9.0) * df * df * df;
    const double r = f_hi / 0.01;
    q.ct = 0.15 * (r > 1.0 ? r * r : 1.0);
    q.kl = 0.05 * part_len;
    q.d2 = 1.3 * 4.0 * df / Om;                        // d^2 Psi_q / dk^2 = 4 df dt_f/dk, dt_f/dk = omega / Omega
    return q;
}

void free_seg_tables(SegTables &t)
{
    cudaFree(t.d_seg_edge); cudaFree(t.d_part_seg); cudaFree(t.d_seg_gbase); cudaFree(t.d_seg_crit); cudaFree(t.d_seg_maxlvl);
    t = SegTables();
}

// Drop every cached segmentation (the partitions or the segment-length option changed).  Earlier evaluations may still
// read the tables: wait for the device first.
void invalidate_segments(fstat_plan *pl)
{
    if (!pl->seg_cache.empty()) cudaDeviceSynchronize();
    for (SegTables &t : pl->seg_cache) free_seg_tables(t);
    pl->seg_cache.clear();
    pl->seg_groups = -1;
    pl->d_seg_edge = pl->d_part_seg = pl->d_seg_gbase = nullptr;
    pl->d_seg_crit = nullptr;
    pl->d_seg_maxlvl = nullptr;
}

void use_seg_tables(fstat_plan *pl, const SegTables &t, int32_t n_groups)
{
    pl->d_seg_edge = t.d_seg_edge; pl->d_part_seg = t.d_part_seg; pl->d_seg_gbase = t.d_seg_gbase;
    pl->d_seg_crit = t.d_seg_crit; pl->d_seg_maxlvl = t.d_seg_maxlvl;
    pl->seg_edge_h = t.seg_edge_h;
    pl->part_seg_h = t.part_seg_h;
    pl->n_seg = t.n_seg;
    pl->seg_len = (int32_t)(t.seg_len < pl->n_bins ? t.seg_len : pl->n_bins);
    pl->seg_groups = n_groups;
}

fstat_status ensure_segments(fstat_plan *pl, int32_t n_groups)
{
    if (pl->seg_groups == n_groups) return FSTAT_OK;
    const int64_t seg_len = auto_segment_len(pl, n_groups);
    for (const SegTables &t : pl->seg_cache)
        if (t.seg_len == seg_len) { use_seg_tables(pl, t, n_groups); return FSTAT_OK; }
    std::vector<int32_t> seg_edge, part_seg;
    const bool aligned = segments_aligned(pl);
    make_segments(pl->edges, seg_len, aligned, &seg_edge, &part_seg);
    const size_t n_seg = seg_edge.size() - 1;
    std::vector<int32_t> gbase(n_seg * kNLevels);
    std::vector<SegCrit> crit(n_seg);
    std::vector<int8_t> maxlvl(n_seg);
    for (size_t k = 0; k + 1 < part_seg.size(); ++k)
        for (int32_t sgi = part_seg[k]; sgi < part_seg[k + 1]; ++sgi) {
            const int64_t lo = seg_edge[sgi], hi = seg_edge[sgi + 1];
            for (int l = 0; l < kNLevels; ++l) {
                const int sh = kLevel0Shift + l;
                const int64_t first = (lo >> sh) + pl->cnt[l][k];
                const int64_t last = first + (((hi - 1) >> sh) - (lo >> sh));           // sub-blocks the item walks
                const int64_t n_sub = ((pl->n_bins + ((int64_t)1 << sh) - 1) >> sh) + pl->cnt[l][pl->n_part - 1];
                if (first < 0 || last >= n_sub)
                    return fail(pl, FSTAT_ECUDA, "internal: Gram table index out of range");
                gbase[(size_t)sgi * kNLevels + l] = (int32_t)first;
            }
            crit[sgi] = make_seg_crit(pl->f0 + (double)lo * pl->df, pl->f0 + (double)hi * pl->df, pl->df,
                                      (double)(pl->edges[k + 1] - pl->edges[k]));
            maxlvl[sgi] = (int8_t)((pl->fast_ok && aligned && segments_fast_capable(seg_len) && hi - lo >= 8) ? kNLevels - 1 : -1);
        }
    if (pl->seg_cache.size() >= 8) {                       // (a ninth segment length: start over)
        const int32_t keep = pl->seg_groups;
        invalidate_segments(pl);
        (void)keep;
    }
    // fresh arrays: no kernel in flight reads them, so the blocking copies below order nothing but themselves
    SegTables t;
    t.seg_len = seg_len;
    t.n_seg = (int32_t)n_seg;
    cudaError_t e = cudaMalloc((void **)&t.d_seg_edge, seg_edge.size() * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc((void **)&t.d_part_seg, part_seg.size() * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc((void **)&t.d_seg_gbase, gbase.size() * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc((void **)&t.d_seg_crit, crit.size() * sizeof(SegCrit));
    if (e == cudaSuccess) e = cudaMalloc((void **)&t.d_seg_maxlvl, maxlvl.size() * sizeof(int8_t));
    if (e == cudaSuccess) e = cudaMemcpy(t.d_seg_edge, seg_edge.data(), seg_edge.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t.d_part_seg, part_seg.data(), part_seg.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t.d_seg_gbase, gbase.data(), gbase.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t.d_seg_crit, crit.data(), crit.size() * sizeof(SegCrit), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t.d_seg_maxlvl, maxlvl.data(), maxlvl.size() * sizeof(int8_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { free_seg_tables(t); CU_TRY(pl, e); }
    t.seg_edge_h = seg_edge;
    t.part_seg_h = part_seg;
    pl->seg_cache.push_back(t);
    use_seg_tables(pl, pl->seg_cache.back(), n_groups);
    return FSTAT_OK;
}

// Gram matrices of every stride level for the plan's current partitions (plan create / set_partitions).
fstat_status build_gram_tables(fstat_plan *pl)
{
    const int32_t n_part = pl->n_part;
    std::vector<int32_t> e32(n_part + 1);
    for (int32_t k = 0; k <= n_part; ++k) e32[k] = (int32_t)pl->edges[k];
    CU_TRY(pl, cudaDeviceSynchronize());       // earlier evaluations may still read the old tables
    CU_TRY(pl, grow(&pl->d_edges32, &pl->edges32_cap, e32.size()));
    CU_TRY(pl, grow(&pl->d_cnt, &pl->cnt_cap, (size_t)n_part));
    CU_TRY(pl, cudaMemcpy(pl->d_edges32, e32.data(), e32.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    for (int l = 0; l < kNLevels; ++l) {
        const int64_t S = (int64_t)kMinStride << l;
        std::vector<int32_t> &cnt = pl->cnt[l];
        cnt.assign(n_part, 0);
        for (int32_t k = 1; k < n_part; ++k) cnt[k] = cnt[k - 1] + ((pl->edges[k] % S) != 0 ? 1 : 0);
        if (!pl->fast_ok || l < pl->min_level) continue;   // (no work item is given a level below min_level)
        const int64_t n_sub = (pl->n_bins + S - 1) / S + cnt[n_part - 1];
        CU_TRY(pl, grow(&pl->d_gram[l], &pl->gram_cap[l], (size_t)n_sub * kNW));
        CU_TRY(pl, cudaMemcpy(pl->d_cnt, cnt.data(), (size_t)n_part * sizeof(int32_t), cudaMemcpyHostToDevice));
        CU_TRY(pl, launch_build_gram(pl->d_fw, pl->d_edges32, n_part, pl->n_bins, l, pl->d_cnt, pl->d_gram[l], 0));
        CU_TRY(pl, cudaDeviceSynchronize());   // d_cnt is reused by the next level
    }
    return FSTAT_OK;
}

}  // namespace

// The orbit of PAPER.md:198 (analytic, second order in the eccentricity e = L / (2 sqrt(3) AU); formulas
// of DESIGN.md reading A9) written as trigonometric polynomials in alpha = 2 pi t / yr + kappa.
void fstat::make_orbit_coef(double L, double lambda_in, int32_t tdi_channel, OrbitCoef *out)
{
    // Y, Z: the Michelson combination centred on spacecraft 2, 3 = X of the constellation relabelled cyclically
    const double lambda = lambda_in + ((tdi_channel == 1 || tdi_channel == 2) ? 2.0 * kPi * tdi_channel / 3.0 : 0.0);
    const long double R = kAU, pi = 3.14159265358979323846264338327950288L;
    const long double e = (long double)L / (2.0L * sqrtl(3.0L) * R);
    long double Pn[3][3][7];
    for (int n = 0; n < 3; ++n) {
        const long double be = 2.0L * pi * n / 3.0L + (long double)lambda;
        const long double cb = cosl(be), sb = sinl(be), c2b = cosl(2 * be), s2b = sinl(2 * be);
        long double(*C)[7] = Pn[n];
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 7; ++j) C[i][j] = 0.0L;
        // x
        C[0][0] = -1.5L * e * R * cb;
        C[0][1] = R - 1.25L * e * e * R - 0.625L * e * e * R * c2b;
        C[0][2] = -0.625L * e * e * R * s2b;
        C[0][3] = 0.5L * e * R * cb;
        C[0][4] = 0.5L * e * R * sb;
        C[0][5] = 0.375L * e * e * R * c2b;
        C[0][6] = 0.375L * e * e * R * s2b;
        // y
        C[1][0] = -1.5L * e * R * sb;
        C[1][1] = -0.625L * e * e * R * s2b;
        C[1][2] = R - 1.25L * e * e * R + 0.625L * e * e * R * c2b;
        C[1][3] = -0.5L * e * R * sb;
        C[1][4] = 0.5L * e * R * cb;
        C[1][5] = -0.375L * e * e * R * s2b;
        C[1][6] = 0.375L * e * e * R * c2b;
        // z = -sqrt3 e R cos(a - b) + sqrt3 e^2 R (3/2 - cos(2a - 2b)/2)
        const long double s3 = sqrtl(3.0L);
        C[2][0] = 1.5L * s3 * e * e * R;
        C[2][1] = -s3 * e * R * cb;
        C[2][2] = -s3 * e * R * sb;
        C[2][3] = -0.5L * s3 * e * e * R * c2b;
        C[2][4] = -0.5L * s3 * e * e * R * s2b;
    }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 7; ++j) {
            out->c[0][i][j] = (double)(4.0L * Pn[0][i][j] / (long double)kC);
            out->c[1][i][j] = (double)((Pn[1][i][j] - Pn[0][i][j]) / (long double)L);
            out->c[2][i][j] = (double)((Pn[2][i][j] - Pn[0][i][j]) / (long double)L);
        }
    // A = (Z - X)/sqrt 2, E = (X - 2Y + Z)/sqrt 6, T = (X + Y + Z)/sqrt 3   (reading A28)
    const double r2 = sqrt(0.5), r6 = sqrt(1.0 / 6.0), r3 = sqrt(1.0 / 3.0);
    const double W[3][3] = {{-r2, 0.0, r2}, {r6, -2.0 * r6, r6}, {r3, r3, r3}};
    for (int i = 0; i < 3; ++i) out->wch[i] = (tdi_channel >= 3 && tdi_channel <= 5) ? W[tdi_channel - 3][i] : 0.0;
}

extern "C" {

void fstat_default_options(fstat_options *o)
{
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->f_ref_e0 = 0.01;
    o->arm_length_m = 2.5e9;
    o->orbit_kappa = 0.0;
    o->orbit_lambda = 0.0;
    o->device = -1;
    o->inputs_on_device = 0;
    o->max_segment_bins = 0;
    o->force_level = -2;
    o->interp_tol = 1.0;
    o->tdi_channel = FSTAT_TDI_X;
    o->min_stride_level = -1;
}

const char *fstat_status_str(fstat_status s)
{
    switch (s) {
        case FSTAT_OK: return "FSTAT_OK";
        case FSTAT_EINVAL: return "FSTAT_EINVAL";
        case FSTAT_ENOMEM: return "FSTAT_ENOMEM";
        case FSTAT_ECUDA: return "FSTAT_ECUDA";
        case FSTAT_EUNSUPPORTED: return "FSTAT_EUNSUPPORTED";
    }
    return "FSTAT_?";
}

const char *fstat_last_error(const fstat_plan *pl) { return pl ? pl->err.c_str() : g_create_err.c_str(); }

fstat_status fstat_edges_equal_bins(int64_t n_bins, int32_t n_part, int64_t *edges_out)
{
    if (!edges_out || n_part < 1 || n_bins < 1 || (int64_t)n_part > n_bins) return FSTAT_EINVAL;
    for (int32_t j = 0; j <= n_part; ++j)
        edges_out[j] = (int64_t)(((__int128)j * (__int128)n_bins) / (__int128)n_part);
    return FSTAT_OK;
}

static fstat_status plan_create_impl(fstat_plan *pl, int64_t n_bins, const double *freq, const double *dw,
                                     const double *isn)
{
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaDeviceProp prop;
    CU_TRY(pl, cudaGetDeviceProperties(&prop, pl->device));
    pl->n_sm = prop.multiProcessorCount;
    if (prop.major < 10)
        return fail(pl, FSTAT_ECUDA, "device is not sm_100-class (this library ships sm_100a code only)");
    CU_TRY(pl, main_kernel_configure());
    CU_TRY(pl, fast_kernel_configure());
    CU_TRY(pl, fastmulti_kernel_configure());
    CU_TRY(pl, band_kernel_configure());
    CU_TRY(pl, fastband_kernel_configure());

    const double *d_freq = freq, *d_dw = dw, *d_isn = isn;
    double *tmp = nullptr;
    if (!pl->opt.inputs_on_device) {
        CU_TRY(pl, cudaMalloc((void **)&tmp, (size_t)n_bins * 4 * sizeof(double)));
        cudaError_t e = cudaMemcpy(tmp, freq, (size_t)n_bins * sizeof(double), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(tmp + n_bins, dw, (size_t)n_bins * 2 * sizeof(double), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(tmp + 3 * n_bins, isn, (size_t)n_bins * sizeof(double), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { cudaFree(tmp); CU_TRY(pl, e); }
        d_freq = tmp; d_dw = tmp + n_bins; d_isn = tmp + 3 * n_bins;
    }
    // df as the oracle-independent statement of the contract: (f[N-1] - f[0]) / (N - 1)
    double fe[2] = {0, 0};
    cudaError_t e = cudaMemcpy(&fe[0], d_freq, sizeof(double), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(&fe[1], d_freq + (n_bins - 1), sizeof(double), cudaMemcpyDeviceToHost);
    uint32_t *d_err = nullptr;
    if (e == cudaSuccess) e = cudaMalloc((void **)&d_err, sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMemset(d_err, 0, sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMalloc((void **)&pl->d_dwp, (size_t)n_bins * 2 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&pl->d_fw, (size_t)n_bins * 2 * sizeof(double));
    // node rows for bins -2 kMaxStride .. (floor((N-1)/kMaxStride) + 3) * kMaxStride in steps of kNodeStride
    pl->n_node_rows = kNodePad + (((n_bins - 1) / kMaxStride + 3) * kMaxStride) / kNodeStride + 1;
    if (e == cudaSuccess) e = cudaMalloc((void **)&pl->d_node, (size_t)pl->n_node_rows * kTabW * sizeof(double));
    uint32_t bits = 0;
    if (e == cudaSuccess) {
        pl->df = (n_bins > 1) ? (fe[1] - fe[0]) / (double)(n_bins - 1) : fe[0];
        if (!(pl->df > 0.0) || !isfinite(pl->df)) bits |= ERR_FREQ_ORDER;
        else {
            pl->f0 = fe[0];
            pl->fast_ok = (fe[0] - (double)(2 * kMaxStride + 1) * pl->df > 0.0) && n_bins > 1;
            e = launch_build_table(d_freq, d_dw, d_isn, n_bins, pl->df, pl->opt.arm_length_m, pl->d_dwp, pl->d_fw,
                                   d_err, 0);
            if (e == cudaSuccess)
                e = launch_build_nodes(d_freq, n_bins, pl->df, pl->opt.arm_length_m, pl->n_node_rows, pl->d_node, 0);
            if (e == cudaSuccess) e = cudaDeviceSynchronize();
            if (e == cudaSuccess) e = cudaMemcpy(&bits, d_err, sizeof(uint32_t), cudaMemcpyDeviceToHost);
        }
    }
    if (tmp) cudaFree(tmp);
    if (d_err) cudaFree(d_err);
    CU_TRY(pl, e);
    if (bits) {
        std::string why;
        if (bits & ERR_FREQ_NONPOS) why += "freq_hz has a non-positive or non-finite entry; ";
        if (bits & ERR_FREQ_ORDER) why += "freq_hz is not strictly ascending; ";
        if (bits & ERR_FREQ_UNIFORM) why += "freq_hz is not a uniform grid; ";
        if (bits & ERR_DW_NONFINITE) why += "dw_re_im has a non-finite entry; ";
        if (bits & ERR_ISN_NONFINITE) why += "inv_sn has a non-finite entry; ";
        if (bits & ERR_ISN_NONPOS) why += "inv_sn has an entry <= 0; ";
        return fail(pl, FSTAT_EINVAL, why);
    }
    make_orbit_coef(pl->opt.arm_length_m, pl->opt.orbit_lambda, pl->opt.tdi_channel, &pl->orb);
    {
        fstat_status gs = build_gram_tables(pl);
        if (gs != FSTAT_OK) return gs;
    }
    for (int i = 0; i < fstat_plan::kRing; ++i) {
        CU_TRY(pl, cudaEventCreate(&pl->ev0[i]));
        CU_TRY(pl, cudaEventCreate(&pl->ev1[i]));
    }
    return FSTAT_OK;
}

static void plan_free(fstat_plan *pl)
{
    if (!pl) return;
    DeviceGuard g(pl->device);
    if (pl->bandplan) { plan_free(pl->bandplan); pl->bandplan = nullptr; }
    if (pl->shares_tables) { pl->d_dwp = nullptr; pl->d_fw = nullptr; pl->d_node = nullptr; }
    for (SegTables &t : pl->seg_cache) free_seg_tables(t);
    cudaFree(pl->d_coef);
    cudaFree(pl->d_valid); cudaFree(pl->d_partial); cudaFree(pl->d_params); cudaFree(pl->d_F); cudaFree(pl->d_Fk);
    cudaFree(pl->d_dwp); cudaFree(pl->d_fw); cudaFree(pl->d_node); cudaFree(pl->d_edges32); cudaFree(pl->d_cnt);
    for (int l = 0; l < kNLevels; ++l) { cudaFree(pl->d_gram[l]); cudaFree(pl->d_pgram[l]); }
    cudaFree(pl->d_band); cudaFree(pl->d_rec); cudaFree(pl->d_err); cudaFree(pl->d_band_fk); cudaFree(pl->d_band_out);
    cudaFree(pl->d_level);
    cudaFree(pl->d_fpart); cudaFree(pl->d_direct); cudaFree(pl->d_slot); cudaFree(pl->d_perm); cudaFree(pl->d_sort);
    for (int i = 0; i < fstat_plan::kRing; ++i) {
        if (pl->ev0[i]) cudaEventDestroy(pl->ev0[i]);
        if (pl->ev1[i]) cudaEventDestroy(pl->ev1[i]);
    }
    for (int i = 0; i < fstat_plan::kPipe; ++i) {
        if (pl->pipe_main[i]) cudaStreamDestroy(pl->pipe_main[i]);
        if (pl->pipe_main_done[i]) cudaEventDestroy(pl->pipe_main_done[i]);
    }
    if (pl->pipe_copy) cudaStreamDestroy(pl->pipe_copy);
    if (pl->pipe_fork) cudaEventDestroy(pl->pipe_fork);
    if (pl->pipe_copy_done) cudaEventDestroy(pl->pipe_copy_done);
    delete pl;
}

fstat_status fstat_plan_create(fstat_plan **out, int64_t n_bins, const double *freq_hz, const double *dw_re_im,
                               const double *inv_sn, int32_t n_part, const int64_t *part_edges,
                               const fstat_options *opts)
{
    if (!out) return fail(nullptr, FSTAT_EINVAL, "out is NULL");
    *out = nullptr;
    if (n_bins < 1) return fail(nullptr, FSTAT_EINVAL, "n_bins < 1");
    if (n_bins >= (int64_t)1 << 31) return fail(nullptr, FSTAT_EUNSUPPORTED, "n_bins >= 2^31");
    if (!freq_hz || !dw_re_im || !inv_sn) return fail(nullptr, FSTAT_EINVAL, "freq_hz, dw_re_im or inv_sn is NULL");
    std::string why;
    if (!edges_valid(n_bins, n_part, part_edges, &why)) return fail(nullptr, FSTAT_EINVAL, why);
    fstat_options o;
    fstat_default_options(&o);
    if (opts) o = *opts;
    if (!(o.f_ref_e0 > 0.0) || !(o.arm_length_m > 0.0) || !isfinite(o.orbit_kappa) || !isfinite(o.orbit_lambda) ||
        o.max_segment_bins < 0 || o.force_level < -2 || o.force_level >= kNLevels || !(o.interp_tol > 0.0) ||
        !isfinite(o.interp_tol) || o.tdi_channel < FSTAT_TDI_X || o.tdi_channel > FSTAT_TDI_T ||
        o.min_stride_level < -1 || o.min_stride_level >= kNLevels)
        return fail(nullptr, FSTAT_EINVAL, "bad option value");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) {
        cudaGetLastError();
        return fail(nullptr, FSTAT_ECUDA, "no CUDA device available (there is no CPU fallback)");
    }
    int dev = o.device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return fail(nullptr, FSTAT_ECUDA, "cudaGetDevice failed");
    if (dev >= n_dev) return fail(nullptr, FSTAT_EINVAL, "device ordinal out of range");

    fstat_plan *pl = new (std::nothrow) fstat_plan;
    if (!pl) return fail(nullptr, FSTAT_ENOMEM, "host allocation failed");
    pl->device = dev;
    pl->n_bins = n_bins;
    pl->opt = o;
    // automatic: stride 32 and up, unless a smaller stride is forced (tests, tuning); never above a forced level
    pl->min_level = o.min_stride_level >= 0 ? o.min_stride_level : 2;
    if (o.force_level >= 0 && o.force_level < pl->min_level) pl->min_level = o.force_level;
    pl->n_part = n_part;
    try {
        pl->edges.assign(part_edges, part_edges + n_part + 1);
    } catch (...) {
        delete pl;
        return fail(nullptr, FSTAT_ENOMEM, "host allocation failed");
    }
    fstat_status s = plan_create_impl(pl, n_bins, freq_hz, dw_re_im, inv_sn);
    if (s != FSTAT_OK) {
        g_create_err = pl->err;
        plan_free(pl);
        return s;
    }
    *out = pl;
    return FSTAT_OK;
}

fstat_status fstat_plan_set_partitions(fstat_plan *pl, int32_t n_part, const int64_t *part_edges)
{
    if (!pl) return FSTAT_EINVAL;
    std::string why;
    if (!edges_valid(pl->n_bins, n_part, part_edges, &why)) return fail(pl, FSTAT_EINVAL, why);
    try {
        pl->edges.assign(part_edges, part_edges + n_part + 1);
    } catch (...) {
        return fail(pl, FSTAT_ENOMEM, "host allocation failed");
    }
    pl->n_part = n_part;
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    invalidate_segments(pl);    // re-segment on the next evaluation
    return build_gram_tables(pl);
}

void fstat_plan_destroy(fstat_plan *pl) { plan_free(pl); }

int64_t fstat_plan_n_bins(const fstat_plan *pl) { return pl ? pl->n_bins : 0; }
int32_t fstat_plan_n_part(const fstat_plan *pl) { return pl ? pl->n_part : 0; }
int32_t fstat_plan_device(const fstat_plan *pl) { return pl ? pl->device : -1; }
int64_t fstat_plan_launch_count(const fstat_plan *pl) { return pl ? pl->n_launches : 0; }

fstat_status fstat_plan_band_stats(fstat_plan *pl, int64_t *out)
{
    if (!pl || !out) return FSTAT_EINVAL;
    for (int i = 0; i < 5; ++i) out[i] = 0;
    if (!pl->d_err) return FSTAT_OK;
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    unsigned long long h[5];
    CU_TRY(pl, cudaDeviceSynchronize());
    CU_TRY(pl, cudaMemcpy(h, pl->d_err, sizeof h, cudaMemcpyDeviceToHost));
    for (int i = 0; i < 4; ++i) out[i] = (int64_t)h[i + 1];
    out[4] = (int64_t)(h[0] & 0xffffffffull);
    return FSTAT_OK;
}

int64_t fstat_plan_table_bytes(const fstat_plan *pl)
{
    if (!pl) return 0;
    int64_t b = (int64_t)pl->n_bins * 4 * (int64_t)sizeof(double)                 // folded data, (f, w')
                + pl->n_node_rows * kTabW * (int64_t)sizeof(double);             // node rows
    for (int l = 0; l < kNLevels; ++l) {
        b += (int64_t)pl->gram_cap[l] * (int64_t)sizeof(double);                 // Gram matrices of the partitions
        if (pl->d_pgram[l]) b += ((pl->n_bins + kMinStride - 1) / kMinStride) * kNGram * (int64_t)sizeof(double);
    }
    return b;
}

int64_t fstat_plan_n_ctas(const fstat_plan *pl, int64_t P)
{
    if (!pl || P < 1) return 0;
    const int64_t n_groups = (P + kThreads - 1) / kThreads;
    const int64_t n_seg = n_segments_for(pl, (int32_t)n_groups);
    const int64_t g = segs_per_cta(pl->n_bins, n_seg);
    return n_groups * ((n_seg + g - 1) / g);
}

fstat_status fstat_plan_level_bins(fstat_plan *pl, int64_t *bins_out, int64_t *subblocks_out)
{
    if (!pl || !bins_out || !subblocks_out) return FSTAT_EINVAL;
    for (int l = 0; l <= kNLevels; ++l) bins_out[l] = subblocks_out[l] = 0;
    if (pl->last_was_band && pl->bandplan) pl = pl->bandplan;      // the most recent evaluation was a row-f2 call
    if (pl->last_groups < 1 || pl->seg_groups != pl->last_groups) return FSTAT_OK;
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    const size_t n = (size_t)pl->n_seg * (size_t)pl->last_groups;
    std::vector<int8_t> lv(n);
    CU_TRY(pl, cudaDeviceSynchronize());
    CU_TRY(pl, cudaMemcpy(lv.data(), pl->d_level, n, cudaMemcpyDeviceToHost));
    for (int32_t gidx = 0; gidx < pl->last_groups; ++gidx)
        for (int32_t sgi = 0; sgi < pl->n_seg; ++sgi) {
            const int l = lv[(size_t)gidx * pl->n_seg + sgi];
            if (l < -1) continue;                           // (skipped work items exist only in row f2's internal plan)
            const int64_t lo = pl->seg_edge_h[sgi], hi = pl->seg_edge_h[sgi + 1];
            bins_out[l + 1] += hi - lo;
            if (l >= 0) subblocks_out[l + 1] += ((hi - 1) >> (kLevel0Shift + l)) - (lo >> (kLevel0Shift + l)) + 1;
        }
    return FSTAT_OK;
}

int32_t fstat_plan_main_kernel_ms(fstat_plan *pl, int32_t n_last, double *ms_out)
{
    if (!pl || !ms_out || n_last < 1) return 0;
    DeviceGuard g(pl->device);
    int64_t n = pl->n_timed < fstat_plan::kRing ? pl->n_timed : fstat_plan::kRing;
    if (n > n_last) n = n_last;
    int32_t w = 0;
    for (int64_t i = pl->n_timed - n; i < pl->n_timed; ++i) {      // oldest first
        const int s = (int)(i % fstat_plan::kRing);
        float ms = -1.f;
        if (cudaEventSynchronize(pl->ev1[s]) != cudaSuccess) { cudaGetLastError(); break; }
        if (cudaEventElapsedTime(&ms, pl->ev0[s], pl->ev1[s]) != cudaSuccess) { cudaGetLastError(); break; }
        ms_out[w++] = (double)ms;
    }
    return w;
}

// a1-a5 for P particles, then a6 (F, F_k) when F != NULL and / or the extrinsic amplitudes when amp != NULL
// Host buffers of fstat_eval_batch_host handed down to eval_impl: when the F_k block is large the evaluation is cut into
// ranges of partitions and fk_copied is set (the caller then copies F only).
struct HostOut {
    double *Fk_host = nullptr;
    bool fk_copied = false;
};

static fstat_status ensure_pipe(fstat_plan *pl)
{
    if (pl->pipe_copy_done) return FSTAT_OK;
    // Priorities (numerically lower = served first): the copy stream highest -- an epilogue becomes ready while later
    // ranges still have CTAs waiting and must not queue behind them -- then the ranges in order, so that concurrent
    // ranges do not share the SMs evenly and finish together.
    int prio_lo = 0, prio_hi = 0;
    CU_TRY(pl, cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    for (int i = 0; i < fstat_plan::kPipe; ++i) {
        const int pr = prio_hi + 1 + i < prio_lo ? prio_hi + 1 + i : prio_lo;
        if (!pl->pipe_main[i]) CU_TRY(pl, cudaStreamCreateWithPriority(&pl->pipe_main[i], cudaStreamNonBlocking, pr));
        if (!pl->pipe_main_done[i]) CU_TRY(pl, cudaEventCreateWithFlags(&pl->pipe_main_done[i], cudaEventDisableTiming));
    }
    if (!pl->pipe_copy) CU_TRY(pl, cudaStreamCreateWithPriority(&pl->pipe_copy, cudaStreamNonBlocking, prio_hi));
    pl->pipe_ranges = prio_lo - prio_hi;
    if (pl->pipe_ranges < 1) pl->pipe_ranges = 1;
    if (pl->pipe_ranges > fstat_plan::kPipe) pl->pipe_ranges = fstat_plan::kPipe;
    if (!pl->pipe_fork) CU_TRY(pl, cudaEventCreateWithFlags(&pl->pipe_fork, cudaEventDisableTiming));
    CU_TRY(pl, cudaEventCreateWithFlags(&pl->pipe_copy_done, cudaEventDisableTiming));
    return FSTAT_OK;
}

// fused != NULL (row f4): pl = fused[0]; the n_fused plans (A / E / T family, same grid, partitions and schedule) are
// evaluated by one pass of the multi-channel interpolating kernel, each into its own partial sums.
static fstat_status eval_impl(fstat_plan *pl, int64_t P, const double *params, double *F, double *Fk, double *amp,
                              void *stream, bool sums_only = false, fstat_plan *const *fused = nullptr,
                              int32_t n_fused = 0, HostOut *host = nullptr)
{
    if (!pl) return FSTAT_EINVAL;
    if (P < 0) return fail(pl, FSTAT_EINVAL, "P < 0");
    if (P == 0) return FSTAT_OK;
    if (!params || (!F && !amp && !sums_only)) return fail(pl, FSTAT_EINVAL, "params or the output pointer is NULL");
    if (P > ((int64_t)1 << 30)) return fail(pl, FSTAT_EUNSUPPORTED, "P > 2^30");
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)stream;

    const int64_t n_groups = (P + kThreads - 1) / kThreads;
    const int64_t P_pad = n_groups * kThreads;
    fstat_status s = ensure_segments(pl, (int32_t)n_groups);
    if (s != FSTAT_OK) return s;
    if ((int64_t)pl->n_seg * n_groups >= ((int64_t)1 << 31))
        return fail(pl, FSTAT_EUNSUPPORTED, "too many work items for one launch");
    CU_TRY(pl, grow(&pl->d_coef, &pl->coef_cap, (size_t)P_pad * kNCoef));
    CU_TRY(pl, grow(&pl->d_valid, &pl->valid_cap, (size_t)P_pad));
    CU_TRY(pl, grow(&pl->d_partial, &pl->partial_cap, (size_t)pl->n_seg * kNPartial * (size_t)P_pad));
    CU_TRY(pl, grow(&pl->d_level, &pl->level_cap, (size_t)pl->n_seg * (size_t)n_groups));
    CU_TRY(pl, grow(&pl->d_direct, &pl->direct_cap, (size_t)pl->n_seg * (size_t)n_groups + 1));
    {
        int32_t chunk = 0;
        const int32_t n_chunk = epilogue_chunks(P, pl->n_part, &chunk);
        CU_TRY(pl, grow(&pl->d_fpart, &pl->fpart_cap, (size_t)n_chunk * (size_t)P_pad));
    }
    pl->last_groups = (int32_t)n_groups;

    CU_TRY(pl, grow(&pl->d_slot, &pl->slot_cap, (size_t)P));
    CU_TRY(pl, grow(&pl->d_perm, &pl->perm_cap, (size_t)P_pad));
    CU_TRY(pl, grow(&pl->d_sort, &pl->sort_cap, prologue_scratch_bytes(P)));
    CU_TRY(pl, launch_prologue(params, P, P_pad, pl->opt.f_ref_e0, pl->opt.orbit_kappa, pl->d_slot, nullptr, pl->d_sort,
                               pl->d_coef, pl->d_valid, pl->d_perm, st));
    BandSched bs{};
    CU_TRY(pl, launch_schedule(pl->d_coef, pl->d_valid, P_pad, (int32_t)n_groups, pl->n_seg, pl->d_seg_crit,
                               pl->d_seg_maxlvl, pl->opt.interp_tol * 1.5e-7 * (2.0 / kPi), pl->opt.interp_tol * 2e-7,
                               pl->opt.force_level, pl->min_level, bs, pl->d_level, pl->d_direct + 1, pl->d_direct, st));
    FastArgs fa;
    fa.dwp = pl->d_dwp;
    fa.node = pl->d_node;
    for (int l = 0; l < kNLevels; ++l) fa.gram[l] = pl->d_gram[l];
    fa.coef = pl->d_coef;
    fa.seg_edge = pl->d_seg_edge;
    fa.seg_gbase = pl->d_seg_gbase;
    fa.level = pl->d_level;
    fa.partial = pl->d_partial;
    fa.part_sk = P_pad;
    fa.part_sp = 1;
    fa.P_pad = P_pad;
    fa.n_groups = (int32_t)n_groups;
    fa.n_seg = pl->n_seg;
    fa.segs_per_cta = segs_per_cta(pl->n_bins, pl->n_seg);
    fa.aet = pl->opt.tdi_channel >= FSTAT_TDI_A ? 1 : 0;
    fa.chunk_begin = 0;
    fa.chunk_count = 0;
    fa.df = pl->df;
    fa.orb = pl->orb;
    MainArgs a;
    a.dwp = pl->d_dwp;
    a.fw = pl->d_fw;
    a.arm_length_m = pl->opt.arm_length_m;
    a.coef = pl->d_coef;
    a.seg_edge = pl->d_seg_edge;
    a.direct_list = pl->d_direct + 1;
    a.direct_count = pl->d_direct;
    a.max_ctas = pl->n_sm * 12;
    a.partial = pl->d_partial;
    a.part_sk = fa.part_sk;
    a.part_sp = fa.part_sp;
    a.P_pad = P_pad;
    a.P = (int32_t)P;
    a.n_groups = (int32_t)n_groups;
    a.n_seg = pl->n_seg;
    a.aet = fa.aet;
    a.orb = pl->orb;
    const int slot = (int)(pl->n_timed % fstat_plan::kRing);
    if (n_fused > 1) {
        FastMultiArgs fm;
        memset(&fm, 0, sizeof(fm));
        for (int32_t c = 0; c < n_fused; ++c) {
            fstat_plan *pc = fused[c];
            if (c) {
                fstat_status sc = ensure_segments(pc, (int32_t)n_groups);
                if (sc != FSTAT_OK) { pl->err = pc->err; return sc; }
                if (pc->n_seg != pl->n_seg || pc->seg_len != pl->seg_len)
                    return fail(pl, FSTAT_ECUDA, "internal: the channels' segmentations differ");
                CU_TRY(pl, grow(&pc->d_partial, &pc->partial_cap, (size_t)pl->n_seg * kNPartial * (size_t)P_pad));
                pc->last_groups = (int32_t)n_groups;
                pc->last_was_band = false;
            }
            fm.dwp[c] = pc->d_dwp;
            for (int l = 0; l < kNLevels; ++l) fm.gram[c][l] = pc->d_gram[l];
            fm.partial[c] = pc->d_partial;
            for (int i = 0; i < 3; ++i) fm.wch[c][i] = pc->orb.wch[i];
        }
        fm.node = pl->d_node;
        fm.coef = pl->d_coef;
        fm.seg_edge = pl->d_seg_edge;
        fm.seg_gbase = pl->d_seg_gbase;
        fm.level = pl->d_level;
        fm.part_sk = fa.part_sk;
        fm.part_sp = fa.part_sp;
        fm.P_pad = P_pad;
        fm.n_groups = (int32_t)n_groups;
        fm.n_seg = pl->n_seg;
        fm.segs_per_cta = fa.segs_per_cta;
        fm.n_ch = n_fused;
        fm.df = pl->df;
        fm.orb = pl->orb;
        CU_TRY(pl, cudaEventRecord(pl->ev0[slot], st));
        CU_TRY(pl, launch_fastmulti(fm, st));
        for (int32_t c = 0; c < n_fused; ++c) {          // work items left to the direct kernel: one pass per channel
            fstat_plan *pc = fused[c];
            MainArgs ac = a;
            ac.dwp = pc->d_dwp;
            ac.fw = pc->d_fw;
            ac.partial = pc->d_partial;
            ac.orb = pc->orb;
            CU_TRY(pl, launch_main(ac, st));
        }
        CU_TRY(pl, cudaEventRecord(pl->ev1[slot], st));
        ++pl->n_timed;
        // keys, rank, prologue, stride selection, fused interpolating kernel, direct kernel per channel
        pl->n_launches += 5 + n_fused;
        pl->last_was_band = false;
        return FSTAT_OK;
    }
    {
        // Host-buffer call with a large F_k block (N_p = 1024, P = 2048: 16.8 MB, 0.3 ms over PCIe against a 5.2 ms step):
        // the interpolating kernel goes out as up to kPipe launches, each a range of partitions, on streams of its own
        // (concurrent: a later range fills the SMs the earlier one's last CTAs leave free); a copy stream follows them
        // range by range with that range's epilogue and the device-to-host copy of its F_k columns.  Only the last
        // range's epilogue and copy remain after the kernels.
        int32_t echunk = 0;
        const int32_t n_echunk = epilogue_chunks(P, pl->n_part, &echunk);
        const bool pipe = host && host->Fk_host && F && Fk && !amp && pl->fast_ok && n_echunk >= 2 &&
                          (size_t)P * (size_t)pl->n_part * sizeof(double) >= ((size_t)2 << 20);
        if (pipe) {
            fstat_status sp = ensure_pipe(pl);
            if (sp != FSTAT_OK) return sp;
            // one range per stream priority below the copy stream's (5 on B200: 5.31 ms end to end against 5.23 ms (first round-2 build) on the
            // device for config 1; ranges that share a priority share the SMs and finish together: 8 ranges 5.33 ms)
            const int32_t K = n_echunk < pl->pipe_ranges ? n_echunk : pl->pipe_ranges;
            const int32_t n_cta_chunks = (pl->n_seg + fa.segs_per_cta - 1) / fa.segs_per_cta;
            PartialSet one{};
            one.p[0] = pl->d_partial;
            one.n = 1;
            CU_TRY(pl, cudaEventRecord(pl->ev0[slot], st));
            CU_TRY(pl, launch_main(a, st));              // work items of the direct kernel: any partition, so first
            CU_TRY(pl, cudaEventRecord(pl->pipe_fork, st));
            int32_t cta_begin = 0;
            for (int32_t r = 0; r < K; ++r) {
                const int32_t c_lo = (int32_t)((int64_t)r * n_echunk / K), c_hi = (int32_t)((int64_t)(r + 1) * n_echunk / K);
                const int32_t k_lo = c_lo * echunk;
                const int32_t k_end = (int64_t)c_hi * echunk < pl->n_part ? c_hi * echunk : pl->n_part;
                const int32_t s_end = pl->part_seg_h[k_end];
                const int32_t cta_end = (r == K - 1) ? n_cta_chunks : (s_end + fa.segs_per_cta - 1) / fa.segs_per_cta;
                cudaStream_t sm = pl->pipe_main[r];
                CU_TRY(pl, cudaStreamWaitEvent(sm, pl->pipe_fork, 0));
                if (cta_end > cta_begin) {
                    fa.chunk_begin = cta_begin;
                    fa.chunk_count = cta_end - cta_begin;
                    CU_TRY(pl, launch_fast(fa, sm));
                    pl->n_launches += 1;
                    cta_begin = cta_end;
                }
                CU_TRY(pl, cudaEventRecord(pl->pipe_main_done[r], sm));
                // the copy stream has already waited for the ranges before this one
                CU_TRY(pl, cudaStreamWaitEvent(pl->pipe_copy, pl->pipe_main_done[r], 0));
                CU_TRY(pl, launch_epilogue_range(one, pl->d_part_seg, pl->d_valid, pl->d_perm, P, P_pad, pl->n_part, pl->n_seg,
                                                 c_lo, c_hi, pl->d_fpart, F, Fk, pl->pipe_copy));
                CU_TRY(pl, cudaMemcpy2DAsync(host->Fk_host + k_lo, (size_t)pl->n_part * sizeof(double), Fk + k_lo,
                                             (size_t)pl->n_part * sizeof(double), (size_t)(k_end - k_lo) * sizeof(double),
                                             (size_t)P, cudaMemcpyDeviceToHost, pl->pipe_copy));
                pl->n_launches += 1;
            }
            CU_TRY(pl, cudaEventRecord(pl->pipe_copy_done, pl->pipe_copy));
            CU_TRY(pl, cudaStreamWaitEvent(st, pl->pipe_copy_done, 0));
            CU_TRY(pl, cudaEventRecord(pl->ev1[slot], st));
            ++pl->n_timed;
            CU_TRY(pl, launch_fsum(pl->d_fpart, pl->d_valid, pl->d_perm, P, P_pad, n_echunk, F, st));
            pl->n_launches += 5 + 1;                      // keys, rank, prologue, stride selection, direct; chunk sums of F
            pl->last_was_band = false;
            host->fk_copied = true;
            return FSTAT_OK;
        }
    }
    CU_TRY(pl, cudaEventRecord(pl->ev0[slot], st));
    if (pl->fast_ok) CU_TRY(pl, launch_fast(fa, st));
    CU_TRY(pl, launch_main(a, st));
    CU_TRY(pl, cudaEventRecord(pl->ev1[slot], st));
    ++pl->n_timed;
    // keys, rank (or radix sort: counted as one), prologue, stride selection, [interpolating], direct
    pl->n_launches += 5 + (pl->fast_ok ? 1 : 0);
    pl->last_was_band = false;
    if (F) {
        PartialSet one{};
        one.p[0] = pl->d_partial;
        one.n = 1;
        CU_TRY(pl, launch_epilogue(one, pl->d_part_seg, pl->d_valid, pl->d_perm, P, P_pad, pl->n_part, pl->n_seg,
                                   pl->d_fpart, F, Fk, st));
        int32_t chunk = 0;                             // epilogue, [chunk sums of F]
        pl->n_launches += 1 + (epilogue_chunks(P, pl->n_part, &chunk) > 1 ? 1 : 0);
    }
    if (amp) {
        CU_TRY(pl, launch_amplitudes(pl->d_partial, pl->d_part_seg, pl->d_valid, pl->d_perm, P, P_pad, pl->n_part, amp, st));
        pl->n_launches += 1;
    }
    return FSTAT_OK;
}

fstat_status fstat_eval_batch(fstat_plan *pl, int64_t P, const double *params, double *F, double *Fk, void *stream)
{
    if (pl && P > 0 && !F) return fail(pl, FSTAT_EINVAL, "params or F is NULL");
    return eval_impl(pl, P, params, F, Fk, nullptr, stream);
}

fstat_status fstat_eval_batch_channels(fstat_plan *const *plans, int32_t n_channels, int64_t P, const double *params,
                                       double *F, double *Fk, void *stream)
{
    if (!plans || n_channels < 1 || !plans[0]) return FSTAT_EINVAL;
    fstat_plan *p0 = plans[0];
    if (n_channels > kMaxChannels) return fail(p0, FSTAT_EUNSUPPORTED, "more than 4 channels");
    if (P < 0) return fail(p0, FSTAT_EINVAL, "P < 0");
    if (P == 0) return FSTAT_OK;
    if (!params || !F) return fail(p0, FSTAT_EINVAL, "params or F is NULL");
    for (int32_t c = 1; c < n_channels; ++c) {
        const fstat_plan *pc = plans[c];
        if (!pc) return fail(p0, FSTAT_EINVAL, "a channel's plan is NULL");
        for (int32_t b = 0; b < c; ++b)
            if (plans[b] == pc) return fail(p0, FSTAT_EINVAL, "the same plan given for two channels");
        if (pc->device != p0->device || pc->n_bins != p0->n_bins || pc->df != p0->df || pc->f0 != p0->f0 ||
            pc->edges != p0->edges || pc->opt.max_segment_bins != p0->opt.max_segment_bins ||
            pc->opt.f_ref_e0 != p0->opt.f_ref_e0 || pc->opt.orbit_kappa != p0->opt.orbit_kappa ||
            pc->opt.arm_length_m != p0->opt.arm_length_m)
            return fail(p0, FSTAT_EINVAL, "the channels' plans differ in device, grid, partitions or options other than the response");
    }
    PartialSet ps{};
    ps.n = n_channels;
    // two or three channels of the A / E / T family with one orbit and one set of tolerances: one fused pass
    bool fuse = (n_channels == 2 || n_channels == 3) && !p0->opt.no_channel_fusion;
    for (int32_t c = 0; fuse && c < n_channels; ++c) {
        const fstat_plan *pc = plans[c];
        fuse = pc->fast_ok && pc->opt.tdi_channel >= FSTAT_TDI_A && pc->opt.tdi_channel <= FSTAT_TDI_T &&
               memcmp(pc->orb.c, p0->orb.c, sizeof(p0->orb.c)) == 0 && pc->opt.interp_tol == p0->opt.interp_tol &&
               pc->opt.force_level == p0->opt.force_level && pc->min_level == p0->min_level;
    }
    if (fuse) {
        fstat_status s = eval_impl(p0, P, params, nullptr, nullptr, nullptr, stream, true, plans, n_channels);
        if (s != FSTAT_OK) return s;
        for (int32_t c = 0; c < n_channels; ++c) ps.p[c] = plans[c]->d_partial;
    }
    for (int32_t c = 0; !fuse && c < n_channels; ++c) {
        fstat_status s = eval_impl(plans[c], P, params, nullptr, nullptr, nullptr, stream, true);
        if (s != FSTAT_OK) { if (c) p0->err = plans[c]->err; return s; }
        if (plans[c]->n_seg != p0->n_seg) return fail(p0, FSTAT_ECUDA, "internal: the channels' segmentations differ");
        ps.p[c] = plans[c]->d_partial;
    }
    DeviceGuard g(p0->device);
    if (!g.ok) return fail(p0, FSTAT_ECUDA, "cudaSetDevice failed");
    const int64_t P_pad = (P + kThreads - 1) / kThreads * kThreads;
    CU_TRY(p0, launch_epilogue(ps, p0->d_part_seg, p0->d_valid, p0->d_perm, P, P_pad, p0->n_part, p0->n_seg, p0->d_fpart, F, Fk,
                               (cudaStream_t)stream));
    int32_t chunk = 0;
    p0->n_launches += 1 + (epilogue_chunks(P, p0->n_part, &chunk) > 1 ? 1 : 0);
    return FSTAT_OK;
}

fstat_status fstat_eval_amplitudes(fstat_plan *pl, int64_t P, const double *params, double *amp, void *stream)
{
    if (pl && P > 0 && !amp) return fail(pl, FSTAT_EINVAL, "params or amp is NULL");
    return eval_impl(pl, P, params, nullptr, nullptr, amp, stream);
}

// Internal plan for row f2: same tables (shared, not copied), ONE partition = the whole grid, so that its segmentation
// is just the work segments (multiples of the segment length) and its stride selection / work lists can be reused.
static fstat_status ensure_band_plan(fstat_plan *pl)
{
    if (pl->bandplan) return FSTAT_OK;
    fstat_plan *cp = new (std::nothrow) fstat_plan;
    if (!cp) return fail(pl, FSTAT_ENOMEM, "host allocation failed");
    cp->device = pl->device; cp->n_sm = pl->n_sm; cp->n_bins = pl->n_bins; cp->df = pl->df; cp->opt = pl->opt;
    cp->f0 = pl->f0; cp->orb = pl->orb; cp->fast_ok = pl->fast_ok;
    cp->d_dwp = pl->d_dwp; cp->d_fw = pl->d_fw; cp->d_node = pl->d_node;
    cp->n_node_rows = pl->n_node_rows;
    cp->shares_tables = true;
    try {
        cp->edges.assign({(int64_t)0, pl->n_bins});
        for (int l = 0; l < kNLevels; ++l) cp->cnt[l].assign(1, 0);
    } catch (...) {
        plan_free(cp);
        return fail(pl, FSTAT_ENOMEM, "host allocation failed");
    }
    cp->n_part = 1;
    pl->bandplan = cp;
    return FSTAT_OK;
}

// Prefix Gram matrices of every stride level (80 bytes per 8 bins and level), built at the first band call.
static fstat_status ensure_prefix_gram(fstat_plan *pl)
{
    if (pl->pgram_built) return FSTAT_OK;
    const int64_t n_lat = (pl->n_bins + kMinStride - 1) / kMinStride;
    for (int l = 0; l < kNLevels; ++l) {
        if (!pl->d_pgram[l]) CU_TRY(pl, cudaMalloc((void **)&pl->d_pgram[l], (size_t)n_lat * kNGram * sizeof(double)));
        CU_TRY(pl, launch_build_prefix_gram(pl->d_fw, pl->n_bins, l, pl->d_pgram[l], 0));
    }
    CU_TRY(pl, cudaDeviceSynchronize());           // built on the default stream; the caller's stream may not wait for it
    pl->pgram_built = true;
    return FSTAT_OK;
}

static fstat_status bands_impl(fstat_plan *pl, int64_t P, const double *params, int32_t n_seg, int32_t edge_lattice,
                               double *F, double *Fk, int64_t *band, double *amp, void *stream)
{
    if (!pl) return FSTAT_EINVAL;
    if (P < 0) return fail(pl, FSTAT_EINVAL, "P < 0");
    if (n_seg < 1 || edge_lattice < 1) return fail(pl, FSTAT_EINVAL, "n_seg < 1 or edge_lattice < 1");
    if (P == 0) return FSTAT_OK;
    if (!params || (!F && !amp)) return fail(pl, FSTAT_EINVAL, "params or the output pointer is NULL");
    if (P > ((int64_t)1 << 30)) return fail(pl, FSTAT_EUNSUPPORTED, "P > 2^30");
    if (pl->n_bins >= ((int64_t)1 << 31) - edge_lattice) return fail(pl, FSTAT_EUNSUPPORTED, "grid too long for 32-bit bins");
    if (pl->opt.tdi_channel >= FSTAT_TDI_A)
        return fail(pl, FSTAT_EUNSUPPORTED, "per-template bands are built for the Michelson responses X, Y, Z only");
    if (P * (int64_t)n_seg >= ((int64_t)1 << 40)) return fail(pl, FSTAT_EUNSUPPORTED, "P x n_seg too large");
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)stream;

    fstat_status s = ensure_band_plan(pl);
    if (s != FSTAT_OK) return s;
    fstat_plan *cp = pl->bandplan;
    if (cp->opt.max_segment_bins != pl->opt.max_segment_bins) invalidate_segments(cp);
    cp->opt = pl->opt;
    const int64_t n_groups = (P + kThreads - 1) / kThreads;
    const int64_t P_pad = n_groups * kThreads;
    s = ensure_segments(cp, (int32_t)n_groups);
    if (s != FSTAT_OK) { pl->err = cp->err; return s; }
    const bool fast = cp->fast_ok && pl->opt.force_level != -1 && segments_fast_capable(auto_segment_len(cp, (int32_t)n_groups));
    if (fast) {
        s = ensure_prefix_gram(pl);
        if (s != FSTAT_OK) return s;
    }
    if ((int64_t)cp->n_seg * n_groups >= ((int64_t)1 << 31))
        return fail(pl, FSTAT_EUNSUPPORTED, "too many work items for one launch");

    if (!F) {                                          // amplitudes only: F goes to scratch
        CU_TRY(pl, grow(&pl->d_F, &pl->F_cap, (size_t)P));
        F = pl->d_F;
    }
    if (!Fk) {
        CU_TRY(pl, grow(&pl->d_band_fk, &pl->band_fk_cap, (size_t)P * (size_t)n_seg));
        Fk = pl->d_band_fk;
    }
    CU_TRY(pl, grow(&cp->d_coef, &cp->coef_cap, (size_t)P_pad * kNCoef));
    CU_TRY(pl, grow(&cp->d_valid, &cp->valid_cap, (size_t)P_pad));
    CU_TRY(pl, grow(&cp->d_slot, &cp->slot_cap, (size_t)P));
    CU_TRY(pl, grow(&cp->d_perm, &cp->perm_cap, (size_t)P_pad));
    CU_TRY(pl, grow(&cp->d_band, &cp->band_cap, (size_t)2 * (size_t)P_pad));
    CU_TRY(pl, grow(&cp->d_level, &cp->level_cap, (size_t)cp->n_seg * (size_t)n_groups));
    CU_TRY(pl, grow(&cp->d_direct, &cp->direct_cap, (size_t)cp->n_seg * (size_t)n_groups + 1));
    CU_TRY(pl, grow(&cp->d_rec, &cp->rec_cap, (size_t)cp->n_seg * 2 * kNPartial * (size_t)P_pad));
    if (!pl->d_err) {                                  // [0]: flag (2 words), then four 64-bit counters
        CU_TRY(pl, cudaMalloc((void **)&pl->d_err, 5 * sizeof(unsigned long long)));
        CU_TRY(pl, cudaMemset(pl->d_err, 0, 5 * sizeof(unsigned long long)));
    }
    CU_TRY(pl, cudaMemsetAsync(reinterpret_cast<unsigned long long *>(pl->d_err) + 1, 0, 4 * sizeof(unsigned long long), st));
    cp->last_groups = (int32_t)n_groups;

    // slots ranked by the position of the band (not by chirp mass): the 128 templates of a CTA overlap at both ends
    const double rank_band[3] = {1.0 / pl->df, pl->f0, pl->f0 + (double)(pl->n_bins - 1) * pl->df};
    CU_TRY(pl, grow(&cp->d_sort, &cp->sort_cap, prologue_scratch_bytes(P)));
    CU_TRY(pl, launch_prologue(params, P, P_pad, pl->opt.f_ref_e0, pl->opt.orbit_kappa, cp->d_slot, rank_band, cp->d_sort,
                               cp->d_coef, cp->d_valid, cp->d_perm, st));
    CU_TRY(pl, launch_band_limits(cp->d_coef, cp->d_valid, cp->d_perm, P_pad, (int32_t)pl->n_bins, pl->f0, pl->df,
                                  1.0 / pl->df, pl->opt.orbit_kappa, cp->d_band, cp->d_band + P_pad, band, st));
    BandSched bs{};
    bs.band_lo = cp->d_band;
    bs.band_hi = cp->d_band + P_pad;
    bs.seg_edge = cp->d_seg_edge;
    bs.n_seg_band = n_seg;
    bs.lattice = edge_lattice;
    bs.n_bins = (int32_t)pl->n_bins;
    CU_TRY(pl, launch_schedule(cp->d_coef, cp->d_valid, P_pad, (int32_t)n_groups, cp->n_seg, cp->d_seg_crit,
                               cp->d_seg_maxlvl, pl->opt.interp_tol * 1.5e-7 * (2.0 / kPi), pl->opt.interp_tol * 2e-7,
                               pl->opt.force_level, 0, bs, cp->d_level, cp->d_direct + 1, cp->d_direct, st));
    // empty partitions and templates without a band: F_k = 0, a = 0
    CU_TRY(pl, cudaMemsetAsync(Fk, 0, (size_t)P * (size_t)n_seg * sizeof(double), st));
    if (amp) CU_TRY(pl, cudaMemsetAsync(amp, 0, (size_t)P * (size_t)n_seg * 4 * sizeof(double), st));

    BandCommon bc;
    bc.band_lo = cp->d_band;
    bc.band_hi = cp->d_band + P_pad;
    bc.valid = cp->d_valid;
    bc.perm = cp->d_perm;
    bc.rec = cp->d_rec;
    bc.Fk = Fk;
    bc.amp = amp;
    bc.err = pl->d_err;
    bc.stats = reinterpret_cast<unsigned long long *>(pl->d_err) + 1;
    bc.N = n_seg;
    bc.C = edge_lattice;
    bc.n_bins = (int32_t)pl->n_bins;

    const int slot = (int)(pl->n_timed % fstat_plan::kRing);
    CU_TRY(pl, cudaEventRecord(pl->ev0[slot], st));
    if (fast) {
        FastBandArgs fa;
        fa.dwp = pl->d_dwp;
        fa.fw = pl->d_fw;
        fa.node = pl->d_node;
        for (int l = 0; l < kNLevels; ++l) fa.pgram[l] = pl->d_pgram[l];
        fa.coef = cp->d_coef;
        fa.seg_edge = cp->d_seg_edge;
        fa.level = cp->d_level;
        fa.b = bc;
        fa.P_pad = P_pad;
        fa.n_groups = (int32_t)n_groups;
        fa.n_seg = cp->n_seg;
        fa.df = pl->df;
        fa.orb = pl->orb;
        CU_TRY(pl, launch_fastband(fa, st));
    }
    BandArgs ba;
    ba.dwp = pl->d_dwp;
    ba.fw = pl->d_fw;
    ba.arm_length_m = pl->opt.arm_length_m;
    ba.coef = cp->d_coef;
    ba.seg_edge = cp->d_seg_edge;
    ba.direct_list = cp->d_direct + 1;
    ba.direct_count = cp->d_direct;
    ba.b = bc;
    ba.P_pad = P_pad;
    ba.n_seg = cp->n_seg;
    ba.orb = pl->orb;
    CU_TRY(pl, launch_band_main(ba, pl->n_sm * 12, st));
    CU_TRY(pl, cudaEventRecord(pl->ev1[slot], st));
    ++pl->n_timed;
    CU_TRY(pl, launch_band_short(pl->d_dwp, pl->d_fw, pl->opt.arm_length_m, cp->d_coef, bc, P_pad, pl->orb, st));
    CU_TRY(pl, launch_band_stitch(bc, P, P_pad, cp->seg_len, cp->n_seg, F, st));
    // keys, rank, keys, rank, prologue, band limits, stride selection, [interpolating], direct, short partitions, stitch, F sums
    pl->n_launches += 11 + (fast ? 1 : 0);
    pl->last_was_band = true;
    return FSTAT_OK;
}

fstat_status fstat_eval_batch_bands(fstat_plan *pl, int64_t P, const double *params, int32_t n_seg, int32_t edge_lattice,
                                    double *F, double *Fk, int64_t *band, void *stream)
{
    if (pl && P > 0 && !F) return fail(pl, FSTAT_EINVAL, "params or F is NULL");
    return bands_impl(pl, P, params, n_seg, edge_lattice, F, Fk, band, nullptr, stream);
}

fstat_status fstat_eval_amplitudes_bands(fstat_plan *pl, int64_t P, const double *params, int32_t n_seg,
                                         int32_t edge_lattice, double *amp, void *stream)
{
    if (pl && P > 0 && !amp) return fail(pl, FSTAT_EINVAL, "params or amp is NULL");
    return bands_impl(pl, P, params, n_seg, edge_lattice, nullptr, nullptr, nullptr, amp, stream);
}

fstat_status fstat_eval_batch_bands_host(fstat_plan *pl, int64_t P, const double *params_host, int32_t n_seg,
                                         int32_t edge_lattice, double *F_host, double *Fk_host, int64_t *band_host,
                                         void *stream)
{
    if (!pl) return FSTAT_EINVAL;
    if (P < 0) return fail(pl, FSTAT_EINVAL, "P < 0");
    if (n_seg < 1 || edge_lattice < 1) return fail(pl, FSTAT_EINVAL, "n_seg < 1 or edge_lattice < 1");
    if (P == 0) return FSTAT_OK;
    if (!params_host || !F_host) return fail(pl, FSTAT_EINVAL, "params_host or F_host is NULL");
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)stream;
    CU_TRY(pl, grow(&pl->d_params, &pl->params_cap, (size_t)P * 6));
    CU_TRY(pl, grow(&pl->d_F, &pl->F_cap, (size_t)P));
    if (Fk_host) CU_TRY(pl, grow(&pl->d_Fk, &pl->Fk_cap, (size_t)P * (size_t)n_seg));
    if (band_host) CU_TRY(pl, grow(&pl->d_band_out, &pl->band_out_cap, (size_t)P * 2));
    CU_TRY(pl, cudaMemcpyAsync(pl->d_params, params_host, (size_t)P * 6 * sizeof(double), cudaMemcpyHostToDevice, st));
    fstat_status s = fstat_eval_batch_bands(pl, P, pl->d_params, n_seg, edge_lattice, pl->d_F, Fk_host ? pl->d_Fk : nullptr,
                                            band_host ? pl->d_band_out : nullptr, stream);
    if (s != FSTAT_OK) return s;
    CU_TRY(pl, cudaMemcpyAsync(F_host, pl->d_F, (size_t)P * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (Fk_host)
        CU_TRY(pl, cudaMemcpyAsync(Fk_host, pl->d_Fk, (size_t)P * (size_t)n_seg * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (band_host)
        CU_TRY(pl, cudaMemcpyAsync(band_host, pl->d_band_out, (size_t)P * 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    CU_TRY(pl, cudaStreamSynchronize(st));
    return FSTAT_OK;
}

fstat_status fstat_eval_batch_host(fstat_plan *pl, int64_t P, const double *params_host, double *F_host,
                                   double *Fk_host, void *stream)
{
    if (!pl) return FSTAT_EINVAL;
    if (P < 0) return fail(pl, FSTAT_EINVAL, "P < 0");
    if (P == 0) return FSTAT_OK;
    if (!params_host || !F_host) return fail(pl, FSTAT_EINVAL, "params_host or F_host is NULL");
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)stream;
    CU_TRY(pl, grow(&pl->d_params, &pl->params_cap, (size_t)P * 6));
    CU_TRY(pl, grow(&pl->d_F, &pl->F_cap, (size_t)P));
    if (Fk_host) CU_TRY(pl, grow(&pl->d_Fk, &pl->Fk_cap, (size_t)P * (size_t)pl->n_part));
    CU_TRY(pl, cudaMemcpyAsync(pl->d_params, params_host, (size_t)P * 6 * sizeof(double), cudaMemcpyHostToDevice, st));
    HostOut ho;
    ho.Fk_host = Fk_host;
    fstat_status s = eval_impl(pl, P, pl->d_params, pl->d_F, Fk_host ? pl->d_Fk : nullptr, nullptr, stream, false, nullptr, 0, &ho);
    if (s != FSTAT_OK) return s;
    CU_TRY(pl, cudaMemcpyAsync(F_host, pl->d_F, (size_t)P * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (Fk_host && !ho.fk_copied)
        CU_TRY(pl, cudaMemcpyAsync(Fk_host, pl->d_Fk, (size_t)P * (size_t)pl->n_part * sizeof(double),
                                   cudaMemcpyDeviceToHost, st));
    CU_TRY(pl, cudaStreamSynchronize(st));
    return FSTAT_OK;
}

fstat_status fstat_eval_template(fstat_plan *pl, const double *params_host, double *u_plus, double *u_cross,
                                 void *stream)
{
    if (!pl) return FSTAT_EINVAL;
    if (!params_host || !u_plus || !u_cross) return fail(pl, FSTAT_EINVAL, "params_host, u_plus or u_cross is NULL");
    const double *q = params_host;
    for (int i = 0; i < 6; ++i)
        if (!isfinite(q[i])) return fail(pl, FSTAT_EINVAL, "non-finite parameter");
    if (!(q[1] > 0.0) || !(q[2] > 0.0 && q[2] <= 0.25) || !(q[5] >= 0.0))
        return fail(pl, FSTAT_EINVAL, "parameter outside the physical domain (M_c > 0, 0 < eta <= 1/4, e0 >= 0)");
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)stream;
    CU_TRY(pl, grow(&pl->d_params, &pl->params_cap, (size_t)6));
    CU_TRY(pl, grow(&pl->d_coef, &pl->coef_cap, (size_t)kThreads * kNCoef));
    CU_TRY(pl, grow(&pl->d_valid, &pl->valid_cap, (size_t)kThreads));
    CU_TRY(pl, cudaMemcpyAsync(pl->d_params, params_host, 6 * sizeof(double), cudaMemcpyHostToDevice, st));
    CU_TRY(pl, launch_prologue(pl->d_params, 1, kThreads, pl->opt.f_ref_e0, pl->opt.orbit_kappa, nullptr, nullptr, nullptr,
                               pl->d_coef, pl->d_valid, nullptr, st));
    CU_TRY(pl, launch_template(pl->d_fw, pl->opt.arm_length_m, pl->d_coef, kThreads, pl->n_bins, pl->orb, pl->opt.tdi_channel >= FSTAT_TDI_A ? 1 : 0,
                               u_plus, u_cross, st));
    CU_TRY(pl, cudaStreamSynchronize(st));
    return FSTAT_OK;
}

fstat_status fstat_probe_pipe_peak(int32_t device, int32_t which, double millis, double *inst_per_s, int32_t *n_sm_out)
{
    if (!inst_per_s || which < 0 || which > 3) return FSTAT_EINVAL;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) { cudaGetLastError(); return FSTAT_ECUDA; }
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return FSTAT_ECUDA;
    if (dev >= n_dev) return FSTAT_EINVAL;
    DeviceGuard g(dev);
    if (!g.ok) return FSTAT_ECUDA;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return FSTAT_ECUDA;
    if (n_sm_out) *n_sm_out = n_sm;
    double *sink = nullptr;
    if (cudaMalloc((void **)&sink, sizeof(double)) != cudaSuccess) return FSTAT_ENOMEM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int n_blocks = n_sm * 8;
    int iters = 2000;
    fstat_status rc = FSTAT_OK;
    double best = 0.0;
    // calibrate, then repeat until about `millis` of kernel time has been spent; keep the best rate
    double spent = 0.0;
    for (int rep = 0; rep < 64 && rc == FSTAT_OK; ++rep) {
        cudaEventRecord(e0, 0);
        if (launch_probe(which, n_blocks, iters, sink, 0) != cudaSuccess) { rc = FSTAT_ECUDA; break; }
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = FSTAT_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double inst = (double)n_blocks * 256.0 * (double)iters * 64.0;
        if (ms > 0.f && rep > 0) { const double r = inst / (ms * 1e-3); if (r > best) best = r; }
        if (rep > 0) spent += ms;
        if (ms < 2.0f && iters < (1 << 24)) iters *= 4;
        if (spent >= millis && rep >= 3) break;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *inst_per_s = best;
    return rc;
}


/* ---- App. B: host arithmetic on one amplitude vector, no device involved ---- */

// Eq. B1 (:413-420): the four amplitudes of (D_L, psi, iota, phi_c), D_L in the inverse units of the amplitudes
static void b1_forward(double d_l, double psi, double iota, double phi_c, double a[4])
{
    const double ci = cos(iota), p = 0.5 * (1.0 + ci * ci);
    const double c2 = cos(2.0 * psi), s2 = sin(2.0 * psi), cp = cos(phi_c), sp = sin(phi_c);
    a[0] = (c2 * p * cp - s2 * ci * sp) / d_l;
    a[1] = -(s2 * p * cp + c2 * ci * sp) / d_l;
    a[2] = -(c2 * p * sp + s2 * ci * cp) / d_l;
    a[3] = (s2 * p * sp - c2 * ci * cp) / d_l;
}

fstat_status fstat_amplitudes_from_extrinsic(double d_l, double psi, double iota, double phi_c, double *a_out)
{
    if (!a_out || !(d_l > 0.0) || !isfinite(d_l) || !isfinite(psi) || !isfinite(iota) || !isfinite(phi_c))
        return FSTAT_EINVAL;
    b1_forward(d_l, psi, iota, phi_c, a_out);
    return FSTAT_OK;
}

fstat_status fstat_extrinsic_from_amplitudes(const double *a, double chirp_mass_msun, double *out)
{
    if (!a || !out) return FSTAT_EINVAL;
    double a1 = a[0], a2 = a[1], a3 = a[2], a4 = a[3];
    if (!isfinite(a1) || !isfinite(a2) || !isfinite(a3) || !isfinite(a4) || !isfinite(chirp_mass_msun)) return FSTAT_EINVAL;
    if (chirp_mass_msun > 0.0) {
        // the templates drop the amplitude constant of Eq. A2 (:402, reading A21): library amplitude = K_A x the
        // paper's a_i with D_L in seconds, K_A = -sqrt(5/24) (G M_c / c^3)^(5/6) / pi^(2/3)
        const double k = -sqrt(5.0 / 24.0) * pow(chirp_mass_msun * kGMsunC3, 5.0 / 6.0) / pow(kPi, 2.0 / 3.0);
        a1 /= k; a2 /= k; a3 /= k; a4 /= k;
    }
    const double r_plus = hypot(a1 + a4, a2 - a3), r_minus = hypot(a1 - a4, a2 + a3);
    const double A_plus = r_plus + r_minus, A_cross = r_plus - r_minus;        // Eq. B3
    const double root = 2.0 * sqrt(r_plus * r_minus);                          // sqrt(A_+^2 - A_x^2), without the cancellation
    const double A = A_plus + root;
    if (!(A > 0.0)) { out[0] = INFINITY; out[1] = 0.0; out[2] = 0.0; out[3] = 0.0; return FSTAT_OK; }
    double r = -A_cross / A;
    r = r < -1.0 ? -1.0 : (r > 1.0 ? 1.0 : r);
    const double iota = acos(r);                                               // Eq. B2
    const double num = A_plus * a4 - A_cross * a1;
    const double den_psi = -(A_cross * a2 + A_plus * a3);
    const double psi = 0.5 * (den_psi != 0.0 ? atan(num / den_psi) : copysign(kPi / 2.0, num));
    const double c = sin(2.0 * psi) >= 0.0 ? 1.0 : -1.0;
    const double den = -c * (A_cross * a3 + A_plus * a2);
    double phi_c = den != 0.0 ? atan(c * num / den) : copysign(kPi / 2.0, c * num);
    // Eq. B2's arctan fixes phi_c only modulo pi, and phi_c -> phi_c + pi flips the sign of all four a_i in Eq. B1:
    // the half-plane is the one that reproduces the sign of the amplitudes (reading A25)
    double back[4];
    b1_forward(2.0 / A, psi, iota, phi_c, back);
    if (back[0] * a1 + back[1] * a2 + back[2] * a3 + back[3] * a4 < 0.0) phi_c = phi_c <= 0.0 ? phi_c + kPi : phi_c - kPi;
    out[0] = (2.0 / A) * (chirp_mass_msun > 0.0 ? kC : 1.0);
    out[1] = iota;
    out[2] = psi;
    out[3] = phi_c;
    return FSTAT_OK;
}

}  // extern "C"

/* ---- fstat_eval_batch_noalloc: the evaluation of fstat_eval_batch with its workspace in a static device array ---- */

// Every GPU that loads the library holds this array until the process exits.  In host code the NAME is only a stand-in
// for the symbol, not a device address: the address comes from cudaGetSymbolAddress, once per device, with that device
// current (noalloc_scratch_base below).
constexpr size_t kNoAllocBytes = (size_t)32 << 20;
constexpr int64_t kNoAllocMaxP = 16384;       // = kRankBrute of fstat_kernels.cu: above it launch_prologue calls the cub radix sort
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

namespace {

constexpr int kNoAllocMaxDevices = 64;
unsigned char *g_noalloc_base[kNoAllocMaxDevices] = {};

// device address of the scratch array on `device` (which must be current); nullptr + *err on failure
unsigned char *noalloc_scratch_base(int device, cudaError_t *err)
{
    *err = cudaSuccess;
    if (device < 0 || device >= kNoAllocMaxDevices) { *err = cudaErrorInvalidDevice; return nullptr; }
    if (!g_noalloc_base[device]) {
        void *ptr = nullptr;
        *err = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (*err != cudaSuccess) { cudaGetLastError(); return nullptr; }
        g_noalloc_base[device] = static_cast<unsigned char *>(ptr);
    }
    return g_noalloc_base[device];
}

// bump allocator over the scratch array: 256-byte aligned pieces
struct Carver {
    unsigned char *base;
    size_t used = 0;
    template <class T> T *take(size_t n)
    {
        T *p = reinterpret_cast<T *>(base + used);
        used += (n * sizeof(T) + 255) / 256 * 256;
        return p;
    }
};

}  // namespace

extern "C" {

int64_t fstat_noalloc_scratch_bytes(void) { return (int64_t)kNoAllocBytes; }

fstat_status fstat_eval_batch_noalloc(fstat_plan *pl, int64_t P, const double *params, double *F, double *Fk, void *stream)
{
    if (!pl) return FSTAT_EINVAL;
    if (P < 0) return fail(pl, FSTAT_EINVAL, "P < 0");
    if (P == 0) return FSTAT_OK;
    if (!params || !F) return fail(pl, FSTAT_EINVAL, "params or F is NULL");
    if (P > kNoAllocMaxP)
        return fail(pl, FSTAT_EUNSUPPORTED, "fstat_eval_batch_noalloc: P > 16384 (the slot ranking above that size uses a library sort)");
    DeviceGuard g(pl->device);
    if (!g.ok) return fail(pl, FSTAT_ECUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)stream;

    const int64_t n_groups = (P + kThreads - 1) / kThreads;
    const int64_t P_pad = n_groups * kThreads;
    // The segment tables of this batch size belong to the plan and are built (cudaMalloc) the first time a batch of this
    // many 128-particle groups is evaluated: this call only looks them up.
    if (pl->seg_groups != (int32_t)n_groups) {
        const int64_t seg_len = auto_segment_len(pl, (int32_t)n_groups);
        const SegTables *hit = nullptr;
        for (const SegTables &t : pl->seg_cache)
            if (t.seg_len == seg_len) { hit = &t; break; }
        if (!hit)
            return fail(pl, FSTAT_EUNSUPPORTED,
                        "fstat_eval_batch_noalloc: the plan has no segment tables for this batch size yet; they are part of "
                        "plan set-up: call fstat_eval_batch once with a batch of this size after fstat_plan_create / "
                        "fstat_plan_set_partitions");
        use_seg_tables(pl, *hit, (int32_t)n_groups);
    }
    if ((int64_t)pl->n_seg * n_groups >= ((int64_t)1 << 31))
        return fail(pl, FSTAT_EUNSUPPORTED, "too many work items for one launch");

    cudaError_t ce = cudaSuccess;
    Carver cv{noalloc_scratch_base(pl->device, &ce)};
    if (!cv.base) return fail(pl, FSTAT_ECUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(ce));
    int32_t chunk = 0;
    const int32_t n_chunk = epilogue_chunks(P, pl->n_part, &chunk);
    double *d_coef = cv.take<double>((size_t)P_pad * kNCoef);
    int32_t *d_valid = cv.take<int32_t>((size_t)P_pad);
    int32_t *d_slot = cv.take<int32_t>((size_t)P);
    int32_t *d_perm = cv.take<int32_t>((size_t)P_pad);
    unsigned char *d_sort = cv.take<unsigned char>(prologue_scratch_bytes(P));
    int8_t *d_level = cv.take<int8_t>((size_t)pl->n_seg * (size_t)n_groups);
    int32_t *d_direct = cv.take<int32_t>((size_t)pl->n_seg * (size_t)n_groups + 1);
    double *d_fpart = cv.take<double>((size_t)n_chunk * (size_t)P_pad);
    double *d_partial = cv.take<double>((size_t)pl->n_seg * kNPartial * (size_t)P_pad);
    if (cv.used > kNoAllocBytes) {
        char msg[256];
        snprintf(msg, sizeof(msg), "fstat_eval_batch_noalloc: this batch needs %zu bytes of workspace (%d work segments x %lld "
                 "slots), the static scratch array holds %zu", cv.used, (int)pl->n_seg, (long long)P_pad, kNoAllocBytes);
        return fail(pl, FSTAT_EUNSUPPORTED, msg);
    }

    // the launch sequence of eval_impl; nothing in the scratch has to start at zero except the direct kernel's work
    // counter, which launch_schedule clears (every partial sum that is read is written by one of the two main kernels)
    CU_TRY(pl, launch_prologue(params, P, P_pad, pl->opt.f_ref_e0, pl->opt.orbit_kappa, d_slot, nullptr, d_sort, d_coef, d_valid,
                               d_perm, st));
    BandSched bs{};
    CU_TRY(pl, launch_schedule(d_coef, d_valid, P_pad, (int32_t)n_groups, pl->n_seg, pl->d_seg_crit, pl->d_seg_maxlvl,
                               pl->opt.interp_tol * 1.5e-7 * (2.0 / kPi), pl->opt.interp_tol * 2e-7, pl->opt.force_level,
                               pl->min_level, bs, d_level, d_direct + 1, d_direct, st));
    FastArgs fa;
    fa.dwp = pl->d_dwp;
    fa.node = pl->d_node;
    for (int l = 0; l < kNLevels; ++l) fa.gram[l] = pl->d_gram[l];
    fa.coef = d_coef;
    fa.seg_edge = pl->d_seg_edge;
    fa.seg_gbase = pl->d_seg_gbase;
    fa.level = d_level;
    fa.partial = d_partial;
    fa.part_sk = P_pad;
    fa.part_sp = 1;
    fa.P_pad = P_pad;
    fa.n_groups = (int32_t)n_groups;
    fa.n_seg = pl->n_seg;
    fa.segs_per_cta = segs_per_cta(pl->n_bins, pl->n_seg);
    fa.aet = pl->opt.tdi_channel >= FSTAT_TDI_A ? 1 : 0;
    fa.chunk_begin = 0;
    fa.chunk_count = 0;
    fa.df = pl->df;
    fa.orb = pl->orb;
    MainArgs a;
    a.dwp = pl->d_dwp;
    a.fw = pl->d_fw;
    a.arm_length_m = pl->opt.arm_length_m;
    a.coef = d_coef;
    a.seg_edge = pl->d_seg_edge;
    a.direct_list = d_direct + 1;
    a.direct_count = d_direct;
    a.max_ctas = pl->n_sm * 12;
    a.partial = d_partial;
    a.part_sk = fa.part_sk;
    a.part_sp = fa.part_sp;
    a.P_pad = P_pad;
    a.P = (int32_t)P;
    a.n_groups = (int32_t)n_groups;
    a.n_seg = pl->n_seg;
    a.aet = fa.aet;
    a.orb = pl->orb;
    if (pl->fast_ok) CU_TRY(pl, launch_fast(fa, st));
    CU_TRY(pl, launch_main(a, st));
    PartialSet one{};
    one.p[0] = d_partial;
    one.n = 1;
    CU_TRY(pl, launch_epilogue(one, pl->d_part_seg, d_valid, d_perm, P, P_pad, pl->n_part, pl->n_seg, d_fpart, F, Fk, st));
    // keys, rank, prologue, stride selection, [interpolating], direct, epilogue, [chunk sums of F]
    pl->n_launches += 5 + (pl->fast_ok ? 1 : 0) + 1 + (n_chunk > 1 ? 1 : 0);
    return FSTAT_OK;
}

}  // extern "C"
