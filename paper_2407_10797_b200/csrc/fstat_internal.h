// fstat_internal.h -- shared between the C-ABI host code (fstat_api.cu) and the kernels
// (fstat_kernels.cu): constants, table layout, launcher prototypes.  Product path only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fstat {

// physical constants
constexpr double kC = 299792458.0;                 // m/s
constexpr double kGMsunC3 = 4.925490947641267e-6;  // G Msun / c^3 [s]
constexpr double kAU = 149597870700.0;             // m
constexpr double kYear = 31557600.0;               // Julian year [s]
constexpr double kEulerGamma = 0.5772156649015329;
constexpr double kPi = 3.14159265358979323846;

// ---- row layout of the per-bin basis ("a0"): kTabW doubles per frequency.  Rows exist in HBM only for the nodes of the
// interpolating kernel (one every 8 bins); the full-model kernels expand their tiles in shared memory (fstat_direct.cuh).  Phase basis B_j and its derivative D_j = (dB_j/df)/year:
//   Psi [quarter turns] = c1 + c0 f + sum_{j=2..9} c_j B_j(f),   alpha [quarter turns] = a0 + sum c_j D_j(f)
enum TabCol : int {
    T_F = 0,      // f
    T_LNF,        // ln f
    T_FM53,       // f^(-5/3)
    T_FM1,        // f^(-1)
    T_FM23,       // f^(-2/3)
    T_FM13,       // f^(-1/3)
    T_FP13,       // f^(1/3)
    T_FP13LN,     // f^(1/3) ln f
    T_FM349,      // f^(-34/9)
    T_XQ,         // 2 f L / c  = (pi f L / c) in quarter turns
    T_D0,         // D_j, j = 2..9 in the order of the B_j above (8 columns: T_D0 .. T_D0+7)
    T_C2X = 18,   // cos(2 pi f L / c)
    T_S2X,        // sin(2 pi f L / c)
    T_DWR,        // Re, Im of  4 df f^(-7/6) conj(K_f) d~/S_n,   K_f = -i (1 - z^2), z = exp(-2 pi i f L/c)
    T_DWI,
    T_W,          // 4 df f^(-7/3) |K_f|^2 / S_n
    T_X,          // pi f L / c [rad]
    kTabW = 24
};

constexpr int kNCoef = 20;   // per-particle coefficients: c0..c9, a0, k[3], u[3], v[3]
constexpr int kNAcc = 8;     // z_+ (re, im), z_x (re, im), m_pp, m_cc, m_pc (re, im)
constexpr int kNPartial = 10;   // per (segment, particle): the eight sums in the basis (u_+, u_x - c u_+), then c (re, im)
constexpr int kThreads = 128;    // particles per CTA of the main kernel (one thread = one particle)
constexpr int kTileBins = 64;    // bins per TMA tile (64 * 24 * 8 B = 12 KiB)
constexpr int kStages = 3;       // TMA ring depth

// Orbit model coefficients: coordinate = C[0] + C[1] cos a + C[2] sin a + C[3] cos 2a + C[4] sin 2a
//                                        + C[5] cos 3a + C[6] sin 3a      (z has C[5] = C[6] = 0)
// vec 0: 4 p_1 / c  [quarter turns per Hz];  vec 1: (p_2 - p_1)/L;  vec 2: (p_3 - p_1)/L.
struct OrbitCoef {
    double c[3][3][7];
    double wch[3];    // A, E, T (options.tdi_channel 3..5): weights of the Michelson X, Y, Z responses; else unused
};

// ---- interpolating ("fast") path: the slow factors of the template (carrier phase without its linear
// term, T'_+, T'_x) are evaluated in full FP64 only at nodes every S = 8 << level bins and carried
// between nodes by the cubic through the four surrounding nodes.
constexpr int kNLevels = 7;                          // S = 8, 16, 32, 64, 128, 256, 512
constexpr int kLevel0Shift = 3;
constexpr int kMinStride = 1 << kLevel0Shift;
constexpr int kMaxStride = kMinStride << (kNLevels - 1);   // 512; segment cuts inside a partition are multiples of it
constexpr int kNodeStride = kMinStride;              // the node table has one row every 8 bins
constexpr int kNodePad = 2 * kMaxStride / kNodeStride;   // rows before bin 0 (nodes down to bin -1024)
constexpr int kWinNodes = 6;                         // nodes m-2 .. m+3 feed the cubic of interval [m, m+1]
constexpr int kNSlow = 5;                            // psi_nl, T'_+ (re, im), T'_x (re, im)
constexpr double kEconGain = 20.0;                   // 4th-order error of the economised cubic vs the 4-node cubic (72 asymptotically)
constexpr int kFastTileShift = 9;
constexpr int kFastTile = 1 << kFastTileShift;       // bins per TMA tile of the folded data (8 KiB), aligned to its size;
                                                     // >= kMaxStride so that no sub-block straddles two tiles
constexpr int kFastStages = 3;
constexpr int kNGram = 10;                           // upper triangle of the 4x4 Gram matrix of a sub-block (prefix tables of row f2)
constexpr int kNW = 24;                              // per sub-block table of the interpolating kernels: W = L^T E (4 x 6), G = L L^T (gram_to_w)

// per-segment factors of the a-priori interpolation error bound (host-made, see make_seg_crit)
struct SegCrit {
    double p1, p2;   // omega [orbital rad / bin] = c3 p1 + |c9| p2
    double q1, q2;   // (3/128) |d^4 Psi / dk^4| = c3 q1 + |c9| q2       [quarter turns per bin^4]
    double ad;       // (3/128) x Doppler phase amplitude                 [quarter turns]
    double ct;       // response: relative error = ct (omega S)^4
    double kl;       // 0.05 x partition length [bins]: sqrt(normalised det M_k) >~ min(1, kl omega)  (hazard H3)
    double r1, r2;   // third phase difference D3 = c3 r1 + |c9| r2 + Doppler part   [quarter turns per bin^3]
    double d2;       // second phase difference [quarter turns / bin^2] = d2 * omega; must stay below 1/64
};

struct MainArgs {
    const double *dwp;        // [n_bins][2] folded data
    const double *fw;         // [n_bins][2] (f, w')
    double arm_length_m;
    const double *coef;       // [kNCoef][P_pad]
    const int32_t *seg_edge;  // [n_seg + 1]
    const int32_t *direct_list;   // work items (group * n_seg + segment) left to the direct kernel ...
    const int32_t *direct_count;  // ... and how many (both written by schedule_kernel)
    int32_t max_ctas;             // persistent grid size
    double *partial;          // [n_seg][kNPartial][P_pad]  (value j of slot p at j * part_sk + p * part_sp)
    int64_t part_sk, part_sp; // (P_pad, 1): value-major, what the epilogue reads coalesced; (1, kNPartial): row f2's
                              // cells epilogue reads one slot's record as 80 contiguous bytes
    int64_t P_pad;
    int32_t P;
    int32_t n_groups;
    int32_t n_seg;
    int32_t aet;                  // 1: the A / E / T response (model_eval<true>)
    OrbitCoef orb;
};

// error bits raised by the table kernel (input validation on the device)
enum : uint32_t {
    ERR_FREQ_NONPOS = 1u, ERR_FREQ_ORDER = 2u, ERR_FREQ_UNIFORM = 4u, ERR_DW_NONFINITE = 8u,
    ERR_ISN_NONFINITE = 16u, ERR_ISN_NONPOS = 32u
};

struct FastArgs {
    const double *dwp;            // [n_bins][2] folded data 4 df f^(-7/6) conj(K_f) d/S_n
    const double *node;           // [n_node_rows][kTabW]; row r <-> bin (r - kNodePad) * kNodeStride
    const double *gram[kNLevels]; // [n_sub(level)][kNW]
    const double *coef;           // [kNCoef][P_pad]
    const int32_t *seg_edge;      // [n_seg + 1]
    const int32_t *seg_gbase;     // [n_seg][kNLevels] index of the segment's first sub-block in gram[level]
    const int8_t *level;          // [n_groups][n_seg]
    double *partial;              // [n_seg][kNPartial][P_pad], strides as in MainArgs
    int64_t part_sk, part_sp;
    int64_t P_pad;
    int32_t n_groups;
    int32_t n_seg;
    int32_t segs_per_cta;         // consecutive segments one CTA walks (tiles, node ring carried across their edges)
    int32_t aet;                  // 1: the A / E / T response (model_eval<true>)
    int32_t chunk_begin;          // this launch walks the CTA chunks [chunk_begin, chunk_begin + chunk_count) ...
    int32_t chunk_count;          // ... of segs_per_cta segments each; chunk_count = 0: all of them
    double df;
    OrbitCoef orb;
};

// row f4: the interpolating kernel for 2 or 3 channels of the A / E / T family in one pass (fstat_fastmulti.cu); the
// channels' plans share grid, partitions, segment tables and schedule, each has its own data, Gram tables and sums
constexpr int kMaxFused = 3;
struct FastMultiArgs {
    const double *dwp[kMaxFused];
    const double *gram[kMaxFused][kNLevels];
    double *partial[kMaxFused];
    double wch[kMaxFused][3];     // weights of the Michelson X', Y', Z' responses
    const double *node;
    const double *coef;
    const int32_t *seg_edge;
    const int32_t *seg_gbase;
    const int8_t *level;
    int64_t part_sk, part_sp;
    int64_t P_pad;
    int32_t n_groups;
    int32_t n_seg;
    int32_t segs_per_cta;
    int32_t n_ch;
    double df;
    OrbitCoef orb;                // of the unrelabelled constellation (wch unused)
};

// row f2: edge j of a template's band, e_j = min(C (q_lo + floor(j D / N)), n_bins)   (reading A26)
__host__ __device__ __forceinline__ int32_t band_edge(int32_t j, int32_t q_lo, int32_t D, int32_t N, int32_t C,
                                                      int32_t n_bins)
{
    const int64_t e = (int64_t)C * ((int64_t)q_lo + ((int64_t)j * D) / N);
    return (int32_t)(e < (int64_t)n_bins ? e : (int64_t)n_bins);
}

// row f2: a template goes through the interpolating kernel when none of its partitions is empty or shorter than the
// smallest stride (partition lengths are C floor(D / N) or C ceil(D / N) lattice cells of C bins); the others are
// evaluated partition by partition with the full model (band_short_kernel)
__host__ __device__ __forceinline__ bool band_fast_eligible(int32_t D, int32_t N, int32_t C)
{
    return D >= N && (int64_t)C * (int64_t)(D / N) >= (int64_t)kMinStride;
}

// what the stride selection needs to know about the bands (nullptr band_lo: fixed data-side partitions)
struct BandSched {
    const int32_t *band_lo;   // [P_pad]
    const int32_t *band_hi;
    const int32_t *seg_edge;  // [n_seg + 1]
    int32_t n_seg_band;       // partitions per template
    int32_t lattice;
    int32_t n_bins;
};

// row f2, both main kernels: per-thread bands, head / tail records of the work segments
struct BandCommon {
    const int32_t *band_lo;   // [P_pad] k_lo, k_hi of every slot (bins of the plan's grid)
    const int32_t *band_hi;
    const int32_t *valid;     // [P_pad]
    const int32_t *perm;      // [P_pad] slot -> particle
    double *rec;              // [n_seg][2][kNPartial][P_pad]: head (0) and tail (1) fragment of every work segment
    double *Fk;               // [P][N]
    double *amp;              // [P][N][4] or nullptr
    uint32_t *err;            // device flag: internal invariant violated
    unsigned long long *stats;// [4] warp-level work of the interpolating kernel in this call: bins, node intervals, intervals with a cut, runs
    int32_t N;                // partitions per template (the paper's N_seg)
    int32_t C;                // edges are multiples of this many bins (reading A26)
    int32_t n_bins;
};

struct FastBandArgs {
    const double *dwp;            // [n_bins][2] folded data
    const double *fw;             // [n_bins][2] (f, w' = 4 df f^(-7/3) |K_f|^2 / S_n)
    const double *node;           // [n_node_rows][kTabW]
    const double *pgram[kNLevels];// [ceil(n_bins / 8)][kNGram] prefix Gram matrices
    const double *coef;           // [kNCoef][P_pad]
    const int32_t *seg_edge;      // [n_seg + 1] work segments (multiples of 512 bins)
    const int8_t *level;          // [n_groups][n_seg]
    BandCommon b;
    int64_t P_pad;
    int32_t n_groups;
    int32_t n_seg;
    double df;
    OrbitCoef orb;
};

// the direct kernel with per-thread edges, for the work items the stride selection leaves to it
struct BandArgs {
    const double *dwp;        // [n_bins][2] folded data
    const double *fw;         // [n_bins][2] (f, w')
    double arm_length_m;
    const double *coef;       // [kNCoef][P_pad]
    const int32_t *seg_edge;  // [n_seg + 1]
    const int32_t *direct_list;
    const int32_t *direct_count;
    BandCommon b;
    int64_t P_pad;
    int32_t n_seg;
    OrbitCoef orb;
};

cudaError_t launch_band_limits(const double *coef, const int32_t *valid, const int32_t *perm, int64_t P_pad,
                               int32_t n_bins, double f0, double df, double T_obs, double kappa, int32_t *band_lo,
                               int32_t *band_hi, int64_t *band_out, cudaStream_t st);
cudaError_t launch_band_main(const BandArgs &a, int32_t max_ctas, cudaStream_t st);
cudaError_t band_kernel_configure();
cudaError_t launch_fastband(const FastBandArgs &a, cudaStream_t st);
cudaError_t fastband_kernel_configure();
cudaError_t launch_build_prefix_gram(const double *fw, int64_t n_bins, int level, double *pgram, cudaStream_t st);
// full model over every partition of the templates the interpolating kernel does not take (band_fast_eligible)
cudaError_t launch_band_short(const double *dwp, const double *fw, double arm_length_m, const double *coef,
                              const BandCommon &b, int64_t P_pad, const OrbitCoef &orb, cudaStream_t st);
// partitions that straddle work segments from their head / tail records; -inf / NaN rows of invalid particles;
// then F = sum_k F_k.  seg_len = bins per work segment (the last one may be shorter)
cudaError_t launch_band_stitch(const BandCommon &b, int64_t P, int64_t P_pad, int32_t seg_len, int32_t n_seg, double *F,
                               cudaStream_t st);

cudaError_t launch_build_table(const double *freq, const double *dw, const double *isn, int64_t n_bins,
                               double df, double arm_length_m, double *dwp, double *fw, uint32_t *err_bits,
                               cudaStream_t st);
cudaError_t launch_build_nodes(const double *freq, int64_t n_bins, double df, double arm_length_m,
                               int64_t n_rows, double *node, cudaStream_t st);
cudaError_t launch_build_gram(const double *fw, const int32_t *edges, int32_t n_part, int64_t n_bins,
                              int level, const int32_t *cnt, double *gram, cudaStream_t st);
cudaError_t launch_schedule(const double *coef, const int32_t *valid, int64_t P_pad, int32_t n_groups,
                            int32_t n_seg, const SegCrit *crit, const int8_t *seg_maxlvl, double tol_phi_qt,
                            double tol_resp, int32_t force_level, int32_t min_level, const BandSched &bands, int8_t *level,
                            int32_t *direct_list, int32_t *direct_count, cudaStream_t st);
cudaError_t launch_fast(const FastArgs &a, cudaStream_t st);
cudaError_t fast_kernel_configure();
cudaError_t launch_fastmulti(const FastMultiArgs &a, cudaStream_t st);
cudaError_t fastmulti_kernel_configure();
// rank_band: nullptr (slots ranked by chirp mass) or HOST {T_obs, f_first, f_last} (row f2: ranked by band)
// scratch: prologue_scratch_bytes(P) bytes of device memory (keys and, for large batches, the radix sort's buffers)
cudaError_t launch_prologue(const double *params, int64_t P, int64_t P_pad, double f_ref_e0, double kappa,
                            int32_t *slot_of, const double *rank_band, void *scratch, double *coef, int32_t *valid,
                            int32_t *perm, cudaStream_t st);
size_t prologue_scratch_bytes(int64_t P);
cudaError_t launch_main(const MainArgs &a, cudaStream_t st);
// row f4 (Eq. 3 :62): the partial sums of up to kMaxChannels TDI channels, all with the same segment / slot layout
constexpr int kMaxChannels = 4;
struct PartialSet {
    const double *p[kMaxChannels];
    int32_t n;
};
cudaError_t launch_epilogue(const PartialSet &partials, const int32_t *part_seg, const int32_t *valid,
                            const int32_t *perm, int64_t P, int64_t P_pad, int32_t n_part, int32_t n_seg,
                            double *Fpart, double *F, double *Fk, cudaStream_t st);
cudaError_t launch_epilogue_range(const PartialSet &partials, const int32_t *part_seg, const int32_t *valid,
                                  const int32_t *perm, int64_t P, int64_t P_pad, int32_t n_part, int32_t n_seg,
                                  int32_t chunk_lo, int32_t chunk_hi, double *Fpart, double *F, double *Fk, cudaStream_t st);
cudaError_t launch_fsum(const double *Fpart, const int32_t *valid, const int32_t *perm, int64_t P, int64_t P_pad,
                        int32_t n_chunk, double *F, cudaStream_t st);
int32_t epilogue_chunks(int64_t P, int32_t n_part, int32_t *chunk_out);
cudaError_t launch_amplitudes(const double *partial, const int32_t *part_seg, const int32_t *valid,
                              const int32_t *perm, int64_t P, int64_t P_pad, int32_t n_part, double *amp,
                              cudaStream_t st);
cudaError_t launch_template(const double *fw, double arm_length_m, const double *coef, int64_t P_pad, int64_t n_bins,
                            const OrbitCoef &orb, int32_t aet, double *u_plus, double *u_cross, cudaStream_t st);
cudaError_t launch_probe(int which, int n_blocks, int iters, double *sink, cudaStream_t st);
size_t main_kernel_smem_bytes();
cudaError_t main_kernel_configure();

void make_orbit_coef(double arm_length_m, double lambda, int32_t tdi_channel, OrbitCoef *out);

}  // namespace fstat
