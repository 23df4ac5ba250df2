// fstat_fast.cu -- the interpolating main kernel of the batched semi-coherent F-statistic and its
// plan-time tables.
//
// Idea: per (particle, bin) the template is u_P = K_f f^(-7/6) T'_P e^{-i Phi} with
// a FAST carrier phase Phi (many radians per bin) and SLOW factors: T'_+, T'_x and the non-linear part
// of Phi vary on the scale of the orbital phase at t_f, i.e. over hundreds to thousands of bins.  The
// kernel therefore evaluates the full FP64 model (model_eval, the same device code the direct kernel runs
// at every bin) only at NODES every S bins and carries the slow factors between nodes with the cubic
// through the four surrounding nodes.  With T'(i) a cubic in the bin index inside a sub-block,
//     z_P  = sum_i dw'_i e^{+i Phi_i} conj(T'_P(i)) = sum_n conj(c^P_n) A_n ,
//     A_n  = sum_i q_i C(j1 - i + n - 1, n)        (n-fold running sums of q_i = dw'_i e^{+i Phi_i}),
//     m_PQ = sum_i w'_i T'_P(i) conj(T'_Q(i))      = sum_ab y^P_a G_ab conj(y^Q_b)
// with c^P_n the Newton (binomial-basis) coefficients of the cubic, y^P_a its four node values and
// G_ab = sum_i w'_i l_a(i) l_b(i) a plan-time Gram matrix of the Lagrange basis.  Per bin that leaves:
// the carrier by a rotation recurrence on the forward differences of the phase cubic, one complex
// product with the folded data and four complex running sums -- 19 FP64 instructions instead of 263.
// S is chosen per (particle group, segment) from an a-priori error bound (schedule_kernel);
// work items for which no stride is accurate enough are left to the direct kernel.
//
// Inner products: PAPER.md:66 Eq. 4, :89-91 Eq. 8-9, :117 Eq. 12.  Template: :397-405 Eq. A1-A3,
// :206-229 Eq. 17-20 (N = 0).
#include "fstat_device.cuh"
#include "fstat_fast.cuh"
#include "fstat_internal.h"
#include "fstat_model.cuh"

#include <math.h>

namespace fstat {

// =================================================================================================
// plan time: node table.  Row r holds the particle-independent basis at bin b = (r - kNodePad) * 8;
// inside the band the frequency is the caller's freq[b] (so that nodes and bins see the same number),
// outside it is the uniform continuation of the grid.
// =================================================================================================
__global__ void build_nodes_kernel(const double *__restrict__ freq, int64_t n_bins, double df, double L,
                                   int64_t n_rows, double *__restrict__ node)
{
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    const int64_t b = (r - kNodePad) * kNodeStride;
    double f;
    if (b < 0) f = freq[0] + (double)b * df;
    else if (b >= n_bins) f = freq[n_bins - 1] + (double)(b - (n_bins - 1)) * df;
    else f = freq[b];
    double *row = node + r * kTabW;
    if (f > 0.0) fill_basis_row(f, L, row);
    else {
#pragma unroll
        for (int j = 0; j < kTabW; ++j) row[j] = 0.0;
        row[T_F] = f;
    }
    row[T_DWR] = 0.0;
    row[T_DWI] = 0.0;
    row[T_W] = 0.0;
}

cudaError_t launch_build_nodes(const double *freq, int64_t n_bins, double df, double arm_length_m,
                               int64_t n_rows, double *node, cudaStream_t st)
{
    const int nt = 128;
    build_nodes_kernel<<<(unsigned)((n_rows + nt - 1) / nt), nt, 0, st>>>(freq, n_bins, df, arm_length_m, n_rows, node);
    return cudaGetLastError();
}

// =================================================================================================
// plan time (per partition set): Gram matrices.  Level `level` cuts every partition at the multiples of
// S = 8 << level; sub-block [j0, j1) of node interval m = j0 / S in partition k has the table index
// m + cnt[k], cnt[k] = number of interior partition edges e_1..e_k that are not multiples of S.
// One thread per node interval; it walks its bins and flushes at every partition edge.
// =================================================================================================
__global__ void build_gram_kernel(const double2 *__restrict__ fw, const int32_t *__restrict__ edges,
                                  int32_t n_part, int64_t n_bins, int level, const int32_t *__restrict__ cnt,
                                  double *__restrict__ gram)
{
    const int S = kMinStride << level;
    const int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t b0 = m * S;
    if (b0 >= n_bins) return;
    const int64_t b1 = (b0 + S < n_bins) ? b0 + S : n_bins;
    // partition of bin b0: largest k with edges[k] <= b0
    int lo = 0, hi = n_part;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)edges[mid] <= b0) lo = mid; else hi = mid;
    }
    int k = lo;
    const double rS = 1.0 / (double)S;
    double g[kNGram];
#pragma unroll
    for (int j = 0; j < kNGram; ++j) g[j] = 0.0;
    for (int64_t i = b0; i < b1; ++i) {
        if (i == (int64_t)edges[k + 1]) {                  // partition edge inside the interval: flush
            double W[kNW];
            gram_to_w(g, W);
            double *out = gram + (m + cnt[k]) * kNW;
#pragma unroll
            for (int j = 0; j < kNW; ++j) out[j] = W[j];
#pragma unroll
            for (int j = 0; j < kNGram; ++j) g[j] = 0.0;
            ++k;
        }
        const double w = fw[i].y;
        double l[4];
        lagrange4((double)(i - b0) * rS, l);
        int j = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a; b < 4; ++b) g[j++] += w * l[a] * l[b];
    }
    double W[kNW];
    gram_to_w(g, W);
    double *out = gram + (m + cnt[k]) * kNW;
#pragma unroll
    for (int j = 0; j < kNW; ++j) out[j] = W[j];
}

cudaError_t launch_build_gram(const double *fw, const int32_t *edges, int32_t n_part, int64_t n_bins,
                              int level, const int32_t *cnt, double *gram, cudaStream_t st)
{
    const int S = kMinStride << level;
    const int64_t n_int = (n_bins + S - 1) / S;
    const int nt = 128;
    build_gram_kernel<<<(unsigned)((n_int + nt - 1) / nt), nt, 0, st>>>(reinterpret_cast<const double2 *>(fw), edges, n_part, n_bins, level, cnt, gram);
    return cudaGetLastError();
}

// =================================================================================================
// a1b: stride selection.  One CTA per particle group: the group's largest chirp coefficient c3 (the
// f^(-5/3) term) and eccentric coefficient |c9| bound, through SegCrit, the orbital phase advance per
// bin omega and with it the interpolation errors of the carrier phase and of the response at stride S:
//     E_phi(S) = S^4 (c3 q1 + |c9| q2 + ad omega^4)   [quarter turns],
//     E_T(S)   = ct (omega S)^4 / min(1, kl omega)     (relative, as seen through M_k^-1).
// The level written is the largest one that meets both tolerances, or -1 (direct kernel).
// =================================================================================================
__global__ void __launch_bounds__(kThreads) schedule_kernel(const double *__restrict__ coef,
                                                            const int32_t *__restrict__ valid, int64_t P_pad,
                                                            int32_t n_seg, const SegCrit *__restrict__ crit,
                                                            const int8_t *__restrict__ seg_maxlvl, double tol_phi_qt,
                                                            double tol_resp, int32_t force_level, int32_t min_level,
                                                            const BandSched bands, int8_t *__restrict__ level,
                                                            int32_t *__restrict__ direct_list,
                                                            int32_t *__restrict__ direct_count)
{
    __shared__ double s3[kThreads / 32], s9[kThreads / 32];
    __shared__ int32_t sLo[kThreads / 32], sHi[kThreads / 32], sLen[kThreads / 32];
    const int tid = threadIdx.x;
    const int grp = blockIdx.x;
    const int64_t p = (int64_t)grp * kThreads + tid;
    double c3 = 0.0, c9 = 0.0;
    if (valid[p]) {
        c3 = fabs(coef[3 * P_pad + p]);
        c9 = fabs(coef[9 * P_pad + p]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        c3 = fmax(c3, __shfl_xor_sync(0xffffffffu, c3, o));
        c9 = fmax(c9, __shfl_xor_sync(0xffffffffu, c9, o));
    }
    if ((tid & 31) == 0) { s3[tid >> 5] = c3; s9[tid >> 5] = c9; }
    __syncthreads();
    c3 = s3[0]; c9 = s9[0];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) { c3 = fmax(c3, s3[w]); c9 = fmax(c9, s9[w]); }

    // row f2: the group's bins [g_lo, g_hi) that at least one template evaluated by the main kernels is in band for,
    // and the group's shortest partition: it sets the H3 amplification (the partitions of the templates, not the work
    // segments) and CAPS the stride, so that a node interval holds at most one partition edge of any thread
    const bool banded = bands.band_lo != nullptr;
    int32_t g_lo = INT32_MAX, g_hi = 0, g_len = INT32_MAX;
    if (banded) {
        if (valid[p]) {
            const int32_t C = bands.lattice, N = bands.n_seg_band;
            const int32_t q_lo = (bands.band_lo[p] + C / 2) / C, D = (bands.band_hi[p] + C / 2) / C - q_lo;
            if (band_fast_eligible(D, N, C)) {
                g_lo = band_edge(0, q_lo, D, N, C, bands.n_bins);
                g_hi = band_edge(N, q_lo, D, N, C, bands.n_bins);
                g_len = C * (D / N);
            }
        }
        g_lo = __reduce_min_sync(0xffffffffu, g_lo);
        g_hi = __reduce_max_sync(0xffffffffu, g_hi);
        g_len = __reduce_min_sync(0xffffffffu, g_len);
        if ((tid & 31) == 0) { sLo[tid >> 5] = g_lo; sHi[tid >> 5] = g_hi; sLen[tid >> 5] = g_len; }
        __syncthreads();
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) { g_lo = min(g_lo, sLo[w]); g_hi = max(g_hi, sHi[w]); g_len = min(g_len, sLen[w]); }
    }

    // blockIdx.y splits the segments of the group (thousands of lattice cells in row f2)
    for (int seg = blockIdx.y * kThreads + tid; seg < n_seg; seg += gridDim.y * kThreads) {
        int mx = seg_maxlvl[seg];
        int lvl;
        SegCrit q = crit[seg];
        if (banded) {
            if (bands.seg_edge[seg + 1] <= g_lo || bands.seg_edge[seg] >= g_hi) {     // nobody is in band here
                level[(int64_t)grp * n_seg + seg] = (int8_t)-2;
                continue;
            }
            q.kl = 0.05 * (double)g_len;
            while (mx >= 0 && (kMinStride << mx) > g_len) --mx;                       // g_len >= 8: mx stays >= 0
        }
        const double om = fma(c3, q.p1, c9 * q.p2);
        const double d3 = fma(c3, q.r1, fma(c9, q.r2, q.ad * (128.0 / 3.0) * om * om * om));   // |D3|, quarter turns
        if (!(q.d2 * om < 0.015625) || !(1.25 * d3 <= 0.25 * tol_phi_qt)) {
            lvl = -1;       // phase differences too large for the small-angle series / the 4-bin hold of D2
        } else if (force_level >= -1) {
            lvl = force_level < mx ? force_level : mx;
        } else {
            const double om2 = om * om, om4 = om2 * om2;
            // per S^4; kEconGain: the economised six-node cubic against the four-node cubic of the bound
            const double ephi1 = fma(c3, q.q1, fma(c9, q.q2, q.ad * om4)) * (1.0 / kEconGain);
            // the response error is seen through M_k^-1: a partition over which the response barely changes
            // (kl omega < 1) has a near-singular M_k and amplifies it by 1 / sqrt(det) (hazard H3)
            const double kom = q.kl * om;
            const double eT1 = ((kom < 1.0) ? q.ct * om2 * om / q.kl : q.ct * om4) * (1.0 / kEconGain);
            lvl = -1;
            for (int l = 0; l <= mx; ++l) {
                const double S = (double)(kMinStride << l), S2 = S * S, S4 = S2 * S2;
                if (ephi1 * S4 <= tol_phi_qt && eT1 * S4 <= tol_resp) lvl = l;
            }
        }
        if (lvl < min_level) lvl = -1;                    // the plan keeps no tables for strides that small: direct kernel
        level[(int64_t)grp * n_seg + seg] = (int8_t)lvl;
        if (lvl < 0) direct_list[atomicAdd(direct_count, 1)] = grp * n_seg + seg;   // order is irrelevant
    }
}

cudaError_t launch_schedule(const double *coef, const int32_t *valid, int64_t P_pad, int32_t n_groups,
                            int32_t n_seg, const SegCrit *crit, const int8_t *seg_maxlvl, double tol_phi_qt,
                            double tol_resp, int32_t force_level, int32_t min_level, const BandSched &bands, int8_t *level,
                            int32_t *direct_list, int32_t *direct_count, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(direct_count, 0, sizeof(int32_t), st);
    if (e != cudaSuccess) return e;
    const unsigned gy = (unsigned)((n_seg + 16 * kThreads - 1) / (16 * kThreads));       // <= 16 segments per thread
    schedule_kernel<<<dim3((unsigned)n_groups, gy < 1 ? 1 : (gy > 64 ? 64 : gy)), kThreads, 0, st>>>(coef, valid, P_pad, n_seg, crit, seg_maxlvl,
                                                            tol_phi_qt, tol_resp, force_level, min_level, bands, level,
                                                            direct_list, direct_count);
    return cudaGetLastError();
}

// =================================================================================================
// a2-a5, interpolating kernel.  Grid = particle groups x segments (same work items as the direct kernel),
// CTA = 128 threads = 128 particles.  The folded data dw' of the segment streams through a 3-stage
// shared-memory ring of 512-bin tiles (TMA bulk copies, mbarrier completion); every thread reads the
// same element (broadcast).  Node rows and Gram matrices are warp-uniform global loads (L1/L2 hits).
// =================================================================================================
struct __align__(16) FastSmem {
    double2 tile[kFastStages][kFastTile];
    double win[kWinNodes][kNSlow][kThreads];   // per-thread ring of the last six node values (column = thread)
    uint64_t full[kFastStages];
};

template <bool AET>
__device__ __forceinline__ void fast_kernel_body(const FastArgs &a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FastSmem &sm = *reinterpret_cast<FastSmem *>(smem_raw);

    const int tid = threadIdx.x;
    const int grp = blockIdx.x % a.n_groups;
    const int chunk = blockIdx.x / a.n_groups + a.chunk_begin;
    const int seg_begin = chunk * a.segs_per_cta, seg_end = min(a.n_seg, seg_begin + a.segs_per_cta);
    const int8_t *level = a.level + (int64_t)grp * a.n_seg;
    const int64_t p = (int64_t)grp * kThreads + tid;         // < P_pad by construction
    const double *cf = a.coef + p;
    const double2 *dwp = reinterpret_cast<const double2 *>(a.dwp);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kFastStages; ++s) mbar_init(&sm.full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();                                         // barriers initialised before anyone waits
    int g0 = 0;                                              // tiles consumed so far by this CTA (ring position)

  // A CTA walks a chunk of consecutive segments.  Consecutive segments with the same stride form a RUN: the
  // data tiles, the node ring and the Gram-table pointer carry on across the partition edges inside a run
  // (sub-blocks are cut there and the eight sums are flushed per segment); segments left to the direct
  // kernel (level < 0) are skipped.
  for (int seg = seg_begin; seg < seg_end;) {
    const int lvl = level[seg];
    if (lvl < 0) { ++seg; continue; }                        // CTA-uniform
    int run_end = seg + 1;
    while (run_end < seg_end && level[run_end] == lvl) ++run_end;
    const int sh = kLevel0Shift + lvl;
    const double rS = 1.0 / (double)(1 << sh);

    const int lo = a.seg_edge[seg], hi = a.seg_edge[run_end];
    const int t_first = lo >> kFastTileShift;
    const int n_tiles = ((hi - 1) >> kFastTileShift) - t_first + 1;

    auto issue_tile = [&](int t) {                           // t = tile number relative to t_first
        const int slot = (g0 + t) % kFastStages;
        const int b0 = max(lo, (t_first + t) << kFastTileShift), b1 = min(hi, (t_first + t + 1) << kFastTileShift);
        const uint32_t bytes = (uint32_t)(b1 - b0) * (uint32_t)sizeof(double2);
        mbar_expect_tx(&sm.full[slot], bytes);
        tma_load_1d(&sm.tile[slot][b0 & (kFastTile - 1)], dwp + b0, bytes, &sm.full[slot]);
    };
    __syncthreads();                                         // every thread has left the previous run's tiles
    if (tid == 0)
        for (int s = 0; s < kFastStages && s < n_tiles; ++s) issue_tile(s);

    // linear phase term 2 pi f t_c in quarter turns: per-bin advance, reduced mod 4
    const double c0 = cf[0];
    const double slope = mulmod4(c0, a.df);

    // node ring: (psi_nl, T'_+ re, im, T'_x re, im) at the last six nodes, slot = (node + 6) % 6
    int m = lo >> sh;
    {
        double c[kNCoef];
        load_coef(cf, a.P_pad, c);
        for (int k = -2; k <= 2; ++k) {
            const double2 *row = reinterpret_cast<const double2 *>(
                a.node + ((int64_t)kNodePad + ((int64_t)(m + k) * (1 << lvl))) * kTabW);
            double v0, v1, v2, v3, v4;
            model_eval<AET>(row, c, a.orb, v0, v1, v2, v3, v4);
            const int slot = (m + k + kWinNodes) % kWinNodes;
            sm.win[slot][0][tid] = v0; sm.win[slot][1][tid] = v1; sm.win[slot][2][tid] = v2;
            sm.win[slot][3][tid] = v3; sm.win[slot][4][tid] = v4;
        }
    }
    int m_have = m + 2;                                      // highest node in the ring

    double acc[kNAcc];
#pragma unroll
    for (int j = 0; j < kNAcc; ++j) acc[j] = 0.0;

    const double *gram = a.gram[lvl] + (int64_t)a.seg_gbase[seg * kNLevels + lvl] * kNW;
    int cur_tile = -1;
    int cur_seg = seg;
    int seg_hi = a.seg_edge[cur_seg + 1];
    // Basis of the segment's sums (hazard H3): (u_+, u_x - c u_+) with c = T'_x / T'_+ at the segment's first
    // node.  F is invariant under it; over a narrow partition u_x is nearly c u_+, and accumulating the small
    // remainder directly keeps m_cc - |m_pc|^2 / m_pp from cancelling (rounding / sqrt(det) instead of / det).
    bool seg_start = true;
    double c_re = 0.0, c_im = 0.0;
    int j0 = lo;
    while (j0 < hi) {
        const int node0 = m << sh;                           // bin of node "0" of this interval
        const int j1 = min(seg_hi, node0 + (1 << sh));       // sub-block = node interval cut at the segment edge
        const int s_base = (m - 2 + kWinNodes) % kWinNodes;  // ring slot of node m-2
        // ---- new node m+3 (unless this sub-block continues an interval already entered)
        const double fnode = a.node[((int64_t)kNodePad + ((int64_t)m << lvl)) * kTabW + T_F];
        if (m + 3 > m_have) {
            m_have = m + 3;
            double c[kNCoef];
            load_coef(cf, a.P_pad, c);
            const double2 *row = reinterpret_cast<const double2 *>(
                a.node + ((int64_t)kNodePad + ((int64_t)(m + 3) * (1 << lvl))) * kTabW);
            double v0, v1, v2, v3, v4;
            model_eval<AET>(row, c, a.orb, v0, v1, v2, v3, v4);
            const int slot = (m + 3 + kWinNodes) % kWinNodes;
            sm.win[slot][0][tid] = v0; sm.win[slot][1][tid] = v1; sm.win[slot][2][tid] = v2;
            sm.win[slot][3][tid] = v3; sm.win[slot][4][tid] = v4;
        }
        // ---- carrier phase: economised cubic + exact linear term, as forward differences
        double t, D1, D2, D3;
        {
            double v[6], yref, e[4];
#pragma unroll
            for (int k = 0; k < 6; ++k) v[k] = sm.win[(s_base + k) % kWinNodes][0][tid];
            economise(v, yref, e);
            const double d0 = e[0] - e[1], d2 = e[2] - e[1], d3 = e[3] - e[1];
            const double a1 = fma(d0, -1.0 / 3.0, fma(d3, -1.0 / 6.0, d2));
            const double a2 = 0.5 * (d0 + d2);
            const double a3 = fma(d2, -0.5, (d3 - d0) * (1.0 / 6.0));
            const double G0 = red4(yref) + e[1] + mulmod4(c0, fnode);
            const double G1 = red4(fma(a1, rS, slope));
            const double G2 = a2 * rS * rS, G3 = a3 * rS * rS * rS;
            const double s0 = (double)(j0 - node0);
            t = fma(s0, fma(s0, fma(s0, G3, G2), G1), G0);
            D1 = fma(G3, fma(3.0 * s0, s0 + 1.0, 1.0), fma(G2, fma(2.0, s0, 1.0), G1));
            D2 = fma(G3, fma(6.0, s0, 6.0), 2.0 * G2);
            D3 = 6.0 * G3;
        }
        // ---- the tile that holds [j0, j1)
        const int tl = (j0 >> kFastTileShift) - t_first;
        if (tl != cur_tile) {
            if (cur_tile >= 0) {
                __syncthreads();                             // every thread is done with the previous tile
                if (tid == 0 && cur_tile + kFastStages < n_tiles) issue_tile(cur_tile + kFastStages);
            }
            cur_tile = tl;
            mbar_wait(&sm.full[(g0 + tl) % kFastStages], (uint32_t)(((g0 + tl) / kFastStages) & 1));
        }
        const double2 *tp = &sm.tile[(g0 + tl) % kFastStages][j0 & (kFastTile - 1)];
        const int nb = j1 - j0;

        // ---- per bin: q = dw' e^{+i Phi}; running sums A_0..A_3.  The carrier e^{+i Phi_i} is carried by a
        // rotation recurrence on the forward differences D1, D2, D3 of the phase cubic:
        //   E <- E R,  R <- R Q  every bin;   Q <- Q C^4  every 4 bins   (R = e^{i D1}, Q = e^{i D2}, C = e^{i D3}).
        // Holding D2 at its mid-run value for 4 bins keeps D1 and the phase exact at the run ends; the D1
        // offset -5/4 D3 centres what is left inside a run: |phase error| <= 1.25 D3, and the stride selection
        // admits only work items with 1.25 D3 below a quarter of the phase tolerance.  19 FP64 instructions
        // per bin, no range reduction; rounding grows like n^2.5 ulp (1e-10 at n = 256) and, like every carrier
        // error, is common to u_+ and u_x, so M_k^-1 does not amplify it.
        double Er, Ei, Rr, Ri, Qr, Qi, Cr, Ci;
        sincos_qt(t, Ei, Er);
        sincos_qt(fma(-1.25, D3, D1), Ri, Rr);
        sincos_qt_small(fma(1.5, D3, D2), Qi, Qr);
        sincos_qt_small(4.0 * D3, Ci, Cr);
        double A0r = 0.0, A0i = 0.0, A1r = 0.0, A1i = 0.0, A2r = 0.0, A2i = 0.0, A3r = 0.0, A3i = 0.0;
#define FSTAT_BIN_STEP(d)                                                                            \
        {                                                                                            \
            A0r = fma((d).x, Er, fma(-(d).y, Ei, A0r));   /* A_0 += q,  q = dw' E (never formed) */ \
            A0i = fma((d).x, Ei, fma((d).y, Er, A0i));                                               \
            A1r += A0r; A1i += A0i;                                                                  \
            A2r += A1r; A2i += A1i;                                                                  \
            A3r += A2r; A3i += A2i;                                                                  \
            const double er = fma(Er, Rr, -Ei * Ri);                                                 \
            Ei = fma(Er, Ri, Ei * Rr);                                                               \
            Er = er;                                                                                 \
            const double rr = fma(Rr, Qr, -Ri * Qi);                                                 \
            Ri = fma(Rr, Qi, Ri * Qr);                                                               \
            Rr = rr;                                                                                 \
        }
        int b = 0;
#pragma unroll 2
        for (; b + 4 <= nb; b += 4) {
            const double2 d0 = tp[b], d1 = tp[b + 1], d2 = tp[b + 2], d3 = tp[b + 3];
            FSTAT_BIN_STEP(d0)
            FSTAT_BIN_STEP(d1)
            FSTAT_BIN_STEP(d2)
            FSTAT_BIN_STEP(d3)
            const double qq = fma(Qr, Cr, -Qi * Ci);
            Qi = fma(Qr, Ci, Qi * Cr);
            Qr = qq;
        }
        for (; b < nb; ++b) {
            const double2 d0 = tp[b];
            FSTAT_BIN_STEP(d0)
        }
#undef FSTAT_BIN_STEP

        // ---- the slow factors of this interval: node values of T'_+, T'_x at t = -2 .. 3 (the economised cubic through
        // them is applied inside the sums, never formed)
        double vpr[6], vpi[6], vcr[6], vci[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const int sl = (s_base + k) % kWinNodes;
            vpr[k] = sm.win[sl][1][tid]; vpi[k] = sm.win[sl][2][tid];
            vcr[k] = sm.win[sl][3][tid]; vci[k] = sm.win[sl][4][tid];
        }
        if (seg_start) {
            seg_start = false;
            const double n2 = fma(vpr[2], vpr[2], vpi[2] * vpi[2]), x2 = fma(vcr[2], vcr[2], vci[2] * vci[2]);
            const bool use = n2 > 1e-6 * x2;                                  // else T'_+ ~ 0 there: keep u_x
            const double inv = use ? 1.0 / n2 : 0.0;
            c_re = fma(vcr[2], vpr[2], vci[2] * vpi[2]) * inv;               // T'_x conj(T'_+) / |T'_+|^2 at node "0"
            c_im = fma(vci[2], vpr[2], -vcr[2] * vpi[2]) * inv;
        }
#pragma unroll
        for (int k = 0; k < 6; ++k) {                                        // node values of T'_x - c T'_+
            vcr[k] -= fma(c_re, vpr[k], -c_im * vpi[k]);
            vci[k] -= fma(c_re, vpi[k], c_im * vpr[k]);
        }
        // ---- z_P += sum_i conj(T'_P(i)) q_i = sum_k conj(v^P_k) B_k
        {
            const double A[8] = {A0r, A0i, A1r, A1i, A2r, A2i, A3r, A3i};
            double Br[6], Bi[6];
            subblock_weights(A, rS, (double)(j1 - node0), Br, Bi);
            z_from_nodes(vpr, vpi, Br, Bi, acc[0], acc[1]);
            z_from_nodes(vcr, vci, Br, Bi, acc[2], acc[3]);
        }
        // ---- m_PQ += (W v^P) . conj(W v^Q)   (W = L^T E of this sub-block: G = L L^T its Gram matrix)
        {
            double mpp, mcc, mre, mim;
            gram_forms(gram, vpr, vpi, vcr, vci, mpp, mcc, mre, mim);
            acc[4] += mpp; acc[5] += mcc; acc[6] += mre; acc[7] += mim;
            gram += kNW;
        }
        if (j1 == seg_hi) {                                  // segment finished: flush its eight sums
            double *out = a.partial + ((int64_t)cur_seg * kNPartial) * a.P_pad + p * a.part_sp;
#pragma unroll
            for (int j = 0; j < kNAcc; ++j) { out[(int64_t)j * a.part_sk] = acc[j]; acc[j] = 0.0; }
            out[(int64_t)8 * a.part_sk] = c_re;
            out[(int64_t)9 * a.part_sk] = c_im;
            seg_start = true;
            ++cur_seg;
            if (cur_seg < run_end) seg_hi = a.seg_edge[cur_seg + 1];
        }
        if (j1 == node0 + (1 << sh)) ++m;                    // node interval finished
        j0 = j1;
    }
    g0 += n_tiles;
    seg = run_end;
  }
}

__global__ void __launch_bounds__(kThreads, 4) fstat_fast_kernel(const __grid_constant__ FastArgs a)
{
    fast_kernel_body<false>(a);
}

// the same with the A / E / T response at the nodes (row f4, reading A28)
__global__ void __launch_bounds__(kThreads, 4) fstat_fast_aet_kernel(const __grid_constant__ FastArgs a)
{
    fast_kernel_body<true>(a);
}

cudaError_t fast_kernel_configure()
{
    cudaError_t e = cudaFuncSetAttribute(fstat_fast_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(FastSmem));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(fstat_fast_aet_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)sizeof(FastSmem));
}

cudaError_t launch_fast(const FastArgs &a, cudaStream_t st)
{
    const int64_t n_chunks = a.chunk_count > 0 ? a.chunk_count : (a.n_seg + a.segs_per_cta - 1) / a.segs_per_cta;
    const int64_t n_cta = (int64_t)a.n_groups * n_chunks;
    if (a.aet) fstat_fast_aet_kernel<<<(unsigned)n_cta, kThreads, sizeof(FastSmem), st>>>(a);
    else fstat_fast_kernel<<<(unsigned)n_cta, kThreads, sizeof(FastSmem), st>>>(a);
    return cudaGetLastError();
}

}  // namespace fstat
