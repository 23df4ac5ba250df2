// fstat_fastband.cu -- SURVEY row f2 (the paper's own segment limits) through the INTERPOLATING
// kernel, with per-THREAD partition edges.
//
// Every template (thread) has its own band [k_lo, k_hi) and its own N_seg partitions of it (reading A26), but all
// 128 threads of a CTA still walk the same bins of the same work segment, read the same folded-data tiles
// (shared-memory broadcast) and use the same node intervals.  What differs per thread is WHERE its running sums
// are cut:
//   * the stride selection caps the stride S of a work item at the shortest partition of its particle group, so a
//     node interval holds at most ONE edge ("cut") of any thread;
//   * in the per-bin loop a thread snapshots its four complex running sums A_0..A_3 at its cut (one warp vote per
//     4-bin run; the 4 x STS.128 are executed only in the runs that hold a cut of some lane);
//   * in the per-interval code the piece in front of the cut is  z = sum_n conj(c_n(U_cut)) A_n^snap  (the Newton
//     coefficients of the same cubic re-expanded at the cut) and  m_PQ = y^P G^pre y^Q  with G^pre a plan-time PREFIX
//     Gram matrix (one per level and 8-bin lattice cell; the <= 7 bins between the lattice and the cut are added
//     directly from the cubic), and the piece behind the cut is the interval's total minus it;
//   * a partition that opens and closes inside one work segment is finished in the thread: 2 F_k = z^H G^-1 z (and,
//     on request, the amplitudes a = M^-1 N) written at once.  Only the fragments at the two ends of a work segment
//     go to memory (head / tail records, ten doubles each) and are stitched by band_stitch_kernel (fstat_band.cu).
// No per-cell records, no full-model pieces, no cells epilogue: the workspace is O(P x work segments).
//
// Inner products: PAPER.md:66 Eq. 4, :89-91 Eq. 8-9, :117 Eq. 12.  Template: :397-405 Eq. A1-A3, :206-229
// Eq. 17-20 (N = 0).  Segment limits: :122 (reading A26).
#include "fstat_device.cuh"
#include "fstat_direct.cuh"
#include "fstat_fast.cuh"
#include "fstat_internal.h"
#include "fstat_model.cuh"

#include <math.h>

namespace fstat {

// =================================================================================================
// plan time (first band call): prefix Gram matrices.  pgram[level][k] = sum over the bins i of node interval
// m = 8 k >> (3 + level) with i < 8 (k + 1) of  w'_i l_a(i) l_b(i)  (upper triangle, Lagrange basis of the interval's
// four nodes): the Gram matrix of the interval's bins up to the END of 8-bin lattice cell k.  The entry of an
// interval's last cell is the interval's total.  One thread per node interval.
// =================================================================================================
__global__ void build_prefix_gram_kernel(const double2 *__restrict__ fw, int64_t n_bins, int level,
                                         double *__restrict__ pgram)
{
    const int S = kMinStride << level;
    const int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t b0 = m * S;
    if (b0 >= n_bins) return;
    const int64_t b1 = (b0 + S < n_bins) ? b0 + S : n_bins;
    const double rS = 1.0 / (double)S;
    double g[kNGram];
#pragma unroll
    for (int j = 0; j < kNGram; ++j) g[j] = 0.0;
    for (int64_t i = b0; i < b1; ++i) {
        const double wi = fw[i].y;
        double l[4];
        lagrange4((double)(i - b0) * rS, l);
        int j = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a; b < 4; ++b) g[j++] += wi * l[a] * l[b];
        if (((i + 1) & (kMinStride - 1)) == 0 || i + 1 == b1) {
            double *out = pgram + (i >> kLevel0Shift) * kNGram;
#pragma unroll
            for (int q = 0; q < kNGram; ++q) out[q] = g[q];
        }
    }
}

cudaError_t launch_build_prefix_gram(const double *fw, int64_t n_bins, int level, double *pgram, cudaStream_t st)
{
    const int S = kMinStride << level;
    const int64_t n_int = (n_bins + S - 1) / S;
    const int nt = 128;
    build_prefix_gram_kernel<<<(unsigned)((n_int + nt - 1) / nt), nt, 0, st>>>(reinterpret_cast<const double2 *>(fw), n_bins, level, pgram);
    return cudaGetLastError();
}

// =================================================================================================
// the kernel
// =================================================================================================
constexpr int kBandStages = 3;

struct __align__(16) BandSmem {
    double2 tile[kBandStages][kFastTile];      // folded data, 512-bin tiles (TMA bulk copies)
    double win[kWinNodes][kNSlow][kThreads];   // per-thread ring of the last six node values
    double2 snap[4][kThreads];                 // A_0..A_3 of a thread at its cut
    uint64_t full[kBandStages];
    uint32_t released[kBandStages];            // warps that have left the tile in this stage
};

// monomial coefficients in s = bin - node0 of the cubic through y0..y3 at t = -1, 0, 1, 2 (t = s / S)
__device__ __forceinline__ void cubic_mono(double y0, double y1, double y2, double y3, double rS, double (&m)[4])
{
    const double d0 = y0 - y1, d2 = y2 - y1, d3 = y3 - y1;
    const double a1 = fma(d0, -1.0 / 3.0, fma(d3, -1.0 / 6.0, d2));
    const double a2 = 0.5 * (d0 + d2);
    const double a3 = fma(d2, -0.5, (d3 - d0) * (1.0 / 6.0));
    m[0] = y1;
    m[1] = a1 * rS;
    m[2] = a2 * rS * rS;
    m[3] = a3 * rS * rS * rS;
}

// Newton-basis coefficients (basis C(u + n - 1, n), u = U - s) of that cubic for running sums that end U bins
// after node 0 (the same arithmetic as newton_coefs of fstat_fast.cuh, split so that one cubic serves two ends)
__device__ __forceinline__ void newton_from_mono(const double (&m)[4], double U, double (&c)[4])
{
    const double e0 = fma(U, fma(U, fma(U, m[3], m[2]), m[1]), m[0]);
    const double e1 = -fma(U, fma(3.0 * U, m[3], 2.0 * m[2]), m[1]);
    const double e2 = fma(3.0 * U, m[3], m[2]);
    const double e3 = -m[3];
    c[0] = e0;
    c[1] = e1 - e2 + e3;
    c[2] = fma(-6.0, e3, 2.0 * e2);
    c[3] = 6.0 * e3;
}

__device__ __forceinline__ double horner3(const double (&m)[4], double s)
{
    return fma(s, fma(s, fma(s, m[3], m[2]), m[1]), m[0]);
}

// z += sum_n conj(c_n) A_n  for one polarisation: c = cr + i ci, A_n = (Ar[n], Ai[n])
__device__ __forceinline__ void z_from_sums(const double (&cr)[4], const double (&ci)[4], const double (&Ar)[4],
                                            const double (&Ai)[4], double &zr, double &zi)
{
    zr = fma(cr[0], Ar[0], fma(ci[0], Ai[0], fma(cr[1], Ar[1], fma(ci[1], Ai[1],
         fma(cr[2], Ar[2], fma(ci[2], Ai[2], fma(cr[3], Ar[3], ci[3] * Ai[3])))))));
    zi = fma(cr[0], Ai[0], fma(-ci[0], Ar[0], fma(cr[1], Ai[1], fma(-ci[1], Ar[1],
         fma(cr[2], Ai[2], fma(-ci[2], Ar[2], fma(cr[3], Ai[3], -ci[3] * Ar[3])))))));
}

// m_PQ = y^P G conj(y^Q) for the 4x4 symmetric G given by its upper triangle g[10]: m = (m_pp, m_cc, Re m_pc, Im m_pc)
__device__ __forceinline__ void gram_quad(const double (&g)[kNGram], const double (&ypr)[4], const double (&ypi)[4],
                                          const double (&ycr)[4], const double (&yci)[4], double (&m)[4])
{
    const double G[4][4] = {{g[0], g[1], g[2], g[3]}, {g[1], g[4], g[5], g[6]}, {g[2], g[5], g[7], g[8]}, {g[3], g[6], g[8], g[9]}};
    double mpp = 0.0, mcc = 0.0, mre = 0.0, mim = 0.0;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const double vpr = fma(G[r][0], ypr[0], fma(G[r][1], ypr[1], fma(G[r][2], ypr[2], G[r][3] * ypr[3])));
        const double vpi = fma(G[r][0], ypi[0], fma(G[r][1], ypi[1], fma(G[r][2], ypi[2], G[r][3] * ypi[3])));
        const double vcr = fma(G[r][0], ycr[0], fma(G[r][1], ycr[1], fma(G[r][2], ycr[2], G[r][3] * ycr[3])));
        const double vci = fma(G[r][0], yci[0], fma(G[r][1], yci[1], fma(G[r][2], yci[2], G[r][3] * yci[3])));
        mpp = fma(ypr[r], vpr, fma(ypi[r], vpi, mpp));
        mcc = fma(ycr[r], vcr, fma(yci[r], vci, mcc));
        mre = fma(ypr[r], vcr, fma(ypi[r], vci, mre));      // Re sum y^+ conj(v^x)
        mim = fma(ypi[r], vcr, fma(-ypr[r], vci, mim));     // Im
    }
    m[0] = mpp; m[1] = mcc; m[2] = mre; m[3] = mim;
}

__device__ __forceinline__ void load_gram(const double *__restrict__ gp, double (&g)[kNGram])
{
    const double2 *p2 = reinterpret_cast<const double2 *>(gp);
    const double2 g01 = p2[0], g23 = p2[1], g45 = p2[2], g67 = p2[3], g89 = p2[4];
    g[0] = g01.x; g[1] = g01.y; g[2] = g23.x; g[3] = g23.y; g[4] = g45.x;
    g[5] = g45.y; g[6] = g67.x; g[7] = g67.y; g[8] = g89.x; g[9] = g89.y;
}

// F_k (and the amplitudes) of a finished partition, written through the slot -> particle map
// 2 F_k as two_F (fstat_direct.cuh) with the two divisions replaced by rcp_fast (relative error ~1e-16: the hardware
// seed and two Newton steps, no slow path): this runs inside the interpolating kernel, once per partition and thread
__device__ __forceinline__ double two_F_inline(const double (&v)[kNAcc])
{
    const double zpr = v[0], zpi = v[1], zcr = v[2], zci = v[3];
    const double mpp = v[4], mcc = v[5], mr = v[6], mi = v[7];
    double twoF = 0.0;
    if (mpp > 0.0) {
        const double inv = rcp_fast(mpp);
        twoF = (zpr * zpr + zpi * zpi) * inv;
        const double cr = mr * inv, ci = mi * inv;                      // m_pc / m_pp
        const double schur = mcc - (mr * mr + mi * mi) * inv;
        if (schur > 1e-13 * mcc) {
            const double yr = zcr - (cr * zpr - ci * zpi);
            const double yi = zci - (cr * zpi + ci * zpr);
            twoF += (yr * yr + yi * yi) * rcp_fast(schur);
        }
    } else if (mcc > 0.0) {
        twoF = (zcr * zcr + zci * zci) * rcp_fast(mcc);
    }
    return twoF;
}

__device__ __forceinline__ void finish_partition(const double (&v)[kNAcc], double c_re, double c_im, int64_t idx,
                                                 double *__restrict__ Fk, double *__restrict__ amp)
{
    Fk[idx] = 0.5 * two_F_inline(v);
    if (amp != nullptr) {
        double a1, a2, a3, a4;
        solve_amplitudes(v, c_re, c_im, a1, a2, a3, a4);
        amp[4 * idx + 0] = a1; amp[4 * idx + 1] = a2; amp[4 * idx + 2] = a3; amp[4 * idx + 3] = a4;
    }
}

// 168 registers, no spills in the per-bin loop, 3 CTAs per SM (at 128 registers / 4 CTAs the per-interval code spills
// ~400 bytes and the call is 4 % slower)
__global__ void __launch_bounds__(kThreads, 3) fstat_fastband_kernel(const __grid_constant__ FastBandArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    BandSmem &sm = *reinterpret_cast<BandSmem *>(smem_raw);

    const int tid = threadIdx.x;
    const int grp = blockIdx.x % a.n_groups;
    const int seg = blockIdx.x / a.n_groups;
    const int lvl = a.level[(int64_t)grp * a.n_seg + seg];
    if (lvl < 0) return;                                     // CTA-uniform: skipped (-2) or left to the direct kernel (-1)
    const int64_t p = (int64_t)grp * kThreads + tid;         // slot, < P_pad by construction
    const double *cf = a.coef + p;
    const double2 *dwp = reinterpret_cast<const double2 *>(a.dwp);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kBandStages; ++s) { mbar_init(&sm.full[s], 1); sm.released[s] = 0u; }
        mbar_fence_init();
    }
    __syncthreads();

    const int sh = kLevel0Shift + lvl;
    const double rS = 1.0 / (double)(1 << sh);
    const int lo = a.seg_edge[seg], hi = a.seg_edge[seg + 1];     // lo is a multiple of 512
    const int t_first = lo >> kFastTileShift;
    const int n_tiles = ((hi - 1) >> kFastTileShift) - t_first + 1;

    auto issue_tile = [&](int t) {
        const int slot = t % kBandStages;
        const int b0 = max(lo, (t_first + t) << kFastTileShift), b1 = min(hi, (t_first + t + 1) << kFastTileShift);
        const uint32_t bytes = (uint32_t)(b1 - b0) * (uint32_t)sizeof(double2);
        mbar_expect_tx(&sm.full[slot], bytes);
        tma_load_1d(&sm.tile[slot][b0 & (kFastTile - 1)], dwp + b0, bytes, &sm.full[slot]);
    };
    if (tid == 0)
        for (int s = 0; s < kBandStages && s < n_tiles; ++s) issue_tile(s);

    // ---- this thread's partitions (reading A26): j = the partition bin `lo` belongs to (-1: below the band, N: above
    // it or not evaluated here), cut = the bin at which it closes
    const int32_t N = a.b.N, C = a.b.C;
    const int32_t q_lo = (a.b.band_lo[p] + C / 2) / C, D = (a.b.band_hi[p] + C / 2) / C - q_lo;
    int32_t j = N, cut = INT32_MAX;
    bool opened = false;                                     // partition j started inside this work segment (or exactly at lo)
    int32_t my_lo = INT32_MAX, my_hi = 0;                    // this thread's band (empty: not evaluated by this kernel)
    if (a.b.valid[p] != 0 && band_fast_eligible(D, N, C)) {
        const int32_t e0 = band_edge(0, q_lo, D, N, C, a.b.n_bins), eN = band_edge(N, q_lo, D, N, C, a.b.n_bins);
        my_lo = e0;
        my_hi = eN;
        if (lo < eN && hi > e0) {
            if (lo < e0) { j = -1; cut = e0; }
            else {
                const int64_t cells = (int64_t)(lo / C) - q_lo;           // largest j with e_j <= lo
                int64_t jj = ((cells + 1) * N + D - 1) / D - 1;
                if (jj > N - 1) jj = N - 1;
                j = (int32_t)jj;
                while (j + 1 < N && band_edge(j + 1, q_lo, D, N, C, a.b.n_bins) <= lo) ++j;
                while (j > 0 && band_edge(j, q_lo, D, N, C, a.b.n_bins) > lo) --j;
                cut = band_edge(j + 1, q_lo, D, N, C, a.b.n_bins);
                opened = band_edge(j, q_lo, D, N, C, a.b.n_bins) == lo;
            }
        }
    }
    // the edges after `cut` follow by stepping floor(j D / N) incrementally: e_(j+1) from e_j costs two additions, not a
    // 64-bit division (cut = min(C (q_lo + eq), n_bins), eq = floor((j + 1) D / N), er the remainder)
    const int32_t dq = D > 0 ? D / N : 0, dr = D > 0 ? D % N : 0;
    int32_t eq = 0, er = 0;
    if (j < N) {
        const int64_t jd = (int64_t)(j + 1) * D;
        eq = (int32_t)(jd / N);
        er = (int32_t)(jd - (int64_t)eq * N);
    }
    // The node intervals of this work segment that hold an in-band bin of some lane of this WARP: [w_lo, w_hi).  The
    // slots are ranked by the position of the band, so the bands of the 32 lanes of a warp nearly coincide while the
    // four warps of a CTA are spread over the group's union: a warp skips the intervals outside its own range
    // (nothing of what it would accumulate there is kept) and starts its node ring where it enters.
    const int S = 1 << sh;
    int w_lo = __reduce_min_sync(0xffffffffu, my_lo), w_hi = __reduce_max_sync(0xffffffffu, my_hi);
    if (w_hi <= 0) w_hi = -1;                                // no lane of this warp is evaluated here
    w_lo = max(lo, w_lo & ~(S - 1));
    w_hi = min(hi, w_hi + 1);                                // + 1: an edge AT w_hi closes its partition in the interval that starts there
    const int32_t particle = a.b.perm[p];
    double *rec_head = a.b.rec + ((int64_t)(seg * 2 + 0) * kNPartial) * a.P_pad + p;
    double *rec_tail = a.b.rec + ((int64_t)(seg * 2 + 1) * kNPartial) * a.P_pad + p;

    // linear phase term 2 pi f t_c in quarter turns: per-bin advance, reduced mod 4
    const double c0 = cf[0];
    const double slope = mulmod4(c0, a.df);

    double acc[kNAcc];
#pragma unroll
    for (int q = 0; q < kNAcc; ++q) acc[q] = 0.0;
    bool need_basis = true;
    double c_re = 0.0, c_im = 0.0;
    bool ring_ok = false;                                    // the node ring holds nodes m-2 .. m+2 of the next interval
    uint32_t st_bins = 0, st_int = 0, st_cut = 0;            // this warp's work, for the roofline of the bench line

  for (int tl = 0; tl < n_tiles; ++tl) {
    const int tb0 = max(lo, (t_first + tl) << kFastTileShift), tb1 = min(hi, (t_first + tl + 1) << kFastTileShift);
    // every warp waits for every tile, also those it skips: a slot is re-armed only after all phases of its barrier
    // have been observed (a warp that skipped a phase would mistake the parity of a later one)
    mbar_wait(&sm.full[tl % kBandStages], (uint32_t)((tl / kBandStages) & 1));
    if (tb0 < w_hi && tb1 > w_lo) {                          // warp-uniform
      for (int j0 = max(tb0, w_lo); j0 < min(tb1, w_hi); j0 += S) {
        const int m = j0 >> sh;
        const int node0 = j0;                                // sub-blocks are whole node intervals (cut short only by the grid end)
        const int j1 = min(hi, node0 + S);
        const int s_base = (m - 2 + kWinNodes) % kWinNodes;  // ring slot of node m-2
        // ---- node ring: (psi_nl, T'_+ re, im, T'_x re, im) at the last six nodes, slot = (node + 6) % 6: the new node
        // m+3, and nodes m-2 .. m+2 where the warp enters its range
        const double fnode = a.node[((int64_t)kNodePad + ((int64_t)m << lvl)) * kTabW + T_F];
        {
            double c[kNCoef];
            load_coef(cf, a.P_pad, c);
            for (int k = ring_ok ? 3 : -2; k <= 3; ++k) {
                const double2 *row = reinterpret_cast<const double2 *>(
                    a.node + ((int64_t)kNodePad + ((int64_t)(m + k) * (1 << lvl))) * kTabW);
                double v0, v1, v2, v3, v4;
                model_eval(row, c, a.orb, v0, v1, v2, v3, v4);
                const int slot = (m + k + kWinNodes) % kWinNodes;
                sm.win[slot][0][tid] = v0; sm.win[slot][1][tid] = v1; sm.win[slot][2][tid] = v2;
                sm.win[slot][3][tid] = v3; sm.win[slot][4][tid] = v4;
            }
            ring_ok = true;
        }
        // ---- carrier phase: economised cubic + exact linear term, as forward differences (s0 = 0: j0 is the node)
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
            t = G0;
            D1 = G3 + G2 + G1;
            D2 = fma(6.0, G3, 2.0 * G2);
            D3 = 6.0 * G3;
        }
        const double2 *tp = &sm.tile[tl % kBandStages][j0 & (kFastTile - 1)];
        const int nb = j1 - j0;
        const uint32_t cut_rel = (uint32_t)(cut - j0);       // >= nb: no cut of this thread in this interval
        st_bins += (uint32_t)nb;
        st_int += 1u;
        st_cut += __any_sync(0xffffffffu, cut_rel < (uint32_t)nb) ? 1u : 0u;

        // ---- per bin: the same recurrences as fstat_fast_kernel (19 FP64 instructions per bin); a thread whose cut
        // falls into a 4-bin run stores A_0..A_3 as they stand IN FRONT of its cut bin
        double Er, Ei, Rr, Ri, Qr, Qi, Cr, Ci;
        sincos_qt(t, Ei, Er);
        sincos_qt(fma(-1.25, D3, D1), Ri, Rr);
        sincos_qt_small(fma(1.5, D3, D2), Qi, Qr);
        sincos_qt_small(4.0 * D3, Ci, Cr);
        double A0r = 0.0, A0i = 0.0, A1r = 0.0, A1i = 0.0, A2r = 0.0, A2i = 0.0, A3r = 0.0, A3i = 0.0;
#define FSTAT_BIN_STEP(d)                                                                            \
        {                                                                                            \
            A0r = fma((d).x, Er, fma(-(d).y, Ei, A0r));                                              \
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
#define FSTAT_SNAP()                                                                                 \
        {                                                                                            \
            sm.snap[0][tid] = make_double2(A0r, A0i); sm.snap[1][tid] = make_double2(A1r, A1i);      \
            sm.snap[2][tid] = make_double2(A2r, A2i); sm.snap[3][tid] = make_double2(A3r, A3i);      \
        }
        // which 4-bin runs hold a cut of some lane of this warp: one bit per 2^msh runs, warp-uniform
        int b = 0;
        for (; b + 4 <= nb; b += 4) {
            const double2 d0 = tp[b], d1 = tp[b + 1], d2 = tp[b + 2], d3 = tp[b + 3];
            const uint32_t dc = cut_rel - (uint32_t)b;
            if (__any_sync(0xffffffffu, dc < 4u)) {          // warp-uniform: some lane cuts inside this run
                if (dc == 0u) FSTAT_SNAP()
                FSTAT_BIN_STEP(d0)
                if (dc == 1u) FSTAT_SNAP()
                FSTAT_BIN_STEP(d1)
                if (dc == 2u) FSTAT_SNAP()
                FSTAT_BIN_STEP(d2)
                if (dc == 3u) FSTAT_SNAP()
                FSTAT_BIN_STEP(d3)
            } else {
                FSTAT_BIN_STEP(d0)
                FSTAT_BIN_STEP(d1)
                FSTAT_BIN_STEP(d2)
                FSTAT_BIN_STEP(d3)
            }
            const double qq = fma(Qr, Cr, -Qi * Ci);
            Qi = fma(Qr, Ci, Qi * Cr);
            Qr = qq;
        }
        for (; b < nb; ++b) {                                // (only at the end of the grid)
            const double2 d0 = tp[b];
            if (cut_rel == (uint32_t)b) FSTAT_SNAP()
            FSTAT_BIN_STEP(d0)
        }
#undef FSTAT_BIN_STEP
#undef FSTAT_SNAP

        // ---- the slow factors of this interval: economised cubic of T'_+, T'_x as values at t = -1, 0, 1, 2
        double ypr[4], ypi[4], ycr[4], yci[4];
        {
            double v[6], yref;
#pragma unroll
            for (int k = 0; k < 6; ++k) v[k] = sm.win[(s_base + k) % kWinNodes][1][tid];
            economise(v, yref, ypr);
#pragma unroll
            for (int q = 0; q < 4; ++q) ypr[q] += yref;
#pragma unroll
            for (int k = 0; k < 6; ++k) v[k] = sm.win[(s_base + k) % kWinNodes][2][tid];
            economise(v, yref, ypi);
#pragma unroll
            for (int q = 0; q < 4; ++q) ypi[q] += yref;
#pragma unroll
            for (int k = 0; k < 6; ++k) v[k] = sm.win[(s_base + k) % kWinNodes][3][tid];
            economise(v, yref, ycr);
#pragma unroll
            for (int q = 0; q < 4; ++q) ycr[q] += yref;
#pragma unroll
            for (int k = 0; k < 6; ++k) v[k] = sm.win[(s_base + k) % kWinNodes][4][tid];
            economise(v, yref, yci);
#pragma unroll
            for (int q = 0; q < 4; ++q) yci[q] += yref;
        }
        if (need_basis) {                                    // basis of the sums (hazard H3): (u_+, u_x - c u_+)
            need_basis = false;
            choose_basis(ypr[1], ypi[1], ycr[1], yci[1], c_re, c_im);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {                        // node values of T'_x - c T'_+
            ycr[q] -= fma(c_re, ypr[q], -c_im * ypi[q]);
            yci[q] -= fma(c_re, ypi[q], c_im * ypr[q]);
        }
        // ---- the whole sub-block [j0, j1): z = sum_n conj(c_n) A_n,  m = y G y
        double mpr[4], mpi[4], mcr[4], mci[4];               // monomial coefficients of the four real cubics
        cubic_mono(ypr[0], ypr[1], ypr[2], ypr[3], rS, mpr);
        cubic_mono(ypi[0], ypi[1], ypi[2], ypi[3], rS, mpi);
        cubic_mono(ycr[0], ycr[1], ycr[2], ycr[3], rS, mcr);
        cubic_mono(yci[0], yci[1], yci[2], yci[3], rS, mci);
        double tot[kNAcc];
        {
            const double U = (double)(j1 - node0);
            const double Ar[4] = {A0r, A1r, A2r, A3r}, Ai[4] = {A0i, A1i, A2i, A3i};
            double cr[4], ci[4];
            newton_from_mono(mpr, U, cr);
            newton_from_mono(mpi, U, ci);
            z_from_sums(cr, ci, Ar, Ai, tot[0], tot[1]);
            newton_from_mono(mcr, U, cr);
            newton_from_mono(mci, U, ci);
            z_from_sums(cr, ci, Ar, Ai, tot[2], tot[3]);
            double g[kNGram], mm[4];
            const int64_t cell_last = ((int64_t)(j1 - 1)) >> kLevel0Shift;       // the interval's last lattice cell
            load_gram(a.pgram[lvl] + cell_last * kNGram, g);
            gram_quad(g, ypr, ypi, ycr, yci, mm);
            tot[4] = mm[0]; tot[5] = mm[1]; tot[6] = mm[2]; tot[7] = mm[3];
        }
        if (cut_rel >= (uint32_t)nb) {                       // no edge of this thread in the interval
#pragma unroll
            for (int q = 0; q < kNAcc; ++q) acc[q] += tot[q];
        } else {
            // ---- the piece [j0, cut) in front of the cut ...
            double pc[kNAcc];
            {
                const double U = (double)(cut - node0);
                const double2 s0 = sm.snap[0][tid], s1 = sm.snap[1][tid], s2 = sm.snap[2][tid], s3 = sm.snap[3][tid];
                const double Ar[4] = {s0.x, s1.x, s2.x, s3.x}, Ai[4] = {s0.y, s1.y, s2.y, s3.y};
                double cr[4], ci[4];
                newton_from_mono(mpr, U, cr);
                newton_from_mono(mpi, U, ci);
                z_from_sums(cr, ci, Ar, Ai, pc[0], pc[1]);
                newton_from_mono(mcr, U, cr);
                newton_from_mono(mci, U, ci);
                z_from_sums(cr, ci, Ar, Ai, pc[2], pc[3]);
                // prefix Gram matrix up to the NEAREST point of the 8-bin lattice (or the interval's end), then the
                // <= 4 bins between that point and the cut added or taken away directly from the cubic
                double mm[4] = {0.0, 0.0, 0.0, 0.0};
                const int uc = cut - node0;
                const int u8 = min((uc + kMinStride / 2) & ~(kMinStride - 1), j1 - node0);
                if (u8 > 0) {
                    double g[kNGram];
                    load_gram(a.pgram[lvl] + ((int64_t)((node0 + u8 - 1) >> kLevel0Shift)) * kNGram, g);
                    gram_quad(g, ypr, ypi, ycr, yci, mm);
                }
                const double sgn = uc >= u8 ? 1.0 : -1.0;
                for (int i = node0 + min(uc, u8); i < node0 + max(uc, u8); ++i) {
                    const double s = (double)(i - node0), wi = sgn * a.fw[2 * (int64_t)i + 1];
                    const double pr = horner3(mpr, s), pi = horner3(mpi, s), xr = horner3(mcr, s), xi = horner3(mci, s);
                    mm[0] = fma(wi, fma(pr, pr, pi * pi), mm[0]);
                    mm[1] = fma(wi, fma(xr, xr, xi * xi), mm[1]);
                    mm[2] = fma(wi, fma(pr, xr, pi * xi), mm[2]);
                    mm[3] = fma(wi, fma(pi, xr, -pr * xi), mm[3]);
                }
                pc[4] = mm[0]; pc[5] = mm[1]; pc[6] = mm[2]; pc[7] = mm[3];
            }
            // ... closes partition j
            if (j >= 0) {
#pragma unroll
                for (int q = 0; q < kNAcc; ++q) acc[q] += pc[q];
                if (opened) {
                    finish_partition(acc, c_re, c_im, (int64_t)particle * N + j, a.b.Fk, a.b.amp);
                } else {                                     // it began in an earlier work segment: head fragment
#pragma unroll
                    for (int q = 0; q < kNAcc; ++q) rec_head[(int64_t)q * a.P_pad] = acc[q];
                    rec_head[(int64_t)8 * a.P_pad] = c_re;
                    rec_head[(int64_t)9 * a.P_pad] = c_im;
                }
            }
            // ---- ... and the piece behind it opens partition j + 1, in a basis of its own
            ++j;
            opened = true;
            if (j >= N) { j = N; cut = INT32_MAX; }
            else {
                eq += dq;
                er += dr;
                if (er >= N) { er -= N; ++eq; }
                const int64_t e = (int64_t)C * ((int64_t)q_lo + eq);
                cut = (int32_t)(e < (int64_t)a.b.n_bins ? e : (int64_t)a.b.n_bins);
            }
            if (cut < j1) atomicOr(a.b.err, 1u);               // (a second edge in one interval: excluded by the stride cap)
            double t10[kNPartial];
#pragma unroll
            for (int q = 0; q < kNAcc; ++q) t10[q] = tot[q] - pc[q];
            t10[8] = c_re; t10[9] = c_im;
            const double xr = ycr[1] + fma(c_re, ypr[1], -c_im * ypi[1]);       // raw T'_x at node 0
            const double xi = yci[1] + fma(c_re, ypi[1], c_im * ypr[1]);
            choose_basis(ypr[1], ypi[1], xr, xi, c_re, c_im);
#pragma unroll
            for (int q = 0; q < kNAcc; ++q) acc[q] = 0.0;
            add_record(t10, c_re, c_im, acc);
        }
      }
    }
    // The warps are not held together tile by tile: a warp that has left this tile says so, and the LAST of the four to
    // leave re-arms the stage with the tile kBandStages further on.  A warp runs ahead of the slowest one by up to
    // kBandStages tiles; nobody waits for anything but the data.
    __syncwarp();
    if ((tid & 31) == 0) {
        __threadfence_block();                               // this warp's reads of the tile come before its release
        const uint32_t old = atomicAdd(&sm.released[tl % kBandStages], 1u);
        if (old == (uint32_t)(kThreads / 32 - 1)) {
            atomicExch(&sm.released[tl % kBandStages], 0u);
            __threadfence_block();
            if (tl + kBandStages < n_tiles) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue_tile(tl + kBandStages);
            }
        }
    }
  }
    if ((tid & 31) == 0 && st_int > 0u && a.b.stats != nullptr) {
        atomicAdd(&a.b.stats[0], (unsigned long long)st_bins);
        atomicAdd(&a.b.stats[1], (unsigned long long)st_int);
        atomicAdd(&a.b.stats[2], (unsigned long long)st_cut);
        atomicAdd(&a.b.stats[3], 1ull);
    }
    // ---- what is left after the last edge.  Partition j either goes on in the next work segment (tail fragment) or
    // closes exactly at the end of this one (cut == hi): finished here if it also began here, else its closing fragment
    if (j >= 0 && j < N) {
        if (cut == hi && opened) {
            finish_partition(acc, c_re, c_im, (int64_t)particle * N + j, a.b.Fk, a.b.amp);
        } else {
            double *out = (cut == hi) ? rec_head : rec_tail;
#pragma unroll
            for (int q = 0; q < kNAcc; ++q) out[(int64_t)q * a.P_pad] = acc[q];
            out[(int64_t)8 * a.P_pad] = c_re;
            out[(int64_t)9 * a.P_pad] = c_im;
        }
    }
}

cudaError_t fastband_kernel_configure()
{
    return cudaFuncSetAttribute(fstat_fastband_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)sizeof(BandSmem));
}

cudaError_t launch_fastband(const FastBandArgs &a, cudaStream_t st)
{
    const int64_t n_cta = (int64_t)a.n_groups * a.n_seg;
    fstat_fastband_kernel<<<(unsigned)n_cta, kThreads, sizeof(BandSmem), st>>>(a);
    return cudaGetLastError();
}

}  // namespace fstat
