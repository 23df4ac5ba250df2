// fstat_band.cu -- SURVEY row f2: the semi-coherent F-statistic with the paper's OWN segment limits
// (PAPER.md:122): the number of segments is fixed for all templates, the outer limits are "the lowest and
// highest instantaneous frequencies occurring during the observation period in the template", i.e. the
// bins whose stationary time t_f (Eq. 20 :220) lies in [0, T_obs].  Partition edges therefore differ from
// particle to particle (reading A26 for where they fall on the grid):
//
//   band_kernel          k_lo = #{bins with t_f < 0}, k_hi = #{bins with t_f <= T_obs} per particle, by
//                        bisection over the per-bin table (t_f increases along the grid)
//
// The normal path is the interpolating kernel over CELLS of the grid: the cells are the (data-side) partitions of
// an internal plan, fstat_fast_kernel / fstat_main_kernel run unchanged and leave one record of sums per (cell,
// particle), the stride selection skips the cells no template of a group is in band for, and
//
//   band_cells_epilogue_kernel   adds, per particle and partition, the records of the cells between its edges
//                                (recentred basis, add_segment) and writes F_k [and the amplitudes a = M^-1 N]
//   band_fsum_kernel             F = sum_k F_k in a fixed order
//
// With edges on a lattice of C >= 32 bins the cells are the lattice.  Below that (default: edges at ANY bin) the
// cells are 64..512 bins wide and an edge may split a cell:
//
//   band_ragged_kernel           full model over the shorter piece of every cell an edge splits (the other piece
//                                is the cell's record minus it), and over every partition that holds no whole
//                                cell, edge to edge (for N_seg >= 128 the pieces go through piece_list_kernel /
//                                band_ragged_sorted_kernel: ordered by length, one list entry per thread)
//
// The first version of the row is kept as the full-size reference of the above (options.force_level == -1, or a
// grid too close to f = 0 for the node table):
//
//   fstat_band_kernel    the direct kernel (full model at every in-band bin) with per-THREAD partition edges: a
//                        partition that opens and closes inside one work segment is finished in the thread
//                        (2 F_k written at once); the fragment before the first edge and the one after the last
//                        edge of a work segment go to head / tail records
//   band_epilogue_kernel stitches head / tail records of consecutive work segments into the partitions that
//                        straddle them, writes their F_k, then F = sum_k F_k in a fixed order
#include "fstat_device.cuh"
#include "fstat_direct.cuh"
#include "fstat_internal.h"
#include "fstat_model.cuh"

#include <math.h>

namespace fstat {

// Orbital phase at t_f in quarter turns of a year, alpha_q = c10 + sum_j c_j D_j(f) (same FMA chain as
// model_eval); t_f = (alpha_q - 2 kappa / pi) year / 4.
__device__ __forceinline__ double tf_seconds(const double *__restrict__ row, const double (&c)[kNCoef], double kappa_qt)
{
    double alq = fma(c[2], row[T_D0 + 0], c[10]);
#pragma unroll
    for (int j = 1; j < 8; ++j) alq = fma(c[2 + j], row[T_D0 + j], alq);
    return (alq - kappa_qt) * (0.25 * kYear);
}

__global__ void __launch_bounds__(128) band_kernel(const double *__restrict__ table, const double *__restrict__ coef,
                                                   const int32_t *__restrict__ valid,
                                                   const int32_t *__restrict__ perm, int64_t P_pad, int32_t n_bins,
                                                   double T_obs, double kappa_qt, int32_t *__restrict__ band_lo,
                                                   int32_t *__restrict__ band_hi, int64_t *__restrict__ band_out)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;       // slot
    if (p >= P_pad) return;
    int32_t k_lo = 0, k_hi = 0;
    if (valid[p] != 0) {
        double c[kNCoef];
#pragma unroll
        for (int j = 0; j < kNCoef; ++j) c[j] = coef[(int64_t)j * P_pad + p];
        // first bin with t_f >= 0
        int32_t a = 0, b = n_bins;
        while (a < b) {
            const int32_t m = a + ((b - a) >> 1);
            if (tf_seconds(table + (int64_t)m * kTabW, c, kappa_qt) < 0.0) a = m + 1; else b = m;
        }
        k_lo = a;
        // first bin with t_f > T_obs
        b = n_bins;
        while (a < b) {
            const int32_t m = a + ((b - a) >> 1);
            if (tf_seconds(table + (int64_t)m * kTabW, c, kappa_qt) <= T_obs) a = m + 1; else b = m;
        }
        k_hi = a;
    }
    band_lo[p] = k_lo;
    band_hi[p] = k_hi;
    const int32_t q = perm[p];
    if (band_out != nullptr && q >= 0) {
        band_out[2 * (int64_t)q] = k_lo;
        band_out[2 * (int64_t)q + 1] = k_hi;
    }
}

// ---------------------------------------------------------------------------------------------------
// Main kernel.  Work item = (group of 128 slots) x (work segment of seg_len bins of the grid); persistent
// CTAs stride over the items and skip those no thread of the group is in band for.
// Thread state: j = the partition the current bin belongs to (-1 below the band, N above it), e_next = the
// bin at which partition j closes.  rec[(w * 2 + h) * 8 + i][slot], rec_idx[(w * 2 + h)][slot]: head (h = 0)
// and tail (h = 1) fragments of work segment w with the partition they belong to (-1: none).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) fstat_band_kernel(const __grid_constant__ BandArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    MainSmem &sm = *reinterpret_cast<MainSmem *>(smem_raw);

    const int tid = threadIdx.x;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&sm.full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    int g0 = 0;                                          // tiles consumed so far by this CTA (ring position)
    const int32_t N = a.n_seg, C = a.lattice;
    const int n_items = a.n_groups * a.n_wseg;

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int grp = item / a.n_wseg;
        const int w = item - grp * a.n_wseg;
        const int64_t p = (int64_t)grp * kThreads + tid;
        const int lo = w * a.seg_len, hi = min(a.n_bins, lo + a.seg_len);

        const int32_t k_lo = a.band_lo[p], k_hi = a.band_hi[p];
        const int32_t q_lo = (k_lo + C / 2) / C, D = (k_hi + C / 2) / C - q_lo;
        const int32_t e0 = band_edge(0, q_lo, D, N, C, a.n_bins), eN = band_edge(N, q_lo, D, N, C, a.n_bins);
        const bool active = (eN > e0) && (lo < eN) && (hi > e0);
        if (!__syncthreads_or(active ? 1 : 0)) continue;

        const int n_bins = hi - lo;
        const int n_tiles = (n_bins + kTileBins - 1) / kTileBins;
        const double *src = a.table + (int64_t)lo * kTabW;
        if (tid == 0) ring_prologue(sm, src, n_bins, n_tiles, g0);

        double c[kNCoef];
#pragma unroll
        for (int j = 0; j < kNCoef; ++j) c[j] = a.coef[(int64_t)j * a.P_pad + p];

        // the partition bin `lo` belongs to
        int32_t j, e_next;
        if (!active) { j = N; e_next = INT32_MAX; }
        else if (lo < e0) { j = -1; e_next = e0; }
        else {
            // largest j with e_j <= lo:  floor(j D / N) <= cells  <=>  j <= ceil((cells + 1) N / D) - 1
            const int64_t cells = (int64_t)(lo / C) - q_lo;
            int64_t jj = ((cells + 1) * N + D - 1) / D - 1;
            if (jj > N - 1) jj = N - 1;
            j = (int32_t)jj;
            while (j + 1 < N && band_edge(j + 1, q_lo, D, N, C, a.n_bins) <= lo) ++j;     // (never taken)
            while (j > 0 && band_edge(j, q_lo, D, N, C, a.n_bins) > lo) --j;
            e_next = band_edge(j + 1, q_lo, D, N, C, a.n_bins);
        }
        bool flushed = false;
        const int32_t particle = a.perm[p];
        double *rec_head = a.rec + ((int64_t)(w * 2 + 0) * kNAcc) * a.P_pad + p;
        double *rec_tail = a.rec + ((int64_t)(w * 2 + 1) * kNAcc) * a.P_pad + p;

        double acc[kNAcc];
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) acc[i] = 0.0;

        for (int t = 0; t < n_tiles; ++t) {
            const double *tile = ring_wait(sm, g0 + t);
            const int nb = min(kTileBins, n_bins - t * kTileBins);
            double in[kNAcc];
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) in[i] = 0.0;

#pragma unroll 1
            for (int b = 0; b < nb; ++b) {
                const int k = lo + t * kTileBins + b;
                while (k == e_next) {                                  // partition j closes in front of bin k
                    if (j >= 0) {
                        double v[kNAcc];
#pragma unroll
                        for (int i = 0; i < kNAcc; ++i) v[i] = acc[i] + in[i];
                        if (!flushed) {
#pragma unroll
                            for (int i = 0; i < kNAcc; ++i) rec_head[(int64_t)i * a.P_pad] = v[i];
                            a.rec_idx[(int64_t)(w * 2 + 0) * a.P_pad + p] = j;
                            flushed = true;
                        } else {
                            a.Fk[(int64_t)particle * N + j] = 0.5 * two_F(v);
                        }
#pragma unroll
                        for (int i = 0; i < kNAcc; ++i) { acc[i] = 0.0; in[i] = 0.0; }
                    }
                    ++j;
                    e_next = (j < N) ? band_edge(j + 1, q_lo, D, N, C, a.n_bins) : INT32_MAX;
                }
                const double mask = (j >= 0 && j < N) ? 1.0 : 0.0;     // the template window (reading A14 lifted)
                const double2 *row = reinterpret_cast<const double2 *>(tile + b * kTabW);
                const double2 dwv = row[10];
                double psi, sps, cps, tpr, tpi, tcr, tci;
                bin_template(row, c, a.orb, psi, sps, cps, tpr, tpi, tcr, tci);
                const double qr = mask * fma(dwv.x, cps, -dwv.y * sps);         // dw' exp(+i Psi)
                const double qi = mask * fma(dwv.x, sps, dwv.y * cps);
                in[0] = fma(qr, tpr, fma(qi, tpi, in[0]));                      // z_+ += q conj(T'_+)
                in[1] = fma(qi, tpr, fma(-qr, tpi, in[1]));
                in[2] = fma(qr, tcr, fma(qi, tci, in[2]));                      // z_x
                in[3] = fma(qi, tcr, fma(-qr, tci, in[3]));
                const double wgt = mask * row[11].x;
                in[4] = fma(wgt, fma(tpr, tpr, tpi * tpi), in[4]);              // m_pp
                in[5] = fma(wgt, fma(tcr, tcr, tci * tci), in[5]);              // m_cc
                in[6] = fma(wgt, fma(tpr, tcr, tpi * tci), in[6]);              // m_pc
                in[7] = fma(wgt, fma(tpi, tcr, -tpr * tci), in[7]);
            }
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) acc[i] += in[i];

            __syncthreads();                             // every thread is done with this slot
            if (tid == 0 && t + kStages < n_tiles) ring_issue(sm, src, n_bins, g0, t + kStages);
        }
        g0 += n_tiles;

        if (j >= 0 && j < N) {                           // the fragment after the last edge: partition j goes on
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) rec_tail[(int64_t)i * a.P_pad] = acc[i];
            a.rec_idx[(int64_t)(w * 2 + 1) * a.P_pad + p] = j;
        }
    }
}

// One thread per slot walks the head / tail records in grid order; consecutive records of the same
// partition are fragments of it.  Fixed order of every sum: results are bit-reproducible.
__global__ void __launch_bounds__(128) band_epilogue_kernel(const double *__restrict__ rec,
                                                            const int32_t *__restrict__ rec_idx,
                                                            const int32_t *__restrict__ valid,
                                                            const int32_t *__restrict__ perm, int64_t P_pad,
                                                            int32_t n_wseg, int32_t N, double *__restrict__ F,
                                                            double *__restrict__ Fk)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P_pad) return;
    const int32_t particle = perm[p];
    if (particle < 0) return;
    double *row = Fk + (int64_t)particle * N;
    if (valid[p] == 0) {
        for (int j = 0; j < N; ++j) row[j] = -INFINITY;
        F[particle] = -INFINITY;
        return;
    }
    int32_t cur = -1;
    double v[kNAcc];
#pragma unroll
    for (int i = 0; i < kNAcc; ++i) v[i] = 0.0;
    for (int r = 0; r < 2 * n_wseg; ++r) {
        const int32_t idx = rec_idx[(int64_t)r * P_pad + p];
        if (idx < 0) continue;
        if (idx != cur) {
            if (cur >= 0) row[cur] = 0.5 * two_F(v);
            cur = idx;
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) v[i] = 0.0;
        }
        const double *src = rec + ((int64_t)r * kNAcc) * P_pad + p;
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) v[i] += src[(int64_t)i * P_pad];
    }
    if (cur >= 0) row[cur] = 0.5 * two_F(v);
    double f = 0.0;
    for (int j = 0; j < N; ++j) f += row[j];             // F = sum_k F_k (Eq. 11 :110, reading A12)
    F[particle] = f;
}

// ---------------------------------------------------------------------------------------------------
// The same pieces ordered by length, for many partitions (cells of at most 128 bins): the piece lengths are
// uniform in 1 .. Cc/2, so a warp of band_ragged_kernel runs with half of its lanes masked.  piece_list_kernel
// enumerates the pieces twice (count, then fill) into a list ordered by length -- per-block shared-memory
// histograms, one global atomic per (block, length) -- and band_ragged_sorted_kernel evaluates one list entry
// per thread: the lanes of a warp then run the same number of bins.  The order inside a length class depends
// on atomics; the values do not.  (Partitions with no whole cell inside stay with band_ragged_kernel.)
// ---------------------------------------------------------------------------------------------------
constexpr int kMaxPieceLen = 64;                              // Cc / 2 for Cc <= 128

template <bool FILL>
__global__ void __launch_bounds__(128) piece_list_kernel(const int32_t *__restrict__ valid,
                                                         const int32_t *__restrict__ band_lo,
                                                         const int32_t *__restrict__ band_hi, int64_t P_pad,
                                                         int32_t n_bins, int32_t N, int32_t C, int32_t Cc,
                                                         int32_t *__restrict__ len_count,          // [kMaxPieceLen + 1]
                                                         const int32_t *__restrict__ len_start,    // [kMaxPieceLen + 2]
                                                         int2 *__restrict__ list)
{
    __shared__ int32_t hist[kMaxPieceLen + 1], base[kMaxPieceLen + 1];
    const int tid = threadIdx.x;
    for (int i = tid; i <= kMaxPieceLen; i += 128) hist[i] = 0;
    __syncthreads();
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + tid;
    const int j = blockIdx.y;                                 // one edge per block row: gridDim.y = N + 1
    int32_t len = 0, rank = 0;
    if (p < P_pad && valid[p] != 0) {
        const int32_t q_lo = (band_lo[p] + C / 2) / C, D = (band_hi[p] + C / 2) / C - q_lo;
        if (D > 0) {
            const int32_t e = band_edge(j, q_lo, D, N, C, n_bins);
            if (e < n_bins && e % Cc != 0 && !(j > 0 && band_edge(j - 1, q_lo, D, N, C, n_bins) == e)) {
                const int32_t c0 = (e / Cc) * Cc, c1 = min(c0 + Cc, n_bins);
                len = min(e - c0, c1 - e);                    // >= 1
                rank = atomicAdd(&hist[len], 1);
            }
        }
    }
    __syncthreads();
    if (tid <= kMaxPieceLen && hist[tid] > 0) base[tid] = atomicAdd(&len_count[tid], hist[tid]);
    if (tid + 128 <= kMaxPieceLen && hist[tid + 128] > 0) base[tid + 128] = atomicAdd(&len_count[tid + 128], hist[tid + 128]);
    __syncthreads();
    if (FILL && len > 0) list[len_start[len] + base[len] + rank] = make_int2((int)p, j);
}

// exclusive prefix of the length classes, longest first (long pieces start first: shorter tail); zeroes the counts
__global__ void piece_scan_kernel(int32_t *__restrict__ len_count, int32_t *__restrict__ len_start)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int32_t run = 0;
    for (int l = kMaxPieceLen; l >= 0; --l) {
        len_start[l] = run;
        run += len_count[l];
        len_count[l] = 0;
    }
    len_start[kMaxPieceLen + 1] = run;                        // the number of pieces
}

__global__ void __launch_bounds__(128) band_ragged_sorted_kernel(const double *__restrict__ table,
                                                                 const double *__restrict__ coef,
                                                                 const int32_t *__restrict__ band_lo,
                                                                 const int32_t *__restrict__ band_hi, int64_t P_pad,
                                                                 int32_t n_bins, int32_t N, int32_t C, int32_t Cc,
                                                                 const int32_t *__restrict__ len_start,
                                                                 const int2 *__restrict__ list,
                                                                 const __grid_constant__ OrbitCoef orb,
                                                                 double *__restrict__ rag)
{
    const int32_t n_pieces = len_start[kMaxPieceLen + 1];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_pieces; i += (int64_t)gridDim.x * blockDim.x) {
        const int2 pj = list[i];
        const int64_t p = pj.x;
        const int32_t q_lo = (band_lo[p] + C / 2) / C, D = (band_hi[p] + C / 2) / C - q_lo;
        const int32_t e = band_edge(pj.y, q_lo, D, N, C, n_bins);
        const int32_t c0 = (e / Cc) * Cc, c1 = min(c0 + Cc, n_bins);
        const bool left = (e - c0) <= (c1 - e);
        const int32_t b0 = left ? c0 : e, b1 = left ? e : c1;
        double c[kNCoef];
#pragma unroll
        for (int q = 0; q < kNCoef; ++q) c[q] = coef[(int64_t)q * P_pad + p];
        double acc[kNAcc];
#pragma unroll
        for (int q = 0; q < kNAcc; ++q) acc[q] = 0.0;
        double2 cur[12], nxt[12];
        {
            const double2 *r0 = reinterpret_cast<const double2 *>(table + (int64_t)b0 * kTabW);
#pragma unroll
            for (int q = 0; q < 12; ++q) cur[q] = r0[q];
        }
#pragma unroll 1
        for (int k = b0; k < b1; ++k) {
            {
                const double2 *rn = reinterpret_cast<const double2 *>(table + (int64_t)min(k + 1, b1 - 1) * kTabW);
#pragma unroll
                for (int q = 0; q < 12; ++q) nxt[q] = rn[q];
            }
            const double2 dwv = cur[10];
            double psi, sps, cps, tpr, tpi, tcr, tci;
            bin_template(cur, c, orb, psi, sps, cps, tpr, tpi, tcr, tci);
            const double qr = fma(dwv.x, cps, -dwv.y * sps);
            const double qi = fma(dwv.x, sps, dwv.y * cps);
            acc[0] = fma(qr, tpr, fma(qi, tpi, acc[0]));
            acc[1] = fma(qi, tpr, fma(-qr, tpi, acc[1]));
            acc[2] = fma(qr, tcr, fma(qi, tci, acc[2]));
            acc[3] = fma(qi, tcr, fma(-qr, tci, acc[3]));
            const double wgt = cur[11].x;
            acc[4] = fma(wgt, fma(tpr, tpr, tpi * tpi), acc[4]);
            acc[5] = fma(wgt, fma(tcr, tcr, tci * tci), acc[5]);
            acc[6] = fma(wgt, fma(tpr, tcr, tpi * tci), acc[6]);
            acc[7] = fma(wgt, fma(tpi, tcr, -tpr * tci), acc[7]);
#pragma unroll
            for (int q = 0; q < 12; ++q) cur[q] = nxt[q];
        }
        double *out = rag + ((int64_t)p * (N + 1) + pj.y) * kNAcc;
#pragma unroll
        for (int q = 0; q < kNAcc; ++q) out[q] = acc[q];
    }
}

// The partitions of the templates from the cell records.  Cell c of the internal plan is its partition c: its
// records are segments part_seg[c] .. part_seg[c + 1], slot-major or value-major (sk, sp).  Cc = width of the
// cells; C = lattice of the edge rule.  rag == nullptr: C == Cc, every edge is a cell boundary.  Otherwise an
// edge may split its cell and rag holds the two pieces (band_ragged_kernel): a partition is
//   right piece of e_j  +  the whole cells between  +  left piece of e_{j+1},
// except that a partition with no whole cell inside is evaluated in full, edge to edge (rag_short): short
// partitions are the ill-conditioned ones.  Everything is brought to one basis (recentred basis, add_record) and
// summed in a fixed order.
//   LANES == 8: block = 32 slots (x) by 8 lanes (y), blockIdx.y walks the partitions and the lanes split the
//               cells of one (slot, partition), combined through shared memory  (few, long partitions);
//   LANES == 1: block = 32 slots by 8 partitions, one thread per (slot, partition)  (many short partitions).
// F_k (and, rows f2 x f3, the extrinsic amplitudes a = M^-1 N of Eq. 10 :96) of one partition from its eight sums:
// invalid particle: -inf / NaN; empty partition: 0 / 0.
__device__ __forceinline__ void write_partition(const double (&v)[kNAcc], double cs_r, double cs_i, bool ok, bool live,
                                                int64_t idx, double *__restrict__ Fk, double *__restrict__ amp)
{
    Fk[idx] = ok ? (live ? 0.5 * two_F(v) : 0.0) : -INFINITY;
    if (amp != nullptr) {
        double a1 = 0.0, a2 = 0.0, a3 = 0.0, a4 = 0.0;
        if (ok && live) solve_amplitudes(v, cs_r, cs_i, a1, a2, a3, a4);
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        amp[4 * idx + 0] = ok ? a1 : nan;
        amp[4 * idx + 1] = ok ? a2 : nan;
        amp[4 * idx + 2] = ok ? a3 : nan;
        amp[4 * idx + 3] = ok ? a4 : nan;
    }
}

template <int LANES>
__global__ void __launch_bounds__(256) band_cells_epilogue_kernel(const double *__restrict__ partial,
                                                                  const double *__restrict__ rag,
                                                                  const double *__restrict__ rag_short,
                                                                  const int32_t *__restrict__ part_seg,
                                                                  const int32_t *__restrict__ valid,
                                                                  const int32_t *__restrict__ perm,
                                                                  const int32_t *__restrict__ band_lo,
                                                                  const int32_t *__restrict__ band_hi, int64_t P_pad,
                                                                  int32_t n_bins, int32_t n_cells, int32_t N, int32_t C,
                                                                  int32_t Cc, int64_t sk, int64_t sp,
                                                                  double *__restrict__ Fk, double *__restrict__ amp)
{
    __shared__ double sV[LANES == 8 ? 8 : 1][kNAcc][32];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int64_t p = (int64_t)blockIdx.x * 32 + tx;         // < P_pad: the grid covers P_pad / 32 blocks exactly
    const int32_t particle = perm[p];
    const bool ok = particle >= 0 && valid[p] != 0;
    const int32_t q_lo = (band_lo[p] + C / 2) / C, D = (band_hi[p] + C / 2) / C - q_lo;
    const int j_first = LANES == 8 ? (int)blockIdx.y : (int)blockIdx.y * 8 + ty;
    const int j_step = LANES == 8 ? gridDim.y : gridDim.y * 8;
    const int lane = LANES == 8 ? ty : 0;
    for (int j = j_first; j < N; j += j_step) {
        double v[kNAcc];
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) v[i] = 0.0;
        bool live = false;                                   // a non-empty partition of a valid particle
        double cs_r = 0.0, cs_i = 0.0;                       // the basis the sums are brought to
        if (ok) {
            const int32_t ea = band_edge(j, q_lo, D, N, C, n_bins), eb = band_edge(j + 1, q_lo, D, N, C, n_bins);
            if (eb > ea) {
                live = true;
                const bool onA = rag == nullptr || (ea % Cc) == 0;
                const bool onB = rag == nullptr || eb >= n_bins || (eb % Cc) == 0;
                const int32_t ca = onA ? ea / Cc : ea / Cc + 1, cb = eb >= n_bins ? n_cells : eb / Cc;
                int ja = j, jb = j + 1;
                if (!onA || !onB) {
                    // the piece of an edge shared by several (empty) partitions is stored under its first index
                    while (ja > 0 && band_edge(ja - 1, q_lo, D, N, C, n_bins) == ea) --ja;
                    while (jb > 0 && band_edge(jb - 1, q_lo, D, N, C, n_bins) == eb) --jb;
                }
                // common basis: the one of the cell that starts at or holds e_j (always evaluated for this group)
                const double *first = partial + ((int64_t)part_seg[ea / Cc] * kNPartial) * P_pad + p * sp;
                cs_r = first[8 * sk];
                cs_i = first[9 * sk];
                // sgn x (left or right piece of the cell edge e splits), e = edge number je of this template
                auto add_piece = [&](int32_t e, int je, bool want_left, double sgn) {
                    const int32_t c0 = (e / Cc) * Cc, c1 = min(c0 + Cc, n_bins);
                    const bool stored_left = (e - c0) <= (c1 - e);
                    const double *r = rag + ((int64_t)p * (N + 1) + je) * kNAcc;
                    double t[kNPartial];
                    const double sg = (stored_left == want_left) ? sgn : -sgn;
#pragma unroll
                    for (int i = 0; i < kNAcc; ++i) t[i] = sg * r[i];
                    t[8] = 0.0; t[9] = 0.0;
                    add_record(t, cs_r, cs_i, v);
                    if (stored_left != want_left) {          // the wanted piece = the cell's record - the stored piece
                        for (int sc = part_seg[e / Cc]; sc < part_seg[e / Cc + 1]; ++sc) {
                            const double *src = partial + ((int64_t)sc * kNPartial) * P_pad + p * sp;
#pragma unroll
                            for (int i = 0; i < kNAcc; ++i) t[i] = sgn * src[(int64_t)i * sk];
                            t[8] = src[8 * sk]; t[9] = src[9 * sk];
                            add_record(t, cs_r, cs_i, v);
                        }
                    }
                };
                if (rag != nullptr && ca >= cb) {            // no whole cell inside: evaluated in full, edge to edge
                    cs_r = 0.0;
                    cs_i = 0.0;
                    if (lane == 0) {
                        const double *r = rag_short + ((int64_t)p * N + j) * kNAcc;
#pragma unroll
                        for (int i = 0; i < kNAcc; ++i) v[i] = r[i];
                    }
                } else {
                    if (!onA && lane == 0) add_piece(ea, ja, false, 1.0);
                    const int s0 = part_seg[ca], s1 = part_seg[cb];
#pragma unroll 2
                    for (int s = s0 + lane; s < s1; s += LANES) add_segment(partial, s, P_pad, sk, sp, p, cs_r, cs_i, v);
                    if (!onB && lane == 0) add_piece(eb, jb, true, 1.0);
                }
            }
        }
        if (LANES == 8) {
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) sV[ty][i][tx] = v[i];
            __syncthreads();
            if (ty == (j & 7) && particle >= 0) {
#pragma unroll
                for (int i = 0; i < kNAcc; ++i) {
                    double acc = 0.0;
#pragma unroll
                    for (int y = 0; y < 8; ++y) acc += sV[y][i][tx];
                    v[i] = acc;
                }
                write_partition(v, cs_r, cs_i, ok, live, (int64_t)particle * N + j, Fk, amp);
            }
            __syncthreads();
        } else if (particle >= 0) {
            write_partition(v, cs_r, cs_i, ok, live, (int64_t)particle * N + j, Fk, amp);
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Edges at ANY bin on top of the cell records (edge_lattice < 32 with the interpolating kernel available): the
// cells are Cc bins wide; an edge e that is not a cell boundary splits its cell [c Cc, (c + 1) Cc) into a left
// piece (the end of partition j - 1) and a right piece (the start of partition j).  band_ragged_kernel evaluates
// the SHORTER of the two pieces with the full model, one thread per (slot, edge), straight from the per-bin
// table: rag[(p (N + 1) + j) 8 + i], plain basis (c = 0); the other piece is the cell's record minus this one
// (the cell's record carries the interpolation error of any other cell, the piece none).  A partition is then
//   right piece of e_j  +  the whole cells between  +  left piece of e_{j+1}
// (a partition with no whole cell inside is evaluated edge to edge instead), combined by band_cells_epilogue_kernel.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) band_ragged_kernel(const double *__restrict__ table, const double *__restrict__ coef,
                                                          const int32_t *__restrict__ valid,
                                                          const int32_t *__restrict__ band_lo,
                                                          const int32_t *__restrict__ band_hi, int64_t P_pad,
                                                          int32_t n_bins, int32_t N, int32_t C, int32_t Cc,
                                                          const __grid_constant__ OrbitCoef orb, double *__restrict__ rag,
                                                          double *__restrict__ rag_short, int32_t short_only)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P_pad || valid[p] == 0) return;
    const int32_t q_lo = (band_lo[p] + C / 2) / C, D = (band_hi[p] + C / 2) / C - q_lo;
    if (D <= 0) return;
    double c[kNCoef];
#pragma unroll
    for (int i = 0; i < kNCoef; ++i) c[i] = coef[(int64_t)i * P_pad + p];
    // sums of the full model over the bins [b0, b1) into out[0..7] (plain basis).  The next bin's table row is
    // fetched while this one is evaluated (every thread walks its own rows: nothing to share through shared
    // memory, and the loads would otherwise sit in front of 263 dependent FP64 instructions).
    auto eval_range = [&](int32_t b0, int32_t b1, double *__restrict__ out) {
        double acc[kNAcc];
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) acc[i] = 0.0;
        double2 cur[12], nxt[12];
        {
            const double2 *r0 = reinterpret_cast<const double2 *>(table + (int64_t)b0 * kTabW);
#pragma unroll
            for (int i = 0; i < 12; ++i) cur[i] = r0[i];
        }
#pragma unroll 1
        for (int k = b0; k < b1; ++k) {
            {
                const double2 *rn = reinterpret_cast<const double2 *>(table + (int64_t)min(k + 1, b1 - 1) * kTabW);
#pragma unroll
                for (int i = 0; i < 12; ++i) nxt[i] = rn[i];
            }
            const double2 dwv = cur[10];
            double psi, sps, cps, tpr, tpi, tcr, tci;
            bin_template(cur, c, orb, psi, sps, cps, tpr, tpi, tcr, tci);
            const double qr = fma(dwv.x, cps, -dwv.y * sps);
            const double qi = fma(dwv.x, sps, dwv.y * cps);
            acc[0] = fma(qr, tpr, fma(qi, tpi, acc[0]));
            acc[1] = fma(qi, tpr, fma(-qr, tpi, acc[1]));
            acc[2] = fma(qr, tcr, fma(qi, tci, acc[2]));
            acc[3] = fma(qi, tcr, fma(-qr, tci, acc[3]));
            const double wgt = cur[11].x;
            acc[4] = fma(wgt, fma(tpr, tpr, tpi * tpi), acc[4]);
            acc[5] = fma(wgt, fma(tcr, tcr, tci * tci), acc[5]);
            acc[6] = fma(wgt, fma(tpr, tcr, tpi * tci), acc[6]);
            acc[7] = fma(wgt, fma(tpi, tcr, -tpr * tci), acc[7]);
#pragma unroll
            for (int i = 0; i < 12; ++i) cur[i] = nxt[i];
        }
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) out[i] = acc[i];
    };
    for (int j = blockIdx.y; j <= N; j += gridDim.y) {
        const int32_t e = band_edge(j, q_lo, D, N, C, n_bins);
        // (1) a partition that holds no whole cell is evaluated in full, edge to edge: short partitions have a
        // near-singular M_k (conditioning note) and must not see the interpolation error of a cell record
        if (j < N) {
            const int32_t eb = band_edge(j + 1, q_lo, D, N, C, n_bins);
            const int32_t ca = (e + Cc - 1) / Cc, cb = eb >= n_bins ? (n_bins + Cc - 1) / Cc : eb / Cc;
            if (eb > e && ca >= cb) eval_range(e, eb, rag_short + ((int64_t)p * N + j) * kNAcc);
        }
        // (2) the shorter piece of the cell this edge splits (the other piece is the cell's record minus it)
        if (short_only) continue;                                       // (done by band_ragged_sorted_kernel)
        if (e >= n_bins || e % Cc == 0) continue;                       // a cell boundary: nothing to split
        if (j > 0 && band_edge(j - 1, q_lo, D, N, C, n_bins) == e) continue;   // same edge as the previous one
        const int32_t c0 = (e / Cc) * Cc, c1 = min(c0 + Cc, n_bins);
        const bool left = (e - c0) <= (c1 - e);
        eval_range(left ? c0 : e, left ? e : c1, rag + ((int64_t)p * (N + 1) + j) * kNAcc);
    }
}

// F = sum_k F_k: one warp per particle, lane l adds k = l, l + 32, ..., then a fixed shuffle tree.
__global__ void __launch_bounds__(128) band_fsum_kernel(const double *__restrict__ Fk, int64_t P, int32_t N,
                                                        double *__restrict__ F)
{
    const int64_t q = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (q >= P) return;
    const int lane = threadIdx.x & 31;
    double f = 0.0;
    for (int j = lane; j < N; j += 32) f += Fk[q * N + j];   // -inf rows (invalid particles) stay -inf
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) f += __shfl_xor_sync(0xffffffffu, f, o);
    if (lane == 0) F[q] = f;
}

// rag == nullptr: every edge is a cell boundary (lattice == cell); else the pieces are computed first.
cudaError_t launch_band_cells_epilogue(const double *table, const double *coef, const double *partial, double *rag,
                                       double *rag_short, int32_t *piece_scratch, int2 *piece_list, const int32_t *part_seg, const int32_t *valid, const int32_t *perm,
                                       const int32_t *band_lo, const int32_t *band_hi, int64_t P, int64_t P_pad,
                                       int32_t n_bins, int32_t n_cells, int32_t n_seg_band, int32_t lattice, int32_t cell,
                                       int64_t part_sk, int64_t part_sp, const OrbitCoef &orb, double *F, double *Fk,
                                       double *amp, cudaStream_t st)
{
    cudaError_t e;
    if (rag != nullptr) {
        int gy = n_seg_band + 1;
        if (gy > 2048) gy = 2048;
        const bool sorted = piece_scratch != nullptr && cell <= 2 * kMaxPieceLen && n_seg_band >= 128 && n_seg_band < 65535;
        band_ragged_kernel<<<dim3((unsigned)(P_pad / 128), (unsigned)gy), 128, 0, st>>>(
            table, coef, valid, band_lo, band_hi, P_pad, n_bins, n_seg_band, lattice, cell, orb, rag, rag_short, sorted ? 1 : 0);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        if (sorted) {                                         // many pieces: evaluate them in the order of their lengths
            int32_t *count = piece_scratch, *start = piece_scratch + (kMaxPieceLen + 1);
            const dim3 grd((unsigned)(P_pad / 128), (unsigned)(n_seg_band + 1));
            if ((e = cudaMemsetAsync(count, 0, (kMaxPieceLen + 1) * sizeof(int32_t), st)) != cudaSuccess) return e;
            piece_list_kernel<false><<<grd, 128, 0, st>>>(valid, band_lo, band_hi, P_pad, n_bins, n_seg_band, lattice, cell, count,
                                                          nullptr, nullptr);
            piece_scan_kernel<<<1, 32, 0, st>>>(count, start);
            piece_list_kernel<true><<<grd, 128, 0, st>>>(valid, band_lo, band_hi, P_pad, n_bins, n_seg_band, lattice, cell, count,
                                                         start, piece_list);
            int64_t nb = (P_pad * (int64_t)(n_seg_band + 1) + 127) / 128;
            if (nb > 148 * 48) nb = 148 * 48;
            band_ragged_sorted_kernel<<<(unsigned)nb, 128, 0, st>>>(table, coef, band_lo, band_hi, P_pad, n_bins, n_seg_band,
                                                                    lattice, cell, start, piece_list, orb, rag);
            if ((e = cudaGetLastError()) != cudaSuccess) return e;
        }
    }
    if ((int64_t)n_cells < (int64_t)32 * n_seg_band) {      // a few cells per partition: one thread per partition
        int gy = (n_seg_band + 7) / 8;
        if (gy > 4096) gy = 4096;
        band_cells_epilogue_kernel<1><<<dim3((unsigned)(P_pad / 32), (unsigned)gy), dim3(32, 8), 0, st>>>(
            partial, rag, rag_short, part_seg, valid, perm, band_lo, band_hi, P_pad, n_bins, n_cells, n_seg_band, lattice, cell,
            part_sk, part_sp, Fk, amp);
    } else {
        const int gy = n_seg_band < 4096 ? n_seg_band : 4096;
        band_cells_epilogue_kernel<8><<<dim3((unsigned)(P_pad / 32), (unsigned)gy), dim3(32, 8), 0, st>>>(
            partial, rag, rag_short, part_seg, valid, perm, band_lo, band_hi, P_pad, n_bins, n_cells, n_seg_band, lattice, cell,
            part_sk, part_sp, Fk, amp);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    band_fsum_kernel<<<(unsigned)((P + 3) / 4), 128, 0, st>>>(Fk, P, n_seg_band, F);
    return cudaGetLastError();
}

cudaError_t band_kernel_configure()
{
    return cudaFuncSetAttribute(fstat_band_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MainSmem));
}

cudaError_t launch_band_limits(const double *table, const double *coef, const int32_t *valid, const int32_t *perm,
                               int64_t P_pad, int32_t n_bins, double T_obs, double kappa, int32_t *band_lo,
                               int32_t *band_hi, int64_t *band_out, cudaStream_t st)
{
    band_kernel<<<(unsigned)((P_pad + 127) / 128), 128, 0, st>>>(table, coef, valid, perm, P_pad, n_bins, T_obs,
                                                                  2.0 * kappa / kPi, band_lo, band_hi, band_out);
    return cudaGetLastError();
}

cudaError_t launch_band_main(const BandArgs &a, int32_t max_ctas, cudaStream_t st)
{
    int64_t n_cta = (int64_t)a.n_groups * a.n_wseg;
    if (n_cta > max_ctas) n_cta = max_ctas;
    fstat_band_kernel<<<(unsigned)n_cta, kThreads, sizeof(MainSmem), st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_band_epilogue(const double *rec, const int32_t *rec_idx, const int32_t *valid, const int32_t *perm,
                                 int64_t P_pad, int32_t n_wseg, int32_t n_seg, double *F, double *Fk, cudaStream_t st)
{
    band_epilogue_kernel<<<(unsigned)((P_pad + 127) / 128), 128, 0, st>>>(rec, rec_idx, valid, perm, P_pad, n_wseg,
                                                                           n_seg, F, Fk);
    return cudaGetLastError();
}

}  // namespace fstat
