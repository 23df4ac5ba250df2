// fstat_band.cu -- SURVEY row f2: the semi-coherent F-statistic with the paper's OWN segment limits
// (PAPER.md:122): the number of segments is fixed for all templates, the outer limits are "the lowest and
// highest instantaneous frequencies occurring during the observation period in the template", i.e. the
// bins whose stationary time t_f (Eq. 20 :220) lies in [0, T_obs].  Partition edges therefore differ from
// particle to particle (reading A26 for where they fall on the grid).  What lives here, around the interpolating
// kernel with per-thread edges (fstat_fastband.cu):
//
//   band_kernel          k_lo = #{bins with t_f < 0}, k_hi = #{bins with t_f <= T_obs} per particle, by
//                        bisection over the grid (t_f increases along it)
//   fstat_band_kernel    the DIRECT kernel (full model at every in-band bin) with per-thread partition edges, for
//                        the (particle group, work segment) items the stride selection leaves to it
//                        (options.force_level == -1: all of them); same head / tail records and in-thread
//                        completion of partitions as the interpolating kernel
//   band_short_kernel    templates with an empty partition or one shorter than 8 bins (band_fast_eligible false)
//                        do not take part in either main kernel: every partition of theirs is evaluated edge to
//                        edge with the full model, one thread per (template, partition)
//   band_stitch_kernel   partitions that straddle work segments: tail fragment of the first segment + whole-segment
//                        fragments + head fragment of the last one, in the recentred basis of the first, fixed order;
//                        also writes the -inf / NaN rows of invalid particles
//   band_fsum_kernel     F = sum_k F_k in a fixed order
#include "fstat_device.cuh"
#include "fstat_direct.cuh"
#include "fstat_internal.h"
#include "fstat_model.cuh"

#include <math.h>

namespace fstat {

// t_f [s] (Eq. 20 :220, from Psi_0 only, reading A4) at frequency f: the orbital phase at t_f in quarter turns of a
// year is alpha_q = c10 + sum_j c_j D_j(f), D_j = (dB_j/df) / year in the order of the phase basis (fill_basis_row),
// and t_f = (alpha_q - 2 kappa / pi) year / 4.  Evaluated from f itself: the bisection below jumps across the whole
// grid, and 42 dependent table reads would cost more than the arithmetic.
__device__ __forceinline__ double tf_seconds(double f, const double (&c)[kNCoef], double kappa_qt)
{
    const double lnf = log(f);
    const double icb = 1.0 / cbrt(f);                  // f^(-1/3)
    const double fm23 = icb * icb, fm1 = 1.0 / f, fm53 = fm1 * fm23;
    const double fm349 = pow(f, -34.0 / 9.0);
    double alq = c[10] * kYear;
    alq = fma(c[2], fm1, alq);
    alq = fma(c[3], (-5.0 / 3.0) * fm53 * fm1, alq);
    alq = fma(c[4], -fm1 * fm1, alq);
    alq = fma(c[5], (-2.0 / 3.0) * fm53, alq);
    alq = fma(c[6], (-1.0 / 3.0) * icb * fm1, alq);
    alq = fma(c[7], (1.0 / 3.0) * fm23, alq);
    alq = fma(c[8], fm23 * (1.0 + lnf / 3.0), alq);
    alq = fma(c[9], (-34.0 / 9.0) * fm349 * fm1, alq);
    return (alq - kappa_qt * kYear) * 0.25;
}

__global__ void __launch_bounds__(128) band_kernel(const double *__restrict__ coef, const int32_t *__restrict__ valid,
                                                   const int32_t *__restrict__ perm, int64_t P_pad, int32_t n_bins,
                                                   double f0, double df, double T_obs, double kappa_qt,
                                                   int32_t *__restrict__ band_lo, int32_t *__restrict__ band_hi,
                                                   int64_t *__restrict__ band_out)
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
            if (tf_seconds(fma((double)m, df, f0), c, kappa_qt) < 0.0) a = m + 1; else b = m;
        }
        k_lo = a;
        // first bin with t_f > T_obs
        b = n_bins;
        while (a < b) {
            const int32_t m = a + ((b - a) >> 1);
            if (tf_seconds(fma((double)m, df, f0), c, kappa_qt) <= T_obs) a = m + 1; else b = m;
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

// F_k and, on request, the amplitudes a = M^-1 N (Eq. 10 :96) of one partition from its eight sums in the basis
// (u_+, u_x - c u_+)
__device__ __forceinline__ void write_partition(const double (&v)[kNAcc], double cs_r, double cs_i, int64_t idx,
                                                double *__restrict__ Fk, double *__restrict__ amp)
{
    Fk[idx] = 0.5 * two_F(v);
    if (amp != nullptr) {
        double a1, a2, a3, a4;
        solve_amplitudes(v, cs_r, cs_i, a1, a2, a3, a4);
        amp[4 * idx + 0] = a1; amp[4 * idx + 1] = a2; amp[4 * idx + 2] = a3; amp[4 * idx + 3] = a4;
    }
}

// ---------------------------------------------------------------------------------------------------
// Direct kernel with per-thread edges.  Work item = (group of 128 slots) x (work segment), taken from the list the
// stride selection wrote; persistent CTAs stride over the list.  All threads of a CTA walk the same bins
// (shared-memory broadcast of the table rows); each thread carries the partition j its current bin belongs to and
// the bin e_next where it closes, compares once per bin, and masks its weights outside the band.  Recentred basis,
// one constant per partition.  Records and completion rules as in fstat_fastband_kernel.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) fstat_band_kernel(const __grid_constant__ BandArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    MainSmem &sm = *reinterpret_cast<MainSmem *>(smem_raw);

    const int tid = threadIdx.x;
    const int n_items = *a.direct_count;
    if ((int)blockIdx.x >= n_items) return;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&sm.full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    int g0 = 0;                                          // tiles consumed so far by this CTA (ring position)
    const int32_t N = a.b.N, C = a.b.C;

    for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const int item = a.direct_list[it];
        const int grp = item / a.n_seg;
        const int w = item - grp * a.n_seg;
        const int64_t p = (int64_t)grp * kThreads + tid;
        const int lo = a.seg_edge[w], hi = a.seg_edge[w + 1];

        const int32_t q_lo = (a.b.band_lo[p] + C / 2) / C, D = (a.b.band_hi[p] + C / 2) / C - q_lo;
        int32_t j = N, e_next = INT32_MAX;
        bool opened = false;
        if (a.b.valid[p] != 0 && band_fast_eligible(D, N, C)) {
            const int32_t e0 = band_edge(0, q_lo, D, N, C, a.b.n_bins), eN = band_edge(N, q_lo, D, N, C, a.b.n_bins);
            if (lo < eN && hi > e0) {
                if (lo < e0) { j = -1; e_next = e0; }
                else {
                    const int64_t cells = (int64_t)(lo / C) - q_lo;       // largest j with e_j <= lo
                    int64_t jj = ((cells + 1) * N + D - 1) / D - 1;
                    if (jj > N - 1) jj = N - 1;
                    j = (int32_t)jj;
                    while (j + 1 < N && band_edge(j + 1, q_lo, D, N, C, a.b.n_bins) <= lo) ++j;
                    while (j > 0 && band_edge(j, q_lo, D, N, C, a.b.n_bins) > lo) --j;
                    e_next = band_edge(j + 1, q_lo, D, N, C, a.b.n_bins);
                    opened = band_edge(j, q_lo, D, N, C, a.b.n_bins) == lo;
                }
            }
        }

        const int n_bins = hi - lo;
        const int n_tiles = (n_bins + kTileBins - 1) / kTileBins;
        const BinSource src{reinterpret_cast<const double2 *>(a.dwp), reinterpret_cast<const double2 *>(a.fw)};
        if (tid == 0) ring_prologue(sm, src, lo, n_bins, n_tiles, g0);

        double c[kNCoef];
#pragma unroll
        for (int q = 0; q < kNCoef; ++q) c[q] = a.coef[(int64_t)q * a.P_pad + p];

        const int32_t particle = a.b.perm[p];
        double *rec_head = a.b.rec + ((int64_t)(w * 2 + 0) * kNPartial) * a.P_pad + p;
        double *rec_tail = a.b.rec + ((int64_t)(w * 2 + 1) * kNPartial) * a.P_pad + p;

        double acc[kNAcc];
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) acc[i] = 0.0;
        bool need_c = true;                                  // recentred basis (hazard H3), one constant per partition
        double c_re = 0.0, c_im = 0.0;

        for (int t = 0; t < n_tiles; ++t) {
            const int nb = min(kTileBins, n_bins - t * kTileBins);
            const double *tile = ring_wait(sm, g0 + t, nb, a.arm_length_m);
            if (tid == 0 && t + kStages < n_tiles) ring_issue(sm, src, lo, n_bins, g0, t + kStages);   // its slot is free: expanded
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
                        if (opened) {
                            write_partition(v, c_re, c_im, (int64_t)particle * N + j, a.b.Fk, a.b.amp);
                        } else {
#pragma unroll
                            for (int i = 0; i < kNAcc; ++i) rec_head[(int64_t)i * a.P_pad] = v[i];
                            rec_head[(int64_t)8 * a.P_pad] = c_re;
                            rec_head[(int64_t)9 * a.P_pad] = c_im;
                        }
                    }
#pragma unroll
                    for (int i = 0; i < kNAcc; ++i) { acc[i] = 0.0; in[i] = 0.0; }
                    need_c = true;
                    ++j;
                    opened = true;
                    e_next = (j < N) ? band_edge(j + 1, q_lo, D, N, C, a.b.n_bins) : INT32_MAX;
                }
                const double mask = (j >= 0 && j < N) ? 1.0 : 0.0;     // the template window (reading A14 lifted)
                const double2 *row = reinterpret_cast<const double2 *>(tile + b * kTabW);
                const double2 dwv = row[10];
                double psi, sps, cps, tpr, tpi, tcr, tci;
                bin_template(row, c, a.orb, psi, sps, cps, tpr, tpi, tcr, tci);
                if (need_c) {                                          // first bin of a partition (or of the work item)
                    need_c = false;
                    choose_basis(tpr, tpi, tcr, tci, c_re, c_im);
                }
                const double qr = mask * fma(dwv.x, cps, -dwv.y * sps);         // dw' exp(+i Psi)
                const double qi = mask * fma(dwv.x, sps, dwv.y * cps);
                accumulate_bin(qr, qi, mask * row[11].x, tpr, tpi, tcr, tci, c_re, c_im, in);
            }
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) acc[i] += in[i];
        }
        g0 += n_tiles;

        if (j >= 0 && j < N) {                           // what is left after the last edge (see fstat_fastband_kernel)
            if (e_next == hi && opened) {
                write_partition(acc, c_re, c_im, (int64_t)particle * N + j, a.b.Fk, a.b.amp);
            } else {
                double *out = (e_next == hi) ? rec_head : rec_tail;
#pragma unroll
                for (int i = 0; i < kNAcc; ++i) out[(int64_t)i * a.P_pad] = acc[i];
                out[(int64_t)8 * a.P_pad] = c_re;
                out[(int64_t)9 * a.P_pad] = c_im;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Templates the main kernels do not take: every partition edge to edge with the full model (every thread walks its
// own bins and expands their rows itself).
// Grid = slots (x) by partitions (y, strided).  Recentred basis (c at the partition's first bin).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) band_short_kernel(const double2 *__restrict__ dwp, const double2 *__restrict__ fw,
                                                         double L, const double *__restrict__ coef, const BandCommon b,
                                                         int64_t P_pad, const __grid_constant__ OrbitCoef orb)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P_pad || b.valid[p] == 0) return;
    const int32_t N = b.N, C = b.C;
    const int32_t q_lo = (b.band_lo[p] + C / 2) / C, D = (b.band_hi[p] + C / 2) / C - q_lo;
    if (D <= 0 || band_fast_eligible(D, N, C)) return;
    const int32_t particle = b.perm[p];
    double c[kNCoef];
#pragma unroll
    for (int i = 0; i < kNCoef; ++i) c[i] = coef[(int64_t)i * P_pad + p];
    for (int j = blockIdx.y; j < N; j += gridDim.y) {
        const int32_t b0 = band_edge(j, q_lo, D, N, C, b.n_bins), b1 = band_edge(j + 1, q_lo, D, N, C, b.n_bins);
        if (b1 <= b0) continue;                                          // empty: F_k = 0 (set by the caller)
        double acc[kNAcc];
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) acc[i] = 0.0;
        double c_re = 0.0, c_im = 0.0;                       // recentred basis: c = T'_x / T'_+ at the partition's first bin
#pragma unroll 1
        for (int k = b0; k < b1; ++k) {
            const double2 dwv = dwp[k], fwv = fw[k];
            __align__(16) double rowbuf[kTabW];
            fill_basis_row(fwv.x, L, rowbuf);                // every thread walks its own bins: rows expanded in registers
            double psi, sps, cps, tpr, tpi, tcr, tci;
            bin_template(reinterpret_cast<const double2 *>(rowbuf), c, orb, psi, sps, cps, tpr, tpi, tcr, tci);
            if (k == b0) choose_basis(tpr, tpi, tcr, tci, c_re, c_im);
            const double qr = fma(dwv.x, cps, -dwv.y * sps);
            const double qi = fma(dwv.x, sps, dwv.y * cps);
            accumulate_bin(qr, qi, fwv.y, tpr, tpi, tcr, tci, c_re, c_im, acc);
        }
        write_partition(acc, c_re, c_im, (int64_t)particle * N + j, b.Fk, b.amp);
    }
}

// ---------------------------------------------------------------------------------------------------
// Partitions that straddle work segments.  Partition j of a template spans the work segments s_a = e_j / W ..
// s_b = (e_{j+1} - 1) / W (both known from the edge rule, no index arrays): if s_a == s_b a main kernel has finished it;
// else its fragments are tail(s_a), tail(s_a + 1 .. s_b - 1) (whole segments) and head(s_b), summed here in the
// recentred basis of the first one (add_segment), in a fixed order.
//   LANES == 1: block = 32 slots by 8 partitions, one thread per (slot, partition)        (many short partitions)
//   LANES == 8: block = 32 slots by 8 lanes; blockIdx.y walks the partitions and the lanes split the fragments of one
//               (slot, partition), combined through shared memory                          (few long partitions)
// Also: invalid particles get F_k = -inf and NaN amplitudes.
// ---------------------------------------------------------------------------------------------------
template <int LANES>
__global__ void __launch_bounds__(256) band_stitch_kernel(const BandCommon b, int64_t P_pad, int32_t W)
{
    __shared__ double sV[LANES == 8 ? 8 : 1][kNAcc][32];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int64_t p = (int64_t)blockIdx.x * 32 + tx;         // < P_pad: the grid covers P_pad / 32 blocks exactly
    const int32_t particle = b.perm[p];
    const bool ok = particle >= 0 && b.valid[p] != 0;
    const int32_t N = b.N, C = b.C;
    const int32_t q_lo = (b.band_lo[p] + C / 2) / C, D = (b.band_hi[p] + C / 2) / C - q_lo;
    const bool fast = ok && band_fast_eligible(D, N, C);
    const int j_first = LANES == 8 ? (int)blockIdx.y : (int)blockIdx.y * 8 + ty;
    const int j_step = LANES == 8 ? gridDim.y : gridDim.y * 8;
    const int lane = LANES == 8 ? ty : 0;
    for (int j = j_first; j < N; j += j_step) {
        double v[kNAcc];
#pragma unroll
        for (int i = 0; i < kNAcc; ++i) v[i] = 0.0;
        bool mine = false;
        double cs_r = 0.0, cs_i = 0.0;
        if (fast) {
            const int32_t ea = band_edge(j, q_lo, D, N, C, b.n_bins), eb = band_edge(j + 1, q_lo, D, N, C, b.n_bins);
            if (eb > ea) {
                const int s_a = ea / W, s_b = (eb - 1) / W;
                if (s_b > s_a) {
                    mine = true;
                    const double *first = b.rec + ((int64_t)(s_a * 2 + 1) * kNPartial) * P_pad + p;
                    cs_r = first[(int64_t)8 * P_pad];
                    cs_i = first[(int64_t)9 * P_pad];
                    const int n_frag = s_b - s_a + 1;
                    for (int i = lane; i < n_frag; i += LANES) {
                        const int r = (i == n_frag - 1) ? s_b * 2 : (s_a + i) * 2 + 1;     // head of the last, else tails
                        add_segment(b.rec, r, P_pad, P_pad, 1, p, cs_r, cs_i, v);
                    }
                }
            }
        }
        if (LANES == 8) {
#pragma unroll
            for (int i = 0; i < kNAcc; ++i) sV[LANES == 8 ? ty : 0][i][tx] = v[i];
            __syncthreads();
            if (ty == (j & 7)) {
#pragma unroll
                for (int i = 0; i < kNAcc; ++i) {
                    double s = 0.0;
#pragma unroll
                    for (int y = 0; y < 8; ++y) s += sV[LANES == 8 ? y : 0][i][tx];
                    v[i] = s;
                }
            }
            __syncthreads();
            if (ty != (j & 7)) continue;
        }
        if (particle < 0) continue;
        const int64_t idx = (int64_t)particle * N + j;
        if (!ok) {
            b.Fk[idx] = -INFINITY;
            if (b.amp != nullptr) {
                const double nan = __longlong_as_double(0x7ff8000000000000LL);
                b.amp[4 * idx + 0] = nan; b.amp[4 * idx + 1] = nan; b.amp[4 * idx + 2] = nan; b.amp[4 * idx + 3] = nan;
            }
        } else if (mine) {
            write_partition(v, cs_r, cs_i, idx, b.Fk, b.amp);
        }
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

cudaError_t launch_band_short(const double *dwp, const double *fw, double arm_length_m, const double *coef,
                              const BandCommon &b, int64_t P_pad, const OrbitCoef &orb, cudaStream_t st)
{
    const int gy = b.N < 32 ? b.N : 32;                     // (usually no template takes this path: keep the grid small)
    band_short_kernel<<<dim3((unsigned)(P_pad / 128), (unsigned)gy), 128, 0, st>>>(
        reinterpret_cast<const double2 *>(dwp), reinterpret_cast<const double2 *>(fw), arm_length_m, coef, b, P_pad, orb);
    return cudaGetLastError();
}

cudaError_t launch_band_stitch(const BandCommon &b, int64_t P, int64_t P_pad, int32_t seg_len, int32_t n_seg, double *F,
                               cudaStream_t st)
{
    if ((int64_t)n_seg < (int64_t)16 * b.N) {               // a partition spans a few work segments at most
        int gy = (b.N + 7) / 8;
        if (gy > 4096) gy = 4096;
        band_stitch_kernel<1><<<dim3((unsigned)(P_pad / 32), (unsigned)gy), dim3(32, 8), 0, st>>>(b, P_pad, seg_len);
    } else {
        const int gy = b.N < 4096 ? b.N : 4096;
        band_stitch_kernel<8><<<dim3((unsigned)(P_pad / 32), (unsigned)gy), dim3(32, 8), 0, st>>>(b, P_pad, seg_len);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    band_fsum_kernel<<<(unsigned)((P + 3) / 4), 128, 0, st>>>(b.Fk, P, b.N, F);
    return cudaGetLastError();
}

cudaError_t band_kernel_configure()
{
    return cudaFuncSetAttribute(fstat_band_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MainSmem));
}

cudaError_t launch_band_limits(const double *coef, const int32_t *valid, const int32_t *perm, int64_t P_pad,
                               int32_t n_bins, double f0, double df, double T_obs, double kappa, int32_t *band_lo,
                               int32_t *band_hi, int64_t *band_out, cudaStream_t st)
{
    band_kernel<<<(unsigned)((P_pad + 127) / 128), 128, 0, st>>>(coef, valid, perm, P_pad, n_bins, f0, df, T_obs,
                                                                  2.0 * kappa / kPi, band_lo, band_hi, band_out);
    return cudaGetLastError();
}

cudaError_t launch_band_main(const BandArgs &a, int32_t max_ctas, cudaStream_t st)
{
    fstat_band_kernel<<<(unsigned)max_ctas, kThreads, sizeof(MainSmem), st>>>(a);
    return cudaGetLastError();
}

}  // namespace fstat
