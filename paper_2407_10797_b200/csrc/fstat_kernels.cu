// fstat_kernels.cu -- sm_100a kernels of the batched semi-coherent F-statistic (arXiv 2407.10797).
//
//   build_table_kernel   (a0, plan time)  per-bin, particle-independent factors of Eq. A1 and Eq. 4 folded into the data
//   prologue_kernel      (a1)             per-particle PN / eccentric phase coefficients and sky vectors
//   fstat_main_kernel    (a2-a5)          fused phase + t_f + orbit + TDI-X response + inner products;
//                                         one thread = one particle, bins streamed through shared memory
//                                         by TMA bulk copies; no template ever leaves the registers
//   epilogue_kernel      (a6)             2 F_k = z^H G^-1 z per partition, F = sum_k F_k
//
// Citations are to /root/reference/PAPER.md (line, equation) and to DESIGN.md readings (A1..A24).
#include "fstat_device.cuh"
#include "fstat_direct.cuh"
#include "fstat_internal.h"
#include "fstat_model.cuh"

#include <cub/device/device_radix_sort.cuh>
#include <math.h>

namespace fstat {

// =================================================================================================
// a0: per-bin table
// =================================================================================================
__global__ void build_table_kernel(const double *__restrict__ freq, const double *__restrict__ dw,
                                   const double *__restrict__ isn, int64_t n_bins, double df, double L,
                                   double2 *__restrict__ dwp, double2 *__restrict__ fw, uint32_t *__restrict__ err_bits)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_bins) return;
    const double f = freq[i];
    uint32_t err = 0;
    if (!(f > 0.0) || !isfinite(f)) err |= ERR_FREQ_NONPOS;
    if (i > 0 && !(f > freq[i - 1])) err |= ERR_FREQ_ORDER;
    if (n_bins > 1 && !(fabs(f - (freq[0] + (double)i * df)) <= 1e-6 * df)) err |= ERR_FREQ_UNIFORM;
    const double dr = dw[2 * i], di = dw[2 * i + 1], w = isn[i];
    if (!isfinite(dr) || !isfinite(di)) err |= ERR_DW_NONFINITE;
    if (!isfinite(w)) err |= ERR_ISN_NONFINITE;
    else if (!(w > 0.0)) err |= ERR_ISN_NONPOS;
    if (err) { atomicOr(err_bits, err); return; }

    double s2x, c2x;
    sincos(2.0 * (kPi * f * L / kC), &s2x, &c2x);          // the same expression as fill_basis_row's T_S2X, T_C2X
    // conj(K_f) = 2 sin 2x (cos 2x + i sin 2x), |K_f|^2 = 4 sin^2 2x   (K_f = -i (1 - z^2))
    const double amp = 4.0 * df * pow(f, -7.0 / 6.0);
    const double kr = 2.0 * s2x * c2x, ki = 2.0 * s2x * s2x;
    dwp[i] = make_double2(amp * (dr * kr - di * ki), amp * (dr * ki + di * kr));
    fw[i] = make_double2(f, 4.0 * df * pow(f, -7.0 / 3.0) * (4.0 * s2x * s2x) * w);
}

cudaError_t launch_build_table(const double *freq, const double *dw, const double *isn, int64_t n_bins,
                               double df, double arm_length_m, double *dwp, double *fw, uint32_t *err_bits,
                               cudaStream_t st)
{
    const int nt = 256;
    const int64_t nb = (n_bins + nt - 1) / nt;
    build_table_kernel<<<(unsigned)nb, nt, 0, st>>>(freq, dw, isn, n_bins, df, arm_length_m,
                                                    reinterpret_cast<double2 *>(dwp), reinterpret_cast<double2 *>(fw),
                                                    err_bits);
    return cudaGetLastError();
}

// =================================================================================================
// a1: per-particle coefficients (PAPER.md:404 Eq. A3 with readings A1-A3; :71 parameter meanings)
// =================================================================================================
// Particles are evaluated in SLOTS sorted by chirp mass (rank_kernel below): the 128 particles of a CTA then
// sweep t_f at nearly the same rate, so the stride selection is not held back by one low-mass particle
// per group.  slot_of == nullptr means the identity (template dump).  perm[slot] = particle, -1 for padding.
__global__ void prologue_kernel(const double *__restrict__ params, int64_t P, int64_t P_pad, double f_ref,
                                double kappa, const int32_t *__restrict__ slot_of, double *__restrict__ coef,
                                int32_t *__restrict__ valid, int32_t *__restrict__ perm)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P_pad) return;
    const int64_t slot = (p < P && slot_of != nullptr) ? (int64_t)slot_of[p] : p;
    double c[kNCoef];
#pragma unroll
    for (int j = 0; j < kNCoef; ++j) c[j] = 0.0;
    int ok = 0;
    if (p < P) {
        const double tc = params[6 * p + 0], Mc = params[6 * p + 1], eta = params[6 * p + 2];
        const double theta = params[6 * p + 3], phi = params[6 * p + 4], e0 = params[6 * p + 5];
        ok = isfinite(tc) && isfinite(Mc) && isfinite(eta) && isfinite(theta) && isfinite(phi) && isfinite(e0) &&
             (Mc > 0.0) && (eta > 0.0) && (eta <= 0.25) && (e0 >= 0.0);          // same rule as particle_ok()
        if (ok) {
            const double pi = kPi;
            const double Mcs = Mc * kGMsunC3;
            const double M = Mcs * pow(eta, -0.6);
            const double V = cbrt(pi * M);                                    // v = V f^(1/3)
            const double Kq = (3.0 / 128.0) * pow(pi * Mcs, -5.0 / 3.0) * (2.0 / pi);   // quarter turns
            const double V2 = V * V, V3 = V2 * V, V4 = V2 * V2, V5 = V4 * V, V6 = V3 * V3;
            const double lnV = log(V);
            const double al2 = 3715.0 / 756.0 + 55.0 * eta / 9.0;
            const double al3 = -16.0 * pi;
            const double al4 = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0;
            const double a5c = pi * (38645.0 / 756.0 - 65.0 * eta / 9.0);    // alpha_5 = a5c (1 + 3 ln(v/v_lso))
            const double a6c = 11583231236531.0 / 4694215680.0 - 640.0 * pi * pi / 3.0 - 6848.0 * kEulerGamma / 21.0 +
                               eta * (-15737765635.0 / 3048192.0 + 2255.0 * pi * pi / 12.0) +
                               76055.0 * eta * eta / 1728.0 - 127825.0 * eta * eta * eta / 1296.0;
            const double ln_vlso = -0.5 * log(6.0);
            c[0] = 4.0 * tc;                                                   // 2 pi f tc
            c[1] = -0.5 + Kq * V5 * a5c * (1.0 + 3.0 * lnV - 3.0 * ln_vlso);   // -pi/4 + constant part of k = 5
            c[2] = Kq * V5 * a5c;                                              // ln f
            c[3] = Kq;                                                         // f^(-5/3), alpha_0 = 1
            c[4] = Kq * al2 * V2;                                              // f^(-1)
            c[5] = Kq * al3 * V3;                                              // f^(-2/3)
            c[6] = Kq * al4 * V4;                                              // f^(-1/3)
            c[7] = Kq * V6 * (a6c - (6848.0 / 21.0) * (log(4.0) + lnV));       // f^(1/3)
            c[8] = -Kq * V6 * (6848.0 / 63.0);                                 // f^(1/3) ln f
            c[9] = -Kq * (2355.0 / 1462.0) * e0 * e0 * pow(f_ref, 19.0 / 9.0); // f^(-34/9)  (reading A3)
            c[10] = 4.0 * tc / kYear + 2.0 * kappa / pi;                       // a0
            double st, ct, sp, cp;
            sincos(theta, &st, &ct);
            sincos(phi, &sp, &cp);
            c[11] = -st * cp; c[12] = -st * sp; c[13] = -ct;                   // k (propagation direction)
            c[14] = ct * cp;  c[15] = ct * sp;  c[16] = -st;                   // u
            c[17] = sp;       c[18] = -cp;      c[19] = 0.0;                   // v
        }
    }
#pragma unroll
    for (int j = 0; j < kNCoef; ++j) coef[(int64_t)j * P_pad + slot] = c[j];
    valid[slot] = ok;
    if (perm != nullptr) perm[slot] = (p < P) ? (int32_t)p : -1;
}

__device__ __forceinline__ bool particle_ok(const double *__restrict__ q)
{
    return isfinite(q[0]) && isfinite(q[1]) && isfinite(q[2]) && isfinite(q[3]) && isfinite(q[4]) && isfinite(q[5]) &&
           (q[1] > 0.0) && (q[2] > 0.0) && (q[2] <= 0.25) && (q[5] >= 0.0);
}

// slot_of[i] = rank of particle i by (chirp mass rounded to float, index): a stable, deterministic order -- the keys
// are computed once (rank_key_kernel), then ranked by brute force (P <= 16384: one launch of P^2 integer comparisons
// through shared-memory tiles) or by a stable radix sort of (key, index) pairs (cub, larger batches: the same order).
// Invalid particles sort last.
// band_T > 0 (row f2; band_T = the observation time, [band_f0, band_f1] = the grid): the key is the Newtonian
// estimate of the template's frequency at t = 0, clipped to the grid,
// f(t) = (1/pi) (5 / (256 (t_c - t)))^(3/8) (G M_c / c^3)^(-5/8); a second pass (rank_key2) re-orders blocks of 256
// slots by the frequency at t = T.  Only the ORDER matters: the bands themselves come from band_kernel.
__device__ __forceinline__ uint32_t rank_key(const double *__restrict__ q, double band_T, double band_f0, double band_f1)
{
    if (!particle_ok(q)) return 0xFFFFFFFFu;
    if (!(band_T > 0.0)) return __float_as_uint((float)q[1]);
    const double tc = q[0];
    if (!(tc > 0.0)) return 0u;
    const double m = pow(q[1] * kGMsunC3, -0.625) * (1.0 / kPi) * pow(5.0 / 256.0, 0.375);
    return __float_as_uint((float)fmin(fmax(m * pow(tc, -0.375), band_f0), band_f1));      // f(t = 0), clipped to the grid
}

// Row f2, second key: blocks of `block` consecutive slots of the first order (by the lower end of the band) are
// re-ordered by the UPPER end f(t = T), so that the 32 templates of a warp have bands that nearly coincide at both ends
// (a warp walks the union of its lanes' bands).  key = block number x 2^20 + the upper end on a 2^20-step scale.
__device__ __forceinline__ uint32_t rank_key2(const double *__restrict__ q, int32_t slot1, int32_t block, double band_T,
                                              double band_f0, double band_f1)
{
    if (!particle_ok(q)) return 0xFFFFFFFFu;
    const double tc = q[0];
    double fb = band_f1;
    if (tc > band_T) {
        const double m = pow(q[1] * kGMsunC3, -0.625) * (1.0 / kPi) * pow(5.0 / 256.0, 0.375);
        fb = fmin(fmax(m * pow(tc - band_T, -0.375), band_f0), band_f1);
    } else if (!(tc > 0.0)) fb = band_f0;
    const double u = band_f1 > band_f0 ? (fb - band_f0) / (band_f1 - band_f0) : 0.0;
    return (uint32_t)(slot1 / block) * (1u << 20) + (uint32_t)(u * 1048575.0);
}

// slot1 == nullptr: first key; else the second key of row f2 (see rank_key2)
__global__ void __launch_bounds__(256) rank_key_kernel(const double *__restrict__ params, int32_t P, double band_T,
                                                       double band_f0, double band_f1, const int32_t *__restrict__ slot1,
                                                       int32_t block, uint32_t *__restrict__ keys,
                                                       int32_t *__restrict__ index)
{
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= P) return;
    keys[i] = slot1 == nullptr ? rank_key(params + 6 * (int64_t)i, band_T, band_f0, band_f1)
                               : rank_key2(params + 6 * (int64_t)i, slot1[i], block, band_T, band_f0, band_f1);
    if (index != nullptr) index[i] = i;
}

// brute-force rank of the keys (P^2 integer comparisons through shared-memory tiles), for P <= kRankBrute: blockIdx.y
// splits the keys a thread compares its own with; the partial counts are added with integer atomics (slot_of zeroed
// by the caller), so the result does not depend on the order
__global__ void __launch_bounds__(256) rank_kernel(const uint32_t *__restrict__ keys, int32_t P,
                                                   int32_t *__restrict__ slot_of)
{
    __shared__ uint32_t skey[256];
    const int i = blockIdx.x * 256 + threadIdx.x;
    const uint32_t my = i < P ? keys[i] : 0xFFFFFFFFu;
    int rank = 0;
    for (int j0 = blockIdx.y * 256; j0 < P; j0 += gridDim.y * 256) {
        const int j = j0 + threadIdx.x;
        __syncthreads();
        skey[threadIdx.x] = j < P ? keys[j] : 0xFFFFFFFFu;
        __syncthreads();
        const int n = min(256, P - j0);
        for (int t = 0; t < n; ++t) {
            const uint32_t kt = skey[t];
            rank += (kt < my) || (kt == my && j0 + t < i);
        }
    }
    if (i < P && rank != 0) atomicAdd(&slot_of[i], rank);
}

// slot_of[particle] = position of the particle in the list sorted by (key, index)
__global__ void scatter_slots_kernel(const int32_t *__restrict__ sorted_index, int32_t P, int32_t *__restrict__ slot_of)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < P) slot_of[sorted_index[s]] = s;
}

constexpr int64_t kRankBrute = 16384;

// bytes of scratch launch_prologue needs for P particles: keys [P] (+ for large batches: sorted keys, indices in and
// out, and the radix sort's own temporary storage)
size_t prologue_scratch_bytes(int64_t P)
{
    size_t n = ((size_t)P * sizeof(uint32_t) + 255) / 256 * 256;
    if (P > kRankBrute) {
        size_t tmp = 0;
        cub::DeviceRadixSort::SortPairs(nullptr, tmp, (const uint32_t *)nullptr, (uint32_t *)nullptr, (const int32_t *)nullptr,
                                        (int32_t *)nullptr, (int)P);
        n += n + 2 * (((size_t)P * sizeof(int32_t) + 255) / 256 * 256) + tmp + 256;
    }
    return n;
}

cudaError_t launch_prologue(const double *params, int64_t P, int64_t P_pad, double f_ref_e0, double kappa,
                            int32_t *slot_of, const double *rank_band, void *scratch, double *coef, int32_t *valid,
                            int32_t *perm, cudaStream_t st)
{
    if (slot_of != nullptr) {
        const size_t kb = ((size_t)P * sizeof(uint32_t) + 255) / 256 * 256, ib = ((size_t)P * sizeof(int32_t) + 255) / 256 * 256;
        unsigned char *base = static_cast<unsigned char *>(scratch);
        uint32_t *keys = reinterpret_cast<uint32_t *>(base);
        const bool big = P > kRankBrute;
        int32_t *idx_in = big ? reinterpret_cast<int32_t *>(base + 2 * kb) : nullptr;
        const double bT = rank_band ? rank_band[0] : 0.0, bf0 = rank_band ? rank_band[1] : 0.0, bf1 = rank_band ? rank_band[2] : 0.0;
        int32_t block = 256;                                 // row f2: slots re-ordered by the upper band end inside blocks
        while ((P + block - 1) / block > 4095) block *= 2;   // (the block number has 12 bits of the second key)
        for (int pass = 0; pass < (rank_band ? 2 : 1); ++pass) {
            rank_key_kernel<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(params, (int32_t)P, bT, bf0, bf1,
                                                                         pass ? slot_of : nullptr, block, keys, idx_in);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            if (!big) {
                const unsigned nb = (unsigned)((P + 255) / 256);
                if ((e = cudaMemsetAsync(slot_of, 0, (size_t)P * sizeof(int32_t), st)) != cudaSuccess) return e;
                rank_kernel<<<dim3(nb, nb < 16 ? nb : 16), 256, 0, st>>>(keys, (int32_t)P, slot_of);
            } else {
                // stable LSD radix sort of (key, index): the same order as the brute-force rank (ties by index)
                uint32_t *keys_out = reinterpret_cast<uint32_t *>(base + kb);
                int32_t *idx_out = reinterpret_cast<int32_t *>(base + 2 * kb + ib);
                void *tmp = base + 2 * kb + 2 * ib;
                size_t tmp_bytes = 0;
                cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys_out, idx_in, idx_out, (int)P);
                e = cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys_out, idx_in, idx_out, (int)P, 0, 32, st);
                if (e != cudaSuccess) return e;
                scatter_slots_kernel<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(idx_out, (int32_t)P, slot_of);
            }
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
    }
    const int nt = 128;
    prologue_kernel<<<(unsigned)((P_pad + nt - 1) / nt), nt, 0, st>>>(params, P, P_pad, f_ref_e0, kappa, slot_of, coef,
                                                                      valid, perm);
    return cudaGetLastError();
}

// =================================================================================================
// a2-a5: the fused main kernel
// =================================================================================================
size_t main_kernel_smem_bytes() { return sizeof(MainSmem); }

// The direct kernel: every bin of a work item evaluated in full.  Persistent CTAs walk the list of work
// items the stride selection left to it (schedule_kernel: items for which no interpolation stride meets
// the error bound -- all of config 0, partitions shorter than 8 bins); an empty list costs one read.
template <bool AET>
__device__ __forceinline__ void main_kernel_body(const MainArgs &a)
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

    for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const int item = a.direct_list[it];
        const int grp = item / a.n_seg;
        const int seg = item - grp * a.n_seg;
        const int64_t p = (int64_t)grp * kThreads + tid;       // < P_pad by construction

        const int lo = a.seg_edge[seg], hi = a.seg_edge[seg + 1];
        const int n_bins = hi - lo;
        const int n_tiles = (n_bins + kTileBins - 1) / kTileBins;
        const BinSource src{reinterpret_cast<const double2 *>(a.dwp), reinterpret_cast<const double2 *>(a.fw)};

        if (tid == 0) ring_prologue(sm, src, lo, n_bins, n_tiles, g0);

        // per-particle coefficients (a1), coalesced
        double c[kNCoef];
#pragma unroll
        for (int j = 0; j < kNCoef; ++j) c[j] = a.coef[(int64_t)j * a.P_pad + p];

        double acc[kNAcc];
#pragma unroll
        for (int j = 0; j < kNAcc; ++j) acc[j] = 0.0;
        bool need_c = true;
        double c_re = 0.0, c_im = 0.0;

        for (int t = 0; t < n_tiles; ++t) {
            const int nb = min(kTileBins, n_bins - t * kTileBins);
            const double *tile = ring_wait(sm, g0 + t, nb, a.arm_length_m);
            if (tid == 0 && t + kStages < n_tiles) ring_issue(sm, src, lo, n_bins, g0, t + kStages);   // its slot is free: expanded
            double in[kNAcc];
#pragma unroll
            for (int j = 0; j < kNAcc; ++j) in[j] = 0.0;

#pragma unroll 1
            for (int b = 0; b < nb; ++b) {
                const double2 *row = reinterpret_cast<const double2 *>(tile + b * kTabW);
                const double2 dwv = row[10];
                double psi, sps, cps, tpr, tpi, tcr, tci;
                bin_template<AET>(row, c, a.orb, psi, sps, cps, tpr, tpi, tcr, tci);

                // ---- a4: inner products (Eq. 4 :66, Eq. 8-9 :89-91, Eq. 12 :117) in the basis (u_+, u_x - c u_+),
                // c = T'_x / T'_+ at the work item's first bin (hazard H3)
                if (need_c) {
                    need_c = false;
                    choose_basis(tpr, tpi, tcr, tci, c_re, c_im);
                }
                const double qr = fma(dwv.x, cps, -dwv.y * sps);               // dw' exp(+i Psi)
                const double qi = fma(dwv.x, sps, dwv.y * cps);
                accumulate_bin(qr, qi, row[11].x, tpr, tpi, tcr, tci, c_re, c_im, in);
            }
#pragma unroll
            for (int j = 0; j < kNAcc; ++j) acc[j] += in[j];
        }
        g0 += n_tiles;

        double *out = a.partial + ((int64_t)seg * kNPartial) * a.P_pad + p * a.part_sp;
#pragma unroll
        for (int j = 0; j < kNAcc; ++j) out[(int64_t)j * a.part_sk] = acc[j];
        out[(int64_t)8 * a.part_sk] = c_re;
        out[(int64_t)9 * a.part_sk] = c_im;
    }
}

__global__ void __launch_bounds__(kThreads) fstat_main_kernel(const __grid_constant__ MainArgs a)
{
    main_kernel_body<false>(a);
}

__global__ void __launch_bounds__(kThreads) fstat_main_aet_kernel(const __grid_constant__ MainArgs a)
{
    main_kernel_body<true>(a);
}

cudaError_t main_kernel_configure()
{
    cudaError_t e = cudaFuncSetAttribute(fstat_main_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(MainSmem));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(fstat_main_aet_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)sizeof(MainSmem));
}

cudaError_t launch_main(const MainArgs &a, cudaStream_t st)
{
    int64_t n_cta = (int64_t)a.n_groups * a.n_seg;
    if (n_cta > a.max_ctas) n_cta = a.max_ctas;
    if (a.aet) fstat_main_aet_kernel<<<(unsigned)n_cta, kThreads, sizeof(MainSmem), st>>>(a);
    else fstat_main_kernel<<<(unsigned)n_cta, kThreads, sizeof(MainSmem), st>>>(a);
    return cudaGetLastError();
}

// =================================================================================================
// Template dump (not on the hot path): u_P(f_k) = f^(-7/6) K_f T'_P exp(-i psi) for ONE particle over the
// whole grid, one thread per bin (its row expanded in registers), through the same bin_template() the main kernel uses.  Serves
// fstat_eval_template (injection synthesis, element-wise parity tests of a2/a3).
// =================================================================================================
template <bool AET>
__global__ void __launch_bounds__(128) template_kernel(const double2 *__restrict__ fw, double L,
                                                       const double *__restrict__ coef, int64_t P_pad,
                                                       int64_t n_bins, const __grid_constant__ OrbitCoef orb,
                                                       double2 *__restrict__ u_plus, double2 *__restrict__ u_cross)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_bins) return;
    double c[kNCoef];
#pragma unroll
    for (int j = 0; j < kNCoef; ++j) c[j] = coef[(int64_t)j * P_pad];
    __align__(16) double rowbuf[kTabW];
    const double f = fw[i].x;
    fill_basis_row(f, L, rowbuf);
    const double2 *row = reinterpret_cast<const double2 *>(rowbuf);
    double psi, sps, cps, tpr, tpi, tcr, tci;
    bin_template<AET>(row, c, orb, psi, sps, cps, tpr, tpi, tcr, tci);
    const double amp = pow(f, -7.0 / 6.0);
    const double c2x = row[9].x, s2x = row[9].y;
    // K_f = 2 sin(2x) exp(-2 i x);  carrier exp(-i psi) = cps - i sps
    const double kr = 2.0 * s2x * c2x * amp, ki = -2.0 * s2x * s2x * amp;
    const double er = kr * cps + ki * sps, ei = ki * cps - kr * sps;      // amp K_f exp(-i psi)
    u_plus[i] = make_double2(er * tpr - ei * tpi, er * tpi + ei * tpr);
    u_cross[i] = make_double2(er * tcr - ei * tci, er * tci + ei * tcr);
}

cudaError_t launch_template(const double *fw, double arm_length_m, const double *coef, int64_t P_pad, int64_t n_bins,
                            const OrbitCoef &orb, int32_t aet, double *u_plus, double *u_cross, cudaStream_t st)
{
    const int nt = 128;
    const unsigned nb = (unsigned)((n_bins + nt - 1) / nt);
    const double2 *fw2 = reinterpret_cast<const double2 *>(fw);
    if (aet)
        template_kernel<true><<<nb, nt, 0, st>>>(fw2, arm_length_m, coef, P_pad, n_bins, orb,
                                                 reinterpret_cast<double2 *>(u_plus), reinterpret_cast<double2 *>(u_cross));
    else
        template_kernel<false><<<nb, nt, 0, st>>>(fw2, arm_length_m, coef, P_pad, n_bins, orb,
                                                  reinterpret_cast<double2 *>(u_plus), reinterpret_cast<double2 *>(u_cross));
    return cudaGetLastError();
}

// =================================================================================================
// a6: epilogue.  2 F_k = z^H G^-1 z, G = [[m_pp, conj(m_pc)], [m_pc, m_cc]]  (the 4x4 real system of
// PAPER.md:85 Eq. 7 is the real embedding of this 2x2 Hermitian one).  Evaluated
// by Gram-Schmidt: 2 F_k = |z_+|^2/m_pp + |z_x - (m_pc/m_pp) z_+|^2 / (m_cc - |m_pc|^2/m_pp).
// Rank-deficient G (reading A15): only the non-degenerate direction(s) contribute.
// Grid = particle tiles (x) by partition chunks (y); block = 32 particles (x) by 8 lanes (y).
//   SEG_PAR = false (many partitions, ~1 segment each): lane y owns partitions y, y + 8, ... of the chunk;
//   SEG_PAR = true  (few partitions, many segments each): the 8 lanes split the segments of one partition
//                   and are combined through shared memory in a fixed order.
// Every sum has a fixed order, so F and F_k are bit-reproducible.  F = sum_k F_k (Eq. 11 :110, reading
// A12) is written directly when there is one chunk, else as per-chunk sums that fsum_kernel adds up.
// =================================================================================================
constexpr int kEpiX = 32, kEpiY = 8;

template <bool SEG_PAR>
__global__ void __launch_bounds__(kEpiX *kEpiY) epilogue_kernel(const PartialSet ps,
                                                               const int32_t *__restrict__ part_seg,
                                                               const int32_t *__restrict__ valid, int64_t P,
                                                               const int32_t *__restrict__ perm, int64_t P_pad,
                                                               int32_t n_part, int32_t chunk, int32_t chunk0,
                                                               int32_t n_chunk_total, double *__restrict__ Fout,
                                                               double *__restrict__ Fk)
{
    __shared__ int32_t sPerm[kEpiX];
    __shared__ double sF[kEpiY][kEpiX];
    __shared__ double sT[kEpiY][kEpiX + 1];
    __shared__ double sV[SEG_PAR ? kEpiY : 1][kNAcc][kEpiX];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int64_t p0 = (int64_t)blockIdx.x * kEpiX;
    const int64_t p = p0 + tx;                            // slot; the particle it holds is perm[p]
    const bool live = p < P;
    const bool ok = live && valid[p] != 0;
    if (threadIdx.y == 0) sPerm[tx] = live ? perm[p] : -1;
    __syncthreads();
    const double ninf = -INFINITY;
    const int cy = (int)blockIdx.y + chunk0;              // chunk of partitions (a launch may cover a range of them)
    const int k_lo = cy * chunk, k_hi = min(n_part, k_lo + chunk);
    double fsum = 0.0;
    for (int k0 = k_lo; k0 < k_hi; k0 += kEpiY) {
        double fk = 0.0;
        if (!SEG_PAR) {
            const int k = k0 + ty;
            if (k < k_hi && live) {
                const int s0 = part_seg[k], s1 = part_seg[k + 1];
                double v[kNAcc];
#pragma unroll
                for (int j = 0; j < kNAcc; ++j) v[j] = 0.0;
                const double cs_r = ps.p[0][((int64_t)s0 * kNPartial + 8) * P_pad + p];   // common basis: the first
                const double cs_i = ps.p[0][((int64_t)s0 * kNPartial + 9) * P_pad + p];   // segment's (of channel 0)
                for (int c = 0; c < ps.n; ++c)            // Eq. 3 :62: N and M add over the TDI channels
                    for (int s = s0; s < s1; ++s) add_segment(ps.p[c], s, P_pad, P_pad, 1, p, cs_r, cs_i, v);
                fk = ok ? 0.5 * two_F(v) : ninf;
                if (ok) fsum += fk;
            }
        } else {
            // partitions k0 .. k0+7 one after the other; lane ty sums segments s0 + ty, s0 + ty + 8, ...
            for (int kk = 0; kk < kEpiY && k0 + kk < k_hi; ++kk) {
                const int s0 = part_seg[k0 + kk], s1 = part_seg[k0 + kk + 1];
                double v[kNAcc];
#pragma unroll
                for (int j = 0; j < kNAcc; ++j) v[j] = 0.0;
                if (live) {
                    const double cs_r = ps.p[0][((int64_t)s0 * kNPartial + 8) * P_pad + p];
                    const double cs_i = ps.p[0][((int64_t)s0 * kNPartial + 9) * P_pad + p];
                    for (int c = 0; c < ps.n; ++c)
                        for (int s = s0 + ty; s < s1; s += kEpiY)
                            add_segment(ps.p[c], s, P_pad, P_pad, 1, p, cs_r, cs_i, v);
                }
#pragma unroll
                for (int j = 0; j < kNAcc; ++j) sV[SEG_PAR ? ty : 0][j][tx] = v[j];
                __syncthreads();
                if (ty == kk) {                           // lane kk finishes partition k0 + kk
#pragma unroll
                    for (int j = 0; j < kNAcc; ++j) {
                        double a = 0.0;
#pragma unroll
                        for (int y = 0; y < kEpiY; ++y) a += sV[SEG_PAR ? y : 0][j][tx];
                        v[j] = a;
                    }
                    if (live) {
                        fk = ok ? 0.5 * two_F(v) : ninf;
                        if (ok) fsum += fk;
                    }
                }
                __syncthreads();
            }
        }
        if (Fk != nullptr) {                              // transpose through shared memory: coalesced rows
            sT[ty][tx] = fk;
            __syncthreads();
            // 256 threads write a 32 (particles) x 8 (partitions) tile: thread -> (particle = id / 8, k = id % 8)
            const int id = ty * kEpiX + tx;
            const int pp = id / kEpiY, kk = id % kEpiY;
            if (p0 + pp < P && k0 + kk < k_hi) Fk[(int64_t)sPerm[pp] * n_part + k0 + kk] = sT[kk][pp];
            __syncthreads();
        }
    }
    sF[ty][tx] = fsum;
    __syncthreads();
    if (ty == 0 && live) {
        double s = 0.0;
#pragma unroll
        for (int y = 0; y < kEpiY; ++y) s += sF[y][tx];
        if (n_chunk_total == 1) Fout[sPerm[tx]] = ok ? s : ninf;            // F itself
        else Fout[(int64_t)cy * P_pad + p] = s;                              // chunk sum, see fsum_kernel
    }
}

__global__ void fsum_kernel(const double *__restrict__ Fpart, const int32_t *__restrict__ valid,
                            const int32_t *__restrict__ perm, int64_t P, int64_t P_pad, int32_t n_chunk,
                            double *__restrict__ F)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    double s = 0.0;
    for (int c = 0; c < n_chunk; ++c) s += Fpart[(int64_t)c * P_pad + p];
    F[perm[p]] = valid[p] != 0 ? s : -INFINITY;
}

// =================================================================================================
// Extrinsic amplitudes (SURVEY row f3; PAPER.md:96 Eq. 10, :413 Eq. B1): a = M^-1 N per partition, from the
// same eight sums.  With alpha_+ = a_1 + i a_3, alpha_x = a_2 + i a_4 (h = alpha_+ u_+ + alpha_x u_x) the
// stationarity condition of Eq. 6 is the 2x2 Hermitian system  G alpha = z,  G = [[m_pp, conj(m_pc)],
// [m_pc, m_cc]], solved by the same Gram-Schmidt steps as the epilogue.  Rank-deficient G: the component
// along the degenerate direction is set to 0.  One thread per (slot, partition).
// =================================================================================================
__global__ void __launch_bounds__(128) amplitude_kernel(const double *__restrict__ partial,
                                                        const int32_t *__restrict__ part_seg,
                                                        const int32_t *__restrict__ valid,
                                                        const int32_t *__restrict__ perm, int64_t P, int64_t P_pad,
                                                        int32_t n_part, double *__restrict__ amp)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const bool ok = valid[p] != 0;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    for (int k = blockIdx.y; k < n_part; k += gridDim.y) {
        double v[kNAcc];
#pragma unroll
        for (int j = 0; j < kNAcc; ++j) v[j] = 0.0;
        const int s_first = part_seg[k];
        const double cs_r = partial[((int64_t)s_first * kNPartial + 8) * P_pad + p];
        const double cs_i = partial[((int64_t)s_first * kNPartial + 9) * P_pad + p];
        for (int s = s_first; s < part_seg[k + 1]; ++s) add_segment(partial, s, P_pad, P_pad, 1, p, cs_r, cs_i, v);
        double apr, acr, api, aci;
        solve_amplitudes(v, cs_r, cs_i, apr, acr, api, aci);
        double *out = amp + ((int64_t)perm[p] * n_part + k) * 4;
        out[0] = ok ? apr : nan;     // a_1
        out[1] = ok ? acr : nan;     // a_2
        out[2] = ok ? api : nan;     // a_3
        out[3] = ok ? aci : nan;     // a_4
    }
}

cudaError_t launch_amplitudes(const double *partial, const int32_t *part_seg, const int32_t *valid,
                              const int32_t *perm, int64_t P, int64_t P_pad, int32_t n_part, double *amp,
                              cudaStream_t st)
{
    const dim3 grd((unsigned)((P + 127) / 128), (unsigned)(n_part < 32768 ? n_part : 32768));
    amplitude_kernel<<<grd, 128, 0, st>>>(partial, part_seg, valid, perm, P, P_pad, n_part, amp);
    return cudaGetLastError();
}

int32_t epilogue_chunks(int64_t P, int32_t n_part, int32_t *chunk_out)
{
    // enough blocks to fill the machine: particle tiles x partition chunks >= ~4 per SM; chunks of >= 8
    const int64_t tiles = (P + kEpiX - 1) / kEpiX;
    int64_t want = (4 * 148 + tiles - 1) / tiles;
    int64_t max_chunks = (n_part + kEpiY - 1) / kEpiY;
    if (want > max_chunks) want = max_chunks;
    if (want < 1) want = 1;
    int32_t chunk = (int32_t)((n_part + want - 1) / want);
    chunk = ((chunk + kEpiY - 1) / kEpiY) * kEpiY;
    *chunk_out = chunk;
    return (n_part + chunk - 1) / chunk;
}

// chunks [chunk_lo, chunk_hi) of the partitions only, without the final sum over chunks (the host-buffer call overlaps
// the copy of one range of F_k with the main kernels of the next, fstat_eval_batch_host)
cudaError_t launch_epilogue_range(const PartialSet &partials, const int32_t *part_seg, const int32_t *valid,
                                  const int32_t *perm, int64_t P, int64_t P_pad, int32_t n_part, int32_t n_seg,
                                  int32_t chunk_lo, int32_t chunk_hi, double *Fpart, double *F, double *Fk, cudaStream_t st)
{
    int32_t chunk = 0;
    const int32_t n_chunk = epilogue_chunks(P, n_part, &chunk);
    if (chunk_lo < 0 || chunk_hi > n_chunk || chunk_lo >= chunk_hi) return cudaErrorInvalidValue;
    const dim3 blk(kEpiX, kEpiY);
    const dim3 grd((unsigned)((P + kEpiX - 1) / kEpiX), (unsigned)(chunk_hi - chunk_lo));
    double *out = (n_chunk == 1) ? F : Fpart;
    if (n_seg >= 4 * n_part)
        epilogue_kernel<true><<<grd, blk, 0, st>>>(partials, part_seg, valid, P, perm, P_pad, n_part, chunk, chunk_lo, n_chunk, out, Fk);
    else
        epilogue_kernel<false><<<grd, blk, 0, st>>>(partials, part_seg, valid, P, perm, P_pad, n_part, chunk, chunk_lo, n_chunk, out, Fk);
    return cudaGetLastError();
}

cudaError_t launch_fsum(const double *Fpart, const int32_t *valid, const int32_t *perm, int64_t P, int64_t P_pad,
                        int32_t n_chunk, double *F, cudaStream_t st)
{
    fsum_kernel<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(Fpart, valid, perm, P, P_pad, n_chunk, F);
    return cudaGetLastError();
}

cudaError_t launch_epilogue(const PartialSet &partials, const int32_t *part_seg, const int32_t *valid,
                            const int32_t *perm, int64_t P, int64_t P_pad, int32_t n_part, int32_t n_seg,
                            double *Fpart, double *F, double *Fk, cudaStream_t st)
{
    int32_t chunk = 0;
    const int32_t n_chunk = epilogue_chunks(P, n_part, &chunk);
    cudaError_t e = launch_epilogue_range(partials, part_seg, valid, perm, P, P_pad, n_part, n_seg, 0, n_chunk, Fpart, F, Fk, st);
    if (e != cudaSuccess || n_chunk == 1) return e;
    return launch_fsum(Fpart, valid, perm, P, P_pad, n_chunk, F, st);
}

// =================================================================================================
// pipe-peak probes: dependent-free instruction streams (8 chains per thread), for the roofline
// denominators.  Thread-level instructions per launch: blocks*256*iters*64.
// =================================================================================================
template <int WHICH>
__global__ void __launch_bounds__(256) probe_kernel(int iters, double *sink)
{
    if (WHICH == 0) {
        double x[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 1.0 + 1e-9 * (threadIdx.x + j);
        const double m = 0.999999999, b = 1e-12;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int j = 0; j < 8; ++j) x[j] = fma(x[j], m, b);
        }
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < 8; ++j) s += x[j];
        if (s == 123.456) sink[0] = s;
    } else if (WHICH == 1) {
        float x[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 1.0f + 1e-6f * (threadIdx.x + j);
        const float m = 0.9999999f, b = 1e-9f;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int j = 0; j < 8; ++j) x[j] = fmaf(x[j], m, b);
        }
        float s = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) s += x[j];
        if (s == 123.456f) sink[0] = s;
    } else if (WHICH == 3) {
        // 8 FP64 FMA : 2 FP32 FMA per round -- what a non-FP64 instruction costs a stream that is bound by the FP64
        // pipe (an FP64 warp instruction occupies the pipe for 2 cycles per SM sub-partition; measured on B200, the
        // other instructions issue in the gaps and cost ~0.2 cycles each at this ratio: profiles/r2.md).  Counted
        // as 64 FP64 instructions per iteration, like WHICH == 0.
        double x[8];
        float y[2];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 1.0 + 1e-9 * (threadIdx.x + j);
        y[0] = 1.0f + 1e-6f * threadIdx.x;
        y[1] = 1.5f + 1e-6f * threadIdx.x;
        const double m = 0.999999999, b = 1e-12;
        const float mf = 0.9999999f, bf = 1e-9f;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int r = 0; r < 8; ++r) {
#pragma unroll
                for (int j = 0; j < 8; ++j) x[j] = fma(x[j], m, b);
                y[0] = fmaf(y[0], mf, bf);
                y[1] = fmaf(y[1], mf, bf);
            }
        }
        double s = (double)(y[0] + y[1]);
#pragma unroll
        for (int j = 0; j < 8; ++j) s += x[j];
        if (s == 123.456) sink[0] = s;
    } else {
        float x[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 0.1f + 1e-3f * (threadIdx.x + j);
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int j = 0; j < 8; ++j) asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(x[j]));
        }
        float s = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) s += x[j];
        if (s == 123.456f) sink[0] = s;
    }
}

cudaError_t launch_probe(int which, int n_blocks, int iters, double *sink, cudaStream_t st)
{
    if (which == 0) probe_kernel<0><<<n_blocks, 256, 0, st>>>(iters, sink);
    else if (which == 1) probe_kernel<1><<<n_blocks, 256, 0, st>>>(iters, sink);
    else if (which == 3) probe_kernel<3><<<n_blocks, 256, 0, st>>>(iters, sink);
    else probe_kernel<2><<<n_blocks, 256, 0, st>>>(iters, sink);
    return cudaGetLastError();
}

}  // namespace fstat
