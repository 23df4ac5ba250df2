// fstat_direct.cuh -- device pieces shared by the two kernels that evaluate the model at every bin
// (fstat_main_kernel in fstat_kernels.cu, fstat_band_kernel in fstat_band.cu) and by the epilogues:
// the TMA ring of per-bin inputs and their expansion into rows, one (particle, bin) of the template, and 2 F_k from
// the eight sums.
#pragma once
#include "fstat_device.cuh"
#include "fstat_internal.h"
#include "fstat_model.cuh"

namespace fstat {

// The full-model kernels stream their bins through shared memory in tiles of kTileBins: the per-bin inputs -- the folded
// data dw' (16 bytes per bin) and the pair (f, w') (16 bytes per bin) -- arrive by TMA bulk copies into a ring of
// staging slots, and the CTA expands each tile into the 24-column rows model_eval reads (the particle-independent
// basis of the phase, its derivative and the arm phases: fill_basis_row, one thread per bin), so that no 192-byte
// per-bin table has to live in HBM.  The expansion costs ~1.5 % of a tile's evaluation (64 threads x ~500
// instructions against 128 threads x 64 bins x ~530).
struct __align__(16) MainSmem {
    double tile[kTileBins * kTabW];            // the expanded rows of the tile being evaluated
    double2 stage[kStages][2][kTileBins];      // [slot][0: dw', 1: (f, w')][bin]
    uint64_t full[kStages];
};

struct BinSource {
    const double2 *dwp;    // [n_bins] folded data
    const double2 *fw;     // [n_bins] (f, w')
};

// (one elected thread issues the TMA bulk copies; g0 = tiles this CTA has consumed so far = ring position of the work
// item's first tile; lo = the work item's first bin)
__device__ __forceinline__ void ring_issue(MainSmem &sm, const BinSource &src, int lo, int n_bins, int g0, int t)
{
    const int slot = (g0 + t) % kStages;
    const int nb = min(kTileBins, n_bins - t * kTileBins);
    const uint32_t bytes = (uint32_t)nb * (uint32_t)sizeof(double2);
    mbar_expect_tx(&sm.full[slot], 2 * bytes);
    tma_load_1d(sm.stage[slot][0], src.dwp + lo + t * kTileBins, bytes, &sm.full[slot]);
    tma_load_1d(sm.stage[slot][1], src.fw + lo + t * kTileBins, bytes, &sm.full[slot]);
}

__device__ __forceinline__ void ring_prologue(MainSmem &sm, const BinSource &src, int lo, int n_bins, int n_tiles, int g0)
{
#pragma unroll
    for (int s = 0; s < kStages; ++s)
        if (s < n_tiles) ring_issue(sm, src, lo, n_bins, g0, s);
}

// Wait for tile g of the ring and expand it into sm.tile (all threads of the CTA call this; two barriers: the previous
// tile's rows are no longer read, the new rows are complete).  Returns the rows.
__device__ __forceinline__ const double *ring_wait(MainSmem &sm, int g, int nb, double L)
{
    const int slot = g % kStages;
    mbar_wait(&sm.full[slot], (uint32_t)((g / kStages) & 1));
    __syncthreads();
    const int b = threadIdx.x;
    if (b < nb) {
        const double2 dw = sm.stage[slot][0][b], fw = sm.stage[slot][1][b];
        double *row = sm.tile + b * kTabW;
        fill_basis_row(fw.x, L, row);
        row[T_DWR] = dw.x;
        row[T_DWI] = dw.y;
        row[T_W] = fw.y;
    }
    __syncthreads();
    return sm.tile;
}

// One (particle, bin) of the direct kernel: model_eval() plus the linear phase term and the carrier.
// Returns the carrier phase psi (quarter turns, Doppler phase of spacecraft 1 included), its sine and
// cosine, and T'_+ , T'_x.
template <bool AET = false>
__device__ __forceinline__ void bin_template(const double2 *__restrict__ row, const double (&c)[kNCoef],
                                             const OrbitCoef &orb, double &psi_out, double &sps, double &cps,
                                             double &tpr, double &tpi, double &tcr, double &tci)
{
    double psi_nl;
    model_eval<AET>(row, c, orb, psi_nl, tpr, tpi, tcr, tci);
    const double psi = fma(c[0], row[0].x, psi_nl);                  // + 2 pi f t_c
    sincos_qt(psi, sps, cps);
    psi_out = psi;
}

// Basis constant c = T'_x / T'_+ (complex) at one point of a partition, or 0 where T'_+ ~ 0 there.  The sums of a
// partition are kept in the basis (u_+, u_x - c u_+) (hazard H3): F is invariant under
// it, and over a narrow partition u_x is nearly c u_+, so the small remainder is accumulated directly instead of
// being left to cancel in m_cc - |m_pc|^2 / m_pp (normalised determinants down to 3e-12 on config 4).
__device__ __forceinline__ void choose_basis(double pr, double pi, double xr, double xi, double &c_re, double &c_im)
{
    const double n2 = fma(pr, pr, pi * pi), x2 = fma(xr, xr, xi * xi);
    const bool use = n2 > 1e-6 * x2;
    const double inv = use ? 1.0 / n2 : 0.0;
    c_re = fma(xr, pr, xi * pi) * inv;               // T'_x conj(T'_+) / |T'_+|^2
    c_im = fma(xi, pr, -xr * pi) * inv;
}

// One bin of the full-model kernels: q = dw' exp(+i Psi), weight w', response (T'_+, T'_x); the eight sums in the
// basis (u_+, u_x - c u_+)  (Eq. 4 :66, Eq. 8-9 :89-91, Eq. 12 :117).
__device__ __forceinline__ void accumulate_bin(double qr, double qi, double w, double tpr, double tpi, double tcr,
                                               double tci, double c_re, double c_im, double (&in)[kNAcc])
{
    const double xr = tcr - fma(c_re, tpr, -c_im * tpi);              // T'_x - c T'_+
    const double xi = tci - fma(c_re, tpi, c_im * tpr);
    in[0] = fma(qr, tpr, fma(qi, tpi, in[0]));                        // z_+ += q conj(T'_+)
    in[1] = fma(qi, tpr, fma(-qr, tpi, in[1]));
    in[2] = fma(qr, xr, fma(qi, xi, in[2]));                          // z_x
    in[3] = fma(qi, xr, fma(-qr, xi, in[3]));
    in[4] = fma(w, fma(tpr, tpr, tpi * tpi), in[4]);                  // m_pp
    in[5] = fma(w, fma(xr, xr, xi * xi), in[5]);                      // m_cc
    in[6] = fma(w, fma(tpr, xr, tpi * xi), in[6]);                    // m_pc = sum w T'_+ conj(T'_x)
    in[7] = fma(w, fma(tpi, xr, -tpr * xi), in[7]);
}

// 2 F_k = z^H G^-1 z by Gram-Schmidt (Eq. 7 in its 2x2 Hermitian form):
// |z_+|^2/m_pp + |z_x - (m_pc/m_pp) z_+|^2 / (m_cc - |m_pc|^2/m_pp); rank-deficient G (reading A15): only
// the non-degenerate direction(s) contribute.
__device__ __forceinline__ double two_F(const double (&v)[kNAcc])
{
    const double zpr = v[0], zpi = v[1], zcr = v[2], zci = v[3];
    const double mpp = v[4], mcc = v[5], mr = v[6], mi = v[7];
    double twoF = 0.0;
    if (mpp > 0.0) {
        const double inv = 1.0 / mpp;
        twoF = (zpr * zpr + zpi * zpi) * inv;
        const double cr = mr * inv, ci = mi * inv;                      // m_pc / m_pp
        const double schur = mcc - (mr * mr + mi * mi) * inv;
        if (schur > 1e-13 * mcc) {
            const double yr = zcr - (cr * zpr - ci * zpi);
            const double yi = zci - (cr * zpi + ci * zpr);
            twoF += (yr * yr + yi * yi) / schur;
        }
    } else if (mcc > 0.0) {
        twoF = (zcr * zcr + zci * zci) / mcc;
    }
    return twoF;
}

// Add the sums of segment s (stored in its own basis (u_+, u_x - c_s u_+)) to v in the basis with constant
// c*:  u_x - c* u_+ = (u_x - c_s u_+) + D u_+,  D = c_s - c*, so
//   z~* = z~ + conj(D) z_+,   m~*_pc = m~_pc + conj(D) m_pp,   m~*_cc = m~_cc + 2 Re(D m~_pc) + |D|^2 m_pp.
// D is a small difference of nearby ratios: nothing cancels here.
// t = the ten values of a record (eight sums in the basis with constant (t[8], t[9])).
__device__ __forceinline__ void add_record(const double (&t)[kNPartial], double cs_r, double cs_i, double (&v)[kNAcc])
{
    const double dr = t[8] - cs_r, di = t[9] - cs_i;
    v[0] += t[0];
    v[1] += t[1];
    v[2] += fma(dr, t[0], fma(di, t[1], t[2]));
    v[3] += fma(dr, t[1], fma(-di, t[0], t[3]));
    v[4] += t[4];
    v[5] += fma(fma(dr, dr, di * di), t[4], fma(2.0, fma(dr, t[6], -di * t[7]), t[5]));
    v[6] += fma(dr, t[4], t[6]);
    v[7] += fma(-di, t[4], t[7]);
}

// (sk, sp): strides of the record's values and of the slots, (P_pad, 1) or (1, kNPartial), see MainArgs.
__device__ __forceinline__ void add_segment(const double *__restrict__ partial, int s, int64_t P_pad, int64_t sk,
                                            int64_t sp, int64_t p, double cs_r, double cs_i, double (&v)[kNAcc])
{
    const double *src = partial + ((int64_t)s * kNPartial) * P_pad + p * sp;
    double t[kNPartial];
#pragma unroll
    for (int j = 0; j < kNPartial; ++j) t[j] = src[(int64_t)j * sk];
    add_record(t, cs_r, cs_i, v);
}

// Extrinsic amplitudes (Eq. 10): alpha = G^-1 z for the 2x2 Hermitian G of the eight sums v, which are
// in the basis (u_+, u_x - c* u_+); returns a_1 = Re alpha_+, a_2 = Re alpha_x, a_3 = Im alpha_+, a_4 = Im alpha_x
// of the plain basis.  Rank-deficient G: the degenerate component is set to 0 (reading A15).
__device__ __forceinline__ void solve_amplitudes(const double (&v)[kNAcc], double cs_r, double cs_i, double &apr,
                                                 double &acr, double &api, double &aci)
{
    const double zpr = v[0], zpi = v[1], zcr = v[2], zci = v[3];
    const double mpp = v[4], mcc = v[5], mr = v[6], mi = v[7];
    apr = 0.0; api = 0.0; acr = 0.0; aci = 0.0;
    if (mpp > 0.0) {
        const double inv = 1.0 / mpp;
        const double cr = mr * inv, ci = mi * inv;                          // m_pc / m_pp
        const double schur = mcc - (mr * mr + mi * mi) * inv;
        if (schur > 1e-13 * mcc) {
            acr = (zcr - (cr * zpr - ci * zpi)) / schur;                    // alpha_x = (z_x - (m_pc/m_pp) z_+) / schur
            aci = (zci - (cr * zpi + ci * zpr)) / schur;
        }
        apr = (zpr - (mr * acr + mi * aci)) * inv;                          // alpha_+ = (z_+ - conj(m_pc) alpha_x) / m_pp
        api = (zpi - (mr * aci - mi * acr)) * inv;
        // the sums are in the basis (u_+, u_x - c* u_+): h = alpha~_+ u_+ + alpha_x (u_x - c* u_+)
        apr -= cs_r * acr - cs_i * aci;
        api -= cs_r * aci + cs_i * acr;
    } else if (mcc > 0.0) {
        acr = zcr / mcc;
        aci = zci / mcc;
    }
}

}  // namespace fstat
