/*
 * fstat_oracle.c -- plain, slow FP64 CPU oracle for the batched semi-coherent F-statistic of
 * arXiv 2407.10797.  THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call it.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2407_10797_b200/csrc/ and neither includes the other.
 *
 * What it computes is the plain definition: F(Theta_I) = max over the four amplitudes a_i of the
 * log-likelihood ratio (PAPER.md:62 Eq. 3, :77 Eq. 5, :85 Eq. 7), per frequency partition
 * (Eq. 12), summed over partitions (Eq. 11, reading A12: sum, not mean).
 * Steps, in the paper's order, with no blocking / fusion / tables / recurrences:
 *   1. per bin, the SPA phase Psi_0(f) (PAPER.md:404 Eq. A3 with readings A1-A4) and the
 *      time-frequency map t_f = (1/2pi) dPsi_0/df (Eq. 20, reading A5);
 *   2. spacecraft positions at t_f from the analytic orbit to O(e^2) (reading A9);
 *   3. the four one-way link responses and first-generation TDI X (Eq. 15,
 *      :206 Eq. 17 with N = 0 and no d(t) corrections, :229; readings A6, A7, A10);
 *   4. the four real basis templates A^1..A^4 = u_+, u_x, i u_+, i u_x written out to arrays,
 *      u_P = T_P f^(-7/6) exp(-i Psi_0) (PAPER.md:397 Eq. A1, amplitude constant dropped, A21);
 *   5. per partition the 4 + 10 inner products N^i, M^ij by direct summation (Eq. 4 as a
 *      rectangle rule, A16; :89-91 Eq. 8-9), a 4x4 Cholesky solve, F_k = N.a / 2 (Eq. 7, 10).
 * It deliberately does NOT use the 2x2 Hermitian closed form the GPU epilogue uses.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): P1 brute-force maximisation of Lambda(a);
 * P2 zero-noise 2F = rho^2; P3 chi^2(4 N_p) over pure noise; P4 N_p = 1 == coherent; P6 Newtonian
 * closed forms, central differences and 40-digit mpmath spot checks of the phase; P7 orbit against
 * exact Kepler ellipses and arm-length formula; P8 long-wavelength limit and polarisation-rotation
 * invariance of the response; P9 a time-domain simulation of the four links + TDI delays.
 * Row f2 (the paper's own segment limits): oracle_template_band below + band_edges /
 * fstat_bands in oracle.py; pins in tests/test_oracle_bands.py: P11 the band limits against the textbook
 * 2PN time-to-coalescence series and against the power of a time-domain simulated signal, P12 edges on
 * hand-computed integers, P13 zero-noise in-band 2F = <h,h>.
 * Row f4 (Eq. 3 :62, the sum over TDI combinations with independent noise): fstat_batch_channels in oracle.py adds
 * the N and M of this file's oracle_fstat_batch over the channels; pins in tests/test_oracle_channels.py: P14 the
 * cyclic relabelling behind orbit_lambda + 2 pi/3, brute-force maximisation of Eq. 3, zero-noise network SNR.
 * The coefficients the paper does not print (alpha_k, phi_e: "details in [85-88]") are pinned by
 * tests/test_oracle_pn_pins.py against independent statements of that literature: P15 t_f = the 3PN TaylorT2
 * t(v) of ref. [88]; P16 Psi_0 = 2 pi f t(v) - 2 phi_orb(v) - pi/4 with TaylorT2's two series; P17 the eccentric
 * term = Peters' time to coalescence (157/43 e^2, e ~ f^(-19/18)); scratch copies of this file with any one of
 * those constants corrupted fail them.
 * PARITY UNPINNED (stated in DESIGN.md): only what needs the authors' own code and files -- whether THEIR
 * alpha_k / phi_e are these textbook ones, and the paper's absolute SNR values (their PSD file and orbit phase
 * are not available, P10/T8).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_C_SI      299792458.0
#define ORC_GMSUN_C3  4.925490947641267e-6   /* G Msun / c^3  [s] */
#define ORC_AU_M      149597870700.0
#define ORC_YEAR_S    31557600.0
#define ORC_EULER     0.5772156649015329
#define ORC_PI        3.14159265358979323846

typedef struct {
    double f_ref_e0;      /* frequency at which e0 is defined, 0.01 Hz */
    double arm_length_m;  /* 2.5e9 */
    double orbit_kappa;   /* initial orbital phase of the constellation centre */
    double orbit_lambda;  /* initial orientation of the constellation */
    int32_t tdi_channel;  /* 0 X (the paper's), 1 Y, 2 Z, 3 A, 4 E, 5 T (reading A28) */
} oracle_options;

void oracle_default_options(oracle_options *o)
{
    o->f_ref_e0 = 0.01; o->arm_length_m = 2.5e9; o->orbit_kappa = 0.0; o->orbit_lambda = 0.0; o->tdi_channel = 0;
}

/* params: tc [s], Mc [Msun], eta, theta [rad, ecliptic colatitude], phi [rad], e0 */
int oracle_params_valid(const double *p)
{
    for (int i = 0; i < 6; ++i) if (!isfinite(p[i])) return 0;
    if (!(p[1] > 0.0)) return 0;
    if (!(p[2] > 0.0 && p[2] <= 0.25)) return 0;
    if (!(p[5] >= 0.0)) return 0;
    return 1;
}

/* Non-spinning TaylorF2 coefficients alpha_0..alpha_6 at PN velocity v (reading A1). */
void oracle_pn_alpha(double eta, double v, double alpha[7])
{
    const double pi = ORC_PI;
    const double v_lso = 1.0 / sqrt(6.0);
    alpha[0] = 1.0;
    alpha[1] = 0.0;
    alpha[2] = 3715.0 / 756.0 + 55.0 * eta / 9.0;
    alpha[3] = -16.0 * pi;
    alpha[4] = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0;
    alpha[5] = pi * (38645.0 / 756.0 - 65.0 * eta / 9.0) * (1.0 + 3.0 * log(v / v_lso));
    alpha[6] = 11583231236531.0 / 4694215680.0 - 640.0 * pi * pi / 3.0 - 6848.0 * ORC_EULER / 21.0
             + eta * (-15737765635.0 / 3048192.0 + 2255.0 * pi * pi / 12.0)
             + 76055.0 * eta * eta / 1728.0 - 127825.0 * eta * eta * eta / 1296.0
             - (6848.0 / 21.0) * log(4.0 * v);
}

/* Psi_0(f) of Eq. A3 (readings A2-A4: x = v^2, v = (pi M f)^(1/3); phi_e leading order in e0;
 * phi_p, phi_D live in the response) and t_f = (1/2pi) dPsi_0/df (Eq. 20), analytic derivative. */
void oracle_phase(const double *par, double f, const oracle_options *opt, double *psi0, double *t_f)
{
    const double pi = ORC_PI;
    const double tc = par[0], Mc = par[1] * ORC_GMSUN_C3, eta = par[2], e0 = par[5];
    const double M = Mc * pow(eta, -0.6);
    const double v = cbrt(pi * M * f);
    double a[7];
    oracle_pn_alpha(eta, v, a);
    double sum = 0.0;
    for (int k = 0; k <= 6; ++k) sum += a[k] * pow(v, (double)k);
    const double ecc = (2355.0 / 1462.0) * e0 * e0 * pow(opt->f_ref_e0 / f, 19.0 / 9.0);
    const double lead = (3.0 / 128.0) * pow(pi * Mc * f, -5.0 / 3.0);
    *psi0 = 2.0 * pi * f * tc - pi / 4.0 + lead * (sum - ecc);

    /* derivative, term by term.  lead = K f^(-5/3), v = V f^(1/3). */
    const double K = (3.0 / 128.0) * pow(pi * Mc, -5.0 / 3.0);
    const double V = cbrt(pi * M);
    const double a5c = pi * (38645.0 / 756.0 - 65.0 * eta / 9.0);           /* alpha_5 = a5c (1 + 3 ln(v/v_lso)) */
    const double a6c = a[6] + (6848.0 / 21.0) * log(4.0 * v);               /* alpha_6 = a6c - (6848/21) ln(4v)  */
    double d = 0.0;
    d += a[0] * (-5.0 / 3.0) * pow(f, -8.0 / 3.0);
    d += a[2] * pow(V, 2.0) * (-1.0) * pow(f, -2.0);
    d += a[3] * pow(V, 3.0) * (-2.0 / 3.0) * pow(f, -5.0 / 3.0);
    d += a[4] * pow(V, 4.0) * (-1.0 / 3.0) * pow(f, -4.0 / 3.0);
    d += a5c * pow(V, 5.0) / f;                                             /* d/df [3 ln v] = 1/f */
    d += pow(V, 6.0) * pow(f, -2.0 / 3.0) / 3.0 * (a6c - (6848.0 / 21.0) * (log(4.0 * v) + 1.0));
    d += (2355.0 / 1462.0) * e0 * e0 * pow(opt->f_ref_e0, 19.0 / 9.0) * (34.0 / 9.0) * pow(f, -43.0 / 9.0);
    *t_f = tc + K * d / (2.0 * pi);
}

/* Spacecraft positions p[n][xyz] (n = 0,1,2 <-> spacecraft 1,2,3) at time t, metres (reading A9). */
void oracle_orbit(double t, const oracle_options *opt, double p[3][3])
{
    const double R = ORC_AU_M;
    const double e = opt->arm_length_m / (2.0 * sqrt(3.0) * R);
    const double al = 2.0 * ORC_PI * t / ORC_YEAR_S + opt->orbit_kappa;
    for (int n = 0; n < 3; ++n) {
        const double be = 2.0 * ORC_PI * n / 3.0 + opt->orbit_lambda;
        p[n][0] = R * cos(al) + 0.5 * e * R * (cos(2.0 * al - be) - 3.0 * cos(be))
                + 0.125 * e * e * R * (3.0 * cos(3.0 * al - 2.0 * be) - 10.0 * cos(al) - 5.0 * cos(al - 2.0 * be));
        p[n][1] = R * sin(al) + 0.5 * e * R * (sin(2.0 * al - be) - 3.0 * sin(be))
                + 0.125 * e * e * R * (3.0 * sin(3.0 * al - 2.0 * be) - 10.0 * sin(al) + 5.0 * sin(al - 2.0 * be));
        const double cd = cos(al - be), sd = sin(al - be);
        p[n][2] = -sqrt(3.0) * e * R * cd + sqrt(3.0) * e * e * R * (cd * cd + 2.0 * sd * sd);
    }
}

static double orc_sinc(double x) { return x == 0.0 ? 1.0 : sin(x) / x; }

/* Sky basis (reading A11): k = propagation direction. */
void oracle_sky_basis(double theta, double phi, double k[3], double u[3], double v[3])
{
    const double st = sin(theta), ct = cos(theta), sp = sin(phi), cp = cos(phi);
    k[0] = -st * cp; k[1] = -st * sp; k[2] = -ct;
    u[0] = ct * cp;  u[1] = ct * sp;  u[2] = -st;
    v[0] = sp;       v[1] = -cp;      v[2] = 0.0;
}

/* One-way link s -> r (photon leaves s, arrives at r), positions taken at time t:
 *   G_P = -i pi f L/c  sinc[pi f L/c (1 - k.n)]  exp[-i pi f (L/c + k.(p_r + p_s)/c)]  (n.e_P.n)
 * (Fourier transform of y = n.[h(t - L/c - k.p_s/c) - h(t - k.p_r/c)].n / (2 (1 - k.n)), Eq. 15 with
 * F(t) the antenna factor and d(t) = -k.p/c; convention h~(f) = int h exp(-2 pi i f t) dt, A5). */
static void orc_link(const double ps[3], const double pr[3], double f, double L,
                     const double k[3], const double u[3], const double v[3],
                     double Gp[2], double Gc[2])
{
    double n[3], kn = 0.0, un = 0.0, vn = 0.0, ksum = 0.0;
    for (int i = 0; i < 3; ++i) {
        n[i] = (pr[i] - ps[i]) / L;                      /* reading A10: nominal L */
        kn += k[i] * n[i]; un += u[i] * n[i]; vn += v[i] * n[i];
        ksum += k[i] * (pr[i] + ps[i]);
    }
    const double xi_p = un * un - vn * vn;               /* n.(uu - vv).n */
    const double xi_c = 2.0 * un * vn;                   /* n.(uv + vu).n */
    const double x = ORC_PI * f * L / ORC_C_SI;
    const double amp = x * orc_sinc(x * (1.0 - kn));
    const double ph = ORC_PI * f * (L / ORC_C_SI + ksum / ORC_C_SI);
    /* -i * amp * exp(-i ph) = amp * (-sin ph - i cos ph) */
    const double re = -amp * sin(ph), im = -amp * cos(ph);
    Gp[0] = re * xi_p; Gp[1] = im * xi_p;
    Gc[0] = re * xi_c; Gc[1] = im * xi_c;
}

/* First-generation Michelson combination centred on spacecraft v (v = 0, 1, 2 <-> X, Y, Z) with the constellation
 * at positions p (reading A7; Y and Z are X with the spacecraft relabelled cyclically):
 *   T_P = (1 - z^2) [ (G^{c->v} + z G^{v->c}) - (G^{b->v} + z G^{v->b}) ],  b = v + 1, c = v + 2 (mod 3),
 *   z = exp(-2 pi i f L/c);   for X: (G^{3->1} + z G^{1->3}) - (G^{2->1} + z G^{1->2}). */
static void orc_michelson(double p[3][3], int vtx, double f, double L, const double k[3], const double u[3],
                          const double v[3], double Tp[2], double Tc[2])
{
    const double *pv = p[vtx], *pb = p[(vtx + 1) % 3], *pc = p[(vtx + 2) % 3];
    double g31p[2], g31c[2], g13p[2], g13c[2], g21p[2], g21c[2], g12p[2], g12c[2];
    orc_link(pc, pv, f, L, k, u, v, g31p, g31c);
    orc_link(pv, pc, f, L, k, u, v, g13p, g13c);
    orc_link(pb, pv, f, L, k, u, v, g21p, g21c);
    orc_link(pv, pb, f, L, k, u, v, g12p, g12c);
    const double w = 2.0 * ORC_PI * f * L / ORC_C_SI;
    const double zr = cos(w), zi = -sin(w);
    const double z2r = zr * zr - zi * zi, z2i = 2.0 * zr * zi;
    const double fr = 1.0 - z2r, fi = -z2i;
    const double *gA[2] = { g31p, g31c }, *gB[2] = { g13p, g13c }, *gC[2] = { g21p, g21c }, *gD[2] = { g12p, g12c };
    double *out[2] = { Tp, Tc };
    for (int P = 0; P < 2; ++P) {
        const double sr = (gA[P][0] + zr * gB[P][0] - zi * gB[P][1]) - (gC[P][0] + zr * gD[P][0] - zi * gD[P][1]);
        const double si = (gA[P][1] + zr * gB[P][1] + zi * gB[P][0]) - (gC[P][1] + zr * gD[P][1] + zi * gD[P][0]);
        out[P][0] = fr * sr - fi * si;
        out[P][1] = fr * si + fi * sr;
    }
}

/* Transfer functions T_+(f), T_x(f) of the TDI combination opt->tdi_channel with the constellation at time t.
 * X, Y, Z: the Michelson combinations above.  A, E, T ("combinations called {A, E, T} that have
 * mutually independent noise of instrumental origin [64]"; the paper prints no formula, reading A28 takes those of
 * its ref. [64]):  A = (Z - X) / sqrt 2,  E = (X - 2 Y + Z) / sqrt 6,  T = (X + Y + Z) / sqrt 3. */
void oracle_response(const double *par, double f, double t, const oracle_options *opt,
                     double Tp[2], double Tc[2])
{
    double p[3][3], k[3], u[3], v[3];
    const double L = opt->arm_length_m;
    oracle_orbit(t, opt, p);
    oracle_sky_basis(par[3], par[4], k, u, v);
    const int ch = opt->tdi_channel;
    if (ch >= 0 && ch <= 2) {
        orc_michelson(p, ch, f, L, k, u, v, Tp, Tc);
        return;
    }
    double Xp[2], Xc[2], Yp[2], Yc[2], Zp[2], Zc[2];
    orc_michelson(p, 0, f, L, k, u, v, Xp, Xc);
    orc_michelson(p, 1, f, L, k, u, v, Yp, Yc);
    orc_michelson(p, 2, f, L, k, u, v, Zp, Zc);
    for (int i = 0; i < 2; ++i) {
        if (ch == 3)      { Tp[i] = (Zp[i] - Xp[i]) / sqrt(2.0);               Tc[i] = (Zc[i] - Xc[i]) / sqrt(2.0); }
        else if (ch == 4) { Tp[i] = (Xp[i] - 2.0 * Yp[i] + Zp[i]) / sqrt(6.0); Tc[i] = (Xc[i] - 2.0 * Yc[i] + Zc[i]) / sqrt(6.0); }
        else              { Tp[i] = (Xp[i] + Yp[i] + Zp[i]) / sqrt(3.0);       Tc[i] = (Xc[i] + Yc[i] + Zc[i]) / sqrt(3.0); }
    }
}

/* u_+(f_k), u_x(f_k), interleaved (re, im), for one particle (steps 1-4 of the header). */
void oracle_template(const double *par, int64_t n, const double *freq, const oracle_options *opt,
                     double *u_plus, double *u_cross)
{
    for (int64_t i = 0; i < n; ++i) {
        const double f = freq[i];
        double psi, tf, Tp[2], Tc[2];
        oracle_phase(par, f, opt, &psi, &tf);
        oracle_response(par, f, tf, opt, Tp, Tc);
        const double amp = pow(f, -7.0 / 6.0);
        const double cr = amp * cos(psi), ci = -amp * sin(psi);        /* f^(-7/6) exp(-i Psi_0) */
        u_plus[2 * i]      = Tp[0] * cr - Tp[1] * ci;
        u_plus[2 * i + 1]  = Tp[0] * ci + Tp[1] * cr;
        u_cross[2 * i]     = Tc[0] * cr - Tc[1] * ci;
        u_cross[2 * i + 1] = Tc[0] * ci + Tc[1] * cr;
    }
}

/* the paper's own outer segment limits ("the lowest and highest
 * instantaneous frequencies occurring during the observation period in the template"): the template is
 * in band at the bins whose stationary time t_f (Eq. 20 :220) falls inside the observation [0, T_obs].
 * Written out as the definition, bin by bin, with no assumption that t_f is monotone:
 *   k_lo = number of bins with t_f < 0,   k_hi = number of bins with t_f <= T_obs,
 * so that, t_f increasing along the grid (checked by *monotone), the in-band bins are [k_lo, k_hi). */
void oracle_template_band(const double *par, int64_t n, const double *freq, double T_obs,
                          const oracle_options *opt, int64_t *k_lo, int64_t *k_hi, int *monotone)
{
    int64_t lo = 0, hi = 0;
    int mono = 1;
    double prev = -INFINITY;
    for (int64_t i = 0; i < n; ++i) {
        double psi, tf;
        oracle_phase(par, freq[i], opt, &psi, &tf);
        if (tf < 0.0) ++lo;
        if (tf <= T_obs) ++hi;
        if (!(tf > prev)) mono = 0;
        prev = tf;
    }
    *k_lo = lo; *k_hi = hi;
    if (monotone) *monotone = mono;
}

/* N^i = <d, A^i>, M^ij = <A^i, A^j> over bins [lo, hi) by direct summation (Eq. 4, 8, 9, 12):
 *   <a, b> = 4 df Re sum a_k conj(b_k) / S_n(f_k), with dw = d / S_n and isn = 1 / S_n given.
 * A^1 = u_+, A^2 = u_x, A^3 = i u_+, A^4 = i u_x.  use_ld != 0 accumulates in long double
 * (hazard H3: near-singular M in narrow partitions); otherwise Neumaier-compensated double.  Either way N and M
 * come back as doubles; oracle_fstat_partition(mode 2) is the variant that never rounds them. */
void oracle_inner_products(const double *dw, const double *isn, const double *u_plus, const double *u_cross,
                           double df, int64_t lo, int64_t hi, int use_ld, double N[4], double M[16])
{
    long double sN[4] = {0, 0, 0, 0}, sM[4][4];
    double kN[4] = {0, 0, 0, 0}, cN[4] = {0, 0, 0, 0}, kM[4][4], cM[4][4];
    memset(sM, 0, sizeof sM); memset(kM, 0, sizeof kM); memset(cM, 0, sizeof cM);
    for (int64_t k = lo; k < hi; ++k) {
        double Ar[4], Ai[4];
        Ar[0] = u_plus[2 * k];       Ai[0] = u_plus[2 * k + 1];
        Ar[1] = u_cross[2 * k];      Ai[1] = u_cross[2 * k + 1];
        Ar[2] = -u_plus[2 * k + 1];  Ai[2] = u_plus[2 * k];          /* i u_+ */
        Ar[3] = -u_cross[2 * k + 1]; Ai[3] = u_cross[2 * k];         /* i u_x */
        const double dr = dw[2 * k], di = dw[2 * k + 1], w = isn[k];
        for (int i = 0; i < 4; ++i) {
            const double tN = dr * Ar[i] + di * Ai[i];               /* Re dw conj(A^i) */
            if (use_ld) sN[i] += (long double)dr * Ar[i] + (long double)di * Ai[i];
            else { double s = kN[i] + tN; cN[i] += (fabs(kN[i]) >= fabs(tN)) ? (kN[i] - s) + tN : (tN - s) + kN[i]; kN[i] = s; }
            for (int j = i; j < 4; ++j) {
                const double tM = (Ar[i] * Ar[j] + Ai[i] * Ai[j]) * w;   /* Re A^i conj(A^j) / S_n */
                if (use_ld) sM[i][j] += ((long double)Ar[i] * Ar[j] + (long double)Ai[i] * Ai[j]) * w;
                else { double s = kM[i][j] + tM; cM[i][j] += (fabs(kM[i][j]) >= fabs(tM)) ? (kM[i][j] - s) + tM : (tM - s) + kM[i][j]; kM[i][j] = s; }
            }
        }
    }
    for (int i = 0; i < 4; ++i) {
        N[i] = 4.0 * df * (use_ld ? (double)sN[i] : kN[i] + cN[i]);
        for (int j = i; j < 4; ++j) {
            const double m = 4.0 * df * (use_ld ? (double)sM[i][j] : kM[i][j] + cM[i][j]);
            M[4 * i + j] = m; M[4 * j + i] = m;
        }
    }
}

/* The same sums kept in long double (x86-64: 64-bit mantissa) all the way to the solve: "use_ld == 2" of the batch
 * calls.  Why (hazard H3, SURVEY section 7 H3(iii) "give the oracle a long double accumulation/epilogue switch to
 * establish truth"): over a narrow partition u_x is nearly a complex multiple of u_+ and the normalised determinant
 * 1 - |m_pc|^2 / (m_pp m_cc) of M falls to 3e-12 on config 4 (N_p = 1024 near 100 mHz, t_f moves 0.35 s per bin).
 * Rounding N and M to double (1e-16) before the solve then costs 1e-16 / det = 3e-5 of F_k -- more than the 1e-5
 * parity bar -- although every step before and after is exact enough.  Same definition (Eq. 4, 8, 9, 12), same
 * order of the sums, no rounding to double in between. */
static void orc_inner_products_ld(const double *dw, const double *isn, const double *u_plus, const double *u_cross,
                                  double df, int64_t lo, int64_t hi, long double N[4], long double M[16])
{
    long double sN[4] = {0, 0, 0, 0}, sM[4][4];
    memset(sM, 0, sizeof sM);
    for (int64_t k = lo; k < hi; ++k) {
        long double Ar[4], Ai[4];
        Ar[0] = u_plus[2 * k];       Ai[0] = u_plus[2 * k + 1];
        Ar[1] = u_cross[2 * k];      Ai[1] = u_cross[2 * k + 1];
        Ar[2] = -u_plus[2 * k + 1];  Ai[2] = u_plus[2 * k];          /* i u_+ */
        Ar[3] = -u_cross[2 * k + 1]; Ai[3] = u_cross[2 * k];         /* i u_x */
        const long double dr = dw[2 * k], di = dw[2 * k + 1], w = isn[k];
        for (int i = 0; i < 4; ++i) {
            sN[i] += dr * Ar[i] + di * Ai[i];                        /* Re dw conj(A^i) */
            for (int j = i; j < 4; ++j) sM[i][j] += (Ar[i] * Ar[j] + Ai[i] * Ai[j]) * w;
        }
    }
    for (int i = 0; i < 4; ++i) {
        N[i] = 4.0L * df * sN[i];
        for (int j = i; j < 4; ++j) { M[4 * i + j] = 4.0L * df * sM[i][j]; M[4 * j + i] = M[4 * i + j]; }
    }
}

/* Symmetric 4x4 eigen-decomposition by cyclic Jacobi (only used for a singular M). */
static void orc_jacobi4(double A[4][4], double Q[4][4], double lam[4])
{
    for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) Q[i][j] = (i == j);
    for (int sweep = 0; sweep < 64; ++sweep) {
        double off = 0.0;
        for (int i = 0; i < 4; ++i) for (int j = i + 1; j < 4; ++j) off += A[i][j] * A[i][j];
        if (off < 1e-60) break;
        for (int p = 0; p < 4; ++p) for (int q = p + 1; q < 4; ++q) {
            if (A[p][q] == 0.0) continue;
            const double th = 0.5 * atan2(2.0 * A[p][q], A[q][q] - A[p][p]);
            const double c = cos(th), s = sin(th);
            for (int k = 0; k < 4; ++k) { double a = A[k][p], b = A[k][q]; A[k][p] = c * a - s * b; A[k][q] = s * a + c * b; }
            for (int k = 0; k < 4; ++k) { double a = A[p][k], b = A[q][k]; A[p][k] = c * a - s * b; A[q][k] = s * a + c * b; }
            for (int k = 0; k < 4; ++k) { double a = Q[k][p], b = Q[k][q]; Q[k][p] = c * a - s * b; Q[k][q] = s * a + c * b; }
        }
    }
    for (int i = 0; i < 4; ++i) lam[i] = A[i][i];
}

/* F = max_a [a.N - a^T M a / 2] = N^T M^-1 N / 2 (Eq. 7): Cholesky solve of M a = N in long double.
 * If M is singular (a template vanishes or the four are linearly dependent on the partition, e.g. a
 * one-bin partition; reading A15) the maximum is N^T M^+ N / 2 with the pseudo-inverse, N being in the
 * range of the Gram matrix M.  Returns 0 (regular) or 1 (singular branch); a[] may be NULL.
 * The arithmetic is written once, for long double N and M; oracle_fstat_from_NM feeds it doubles. */
static int orc_fstat_from_NM_ld(const long double N[4], const long double M[16], double *F, double a_out[4])
{
    double s[4];
    int zero = 0;
    for (int i = 0; i < 4; ++i) { if (M[5 * i] > 0.0L) s[i] = 1.0 / sqrt((double)M[5 * i]); else { s[i] = 0.0; zero = 1; } }
    long double C[4][4], y[4], a[4];
    int singular = zero;
    if (!singular) {
        /* Cholesky of the unit-diagonal scaled matrix S M S */
        for (int i = 0; i < 4 && !singular; ++i) {
            for (int j = 0; j <= i; ++j) {
                long double acc = M[4 * i + j] * s[i] * s[j];
                for (int k = 0; k < j; ++k) acc -= C[i][k] * C[j][k];
                if (i == j) { if (acc <= 1e-13L) { singular = 1; break; } C[i][i] = sqrtl(acc); }
                else C[i][j] = acc / C[j][j];
            }
        }
    }
    if (!singular) {
        for (int i = 0; i < 4; ++i) { long double acc = N[i] * s[i]; for (int k = 0; k < i; ++k) acc -= C[i][k] * y[k]; y[i] = acc / C[i][i]; }
        for (int i = 3; i >= 0; --i) { long double acc = y[i]; for (int k = i + 1; k < 4; ++k) acc -= C[k][i] * a[k]; a[i] = acc / C[i][i]; }
        long double f = 0.0L;
        for (int i = 0; i < 4; ++i) f += N[i] * s[i] * a[i];
        *F = (double)(0.5L * f);
        if (a_out) for (int i = 0; i < 4; ++i) a_out[i] = (double)(a[i] * s[i]);
        return 0;
    }
    double A[4][4], Q[4][4], lam[4], lmax = 0.0, f = 0.0, coef[4] = {0, 0, 0, 0};
    for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) A[i][j] = (double)M[4 * i + j] * s[i] * s[j];
    orc_jacobi4(A, Q, lam);
    for (int i = 0; i < 4; ++i) if (lam[i] > lmax) lmax = lam[i];
    for (int i = 0; i < 4; ++i) {
        if (!(lam[i] > 1e-12 * lmax) || lmax <= 0.0) continue;
        double proj = 0.0;
        for (int k = 0; k < 4; ++k) proj += Q[k][i] * (double)N[k] * s[k];
        f += proj * proj / lam[i];
        for (int k = 0; k < 4; ++k) coef[k] += Q[k][i] * proj / lam[i];
    }
    *F = 0.5 * f;
    if (a_out) for (int i = 0; i < 4; ++i) a_out[i] = coef[i] * s[i];
    return 1;
}

int oracle_fstat_from_NM(const double N[4], const double M[16], double *F, double a_out[4])
{
    long double Nl[4], Ml[16];
    for (int i = 0; i < 4; ++i) Nl[i] = N[i];
    for (int i = 0; i < 16; ++i) Ml[i] = M[i];
    return orc_fstat_from_NM_ld(Nl, Ml, F, a_out);
}

/* Steps 5 of the header for one partition [lo, hi) of given templates.  mode 0: compensated double sums; 1: long
 * double sums rounded to double; 2: long double sums handed to the solve unrounded (see orc_inner_products_ld).
 * N_out[4], M_out[16] (may be NULL) receive the sums as doubles; a_out[4] (may be NULL) the amplitudes. */
int oracle_fstat_partition(const double *dw, const double *isn, const double *u_plus, const double *u_cross,
                           double df, int64_t lo, int64_t hi, int mode, double *F, double *N_out, double *M_out,
                           double *a_out)
{
    if (mode == 2) {
        long double Nl[4], Ml[16];
        orc_inner_products_ld(dw, isn, u_plus, u_cross, df, lo, hi, Nl, Ml);
        if (N_out) for (int i = 0; i < 4; ++i) N_out[i] = (double)Nl[i];
        if (M_out) for (int i = 0; i < 16; ++i) M_out[i] = (double)Ml[i];
        return orc_fstat_from_NM_ld(Nl, Ml, F, a_out);
    }
    double N[4], M[16];
    oracle_inner_products(dw, isn, u_plus, u_cross, df, lo, hi, mode, N, M);
    if (N_out) memcpy(N_out, N, sizeof N);
    if (M_out) memcpy(M_out, M, sizeof M);
    return oracle_fstat_from_NM(N, M, F, a_out);
}

/* Whole path for P particles: F[P], Fk[P][n_part] (may be NULL), optional N/M dump NM[P][n_part][20]
 * (N then row-major M; may be NULL), flags[P][n_part] = 1 where the singular branch ran (may be NULL).
 * Invalid particles get -inf (let-them-fly).  Returns 0, or -1 on allocation failure. */
int oracle_fstat_batch(int64_t n_bins, const double *freq, const double *dw, const double *isn,
                       int32_t n_part, const int64_t *edges, int64_t P, const double *params,
                       const oracle_options *opt, int use_ld, int n_threads,
                       double *F, double *Fk, double *NM, int32_t *flags)
{
    const double df = (n_bins > 1) ? (freq[n_bins - 1] - freq[0]) / (double)(n_bins - 1) : freq[0];
    int fail = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel
    {
        double *up = (double *)malloc(sizeof(double) * 2 * (size_t)(n_bins > 0 ? n_bins : 1));
        double *uc = (double *)malloc(sizeof(double) * 2 * (size_t)(n_bins > 0 ? n_bins : 1));
        if (!up || !uc) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int64_t p = 0; p < P; ++p) {
            if (!up || !uc) continue;
            const double *par = params + 6 * p;
            if (!oracle_params_valid(par)) {
                F[p] = -INFINITY;
                if (Fk) for (int j = 0; j < n_part; ++j) Fk[p * n_part + j] = -INFINITY;
                continue;
            }
            oracle_template(par, n_bins, freq, opt, up, uc);
            long double tot = 0.0L;
            for (int j = 0; j < n_part; ++j) {
                double N[4], M[16], Fj;
                const int sing = oracle_fstat_partition(dw, isn, up, uc, df, edges[j], edges[j + 1], use_ld, &Fj, N, M, NULL);
                if (Fk) Fk[p * n_part + j] = Fj;
                if (flags) flags[p * n_part + j] = sing;
                if (NM) { double *o = NM + ((size_t)p * n_part + j) * 20; memcpy(o, N, 4 * sizeof(double)); memcpy(o + 4, M, 16 * sizeof(double)); }
                tot += Fj;
            }
            F[p] = (double)tot;
        }
        free(up); free(uc);
    }
    return fail ? -1 : 0;
}

/* The same path for several partition sets over the same data (the hierarchy stages of PAPER.md:168-174 differ
 * only in N_seg): the templates of a particle are written out ONCE (steps 1-4) and step 5 is repeated per set.
 * Nothing else differs from oracle_fstat_batch -- same functions, same order of the sums -- so its results are
 * bit-equal to one oracle_fstat_batch call per set (tests/test_oracle_pins.py checks that).
 *   n_part[s], s < n_sets; edges = the sets' edge arrays one after the other (n_part[s] + 1 entries each);
 *   F[s * P + p];  Fk = the sets' [P][n_part[s]] blocks one after the other. */
int oracle_fstat_batch_multi(int64_t n_bins, const double *freq, const double *dw, const double *isn,
                             int32_t n_sets, const int32_t *n_part, const int64_t *edges, int64_t P,
                             const double *params, const oracle_options *opt, int use_ld, int n_threads,
                             double *F, double *Fk)
{
    const double df = (n_bins > 1) ? (freq[n_bins - 1] - freq[0]) / (double)(n_bins - 1) : freq[0];
    int fail = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel
    {
        double *up = (double *)malloc(sizeof(double) * 2 * (size_t)(n_bins > 0 ? n_bins : 1));
        double *uc = (double *)malloc(sizeof(double) * 2 * (size_t)(n_bins > 0 ? n_bins : 1));
        if (!up || !uc) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int64_t p = 0; p < P; ++p) {
            if (!up || !uc) continue;
            const double *par = params + 6 * p;
            const int ok = oracle_params_valid(par);
            if (ok) oracle_template(par, n_bins, freq, opt, up, uc);
            const int64_t *e = edges;
            double *fk = Fk;
            for (int32_t s = 0; s < n_sets; ++s) {
                long double tot = 0.0L;
                for (int j = 0; j < n_part[s]; ++j) {
                    double N[4], M[16], Fj = -INFINITY;
                    if (ok) {
                        oracle_fstat_partition(dw, isn, up, uc, df, e[j], e[j + 1], use_ld, &Fj, N, M, NULL);
                        tot += Fj;
                    }
                    fk[p * n_part[s] + j] = Fj;
                }
                F[(int64_t)s * P + p] = ok ? (double)tot : -INFINITY;
                e += n_part[s] + 1;
                fk += P * (int64_t)n_part[s];
            }
        }
        free(up); free(uc);
    }
    return fail ? -1 : 0;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
