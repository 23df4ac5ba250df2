// fstat_model.cuh -- the per-(particle, frequency) model evaluated in full FP64: SPA phase without its
// linear term, orbital phase at t_f, LISA orbit, TDI-X response (steps a2-a3 of DESIGN.md).  Used by
// the direct kernel at every bin and by the interpolating kernel at its nodes.  Product path only.
#pragma once
#include "fstat_device.cuh"
#include "fstat_internal.h"

namespace fstat {

// one orbit coordinate from the trig basis (1, c1, s1, c2, s2, c3, s3)
__device__ __forceinline__ double orb7(const double *C, double c1, double s1, double c2, double s2, double c3, double s3)
{
    double r = fma(C[1], c1, C[0]);
    r = fma(C[2], s1, r);
    r = fma(C[3], c2, r);
    r = fma(C[4], s2, r);
    r = fma(C[5], c3, r);
    return fma(C[6], s3, r);
}
__device__ __forceinline__ double orb5(const double *C, double c1, double s1, double c2, double s2)
{
    double r = fma(C[1], c1, C[0]);
    r = fma(C[2], s1, r);
    r = fma(C[3], c2, r);
    return fma(C[4], s2, r);
}

// 1 + k.n and 1 - k.n are divided by; an exact zero (the only value too small: they are sums with 1) is
// replaced by 2^-60, for which sin(x P) / P = x to rounding.  They may be slightly NEGATIVE: the arm vector
// n = (p_j - p_1)/L uses the nominal L (reading A10), so |k.n| reaches 1.0024 for a source along a breathing
// arm; sin(x P) / P is even in P, nothing special happens there.
__device__ __forceinline__ double arm_nonzero(double P) { return P == 0.0 ? 0x1p-60 : P; }

// One arm 1 -> j of TDI-X at one frequency.  mu = k.n, with n = (p_j - p_1)/L; Pm = 1 + mu, Qm = 1 - mu
// (both non-zero), rho = 1 / (Pm Qm).
//   g = exp(-i a) [ sinc(a) + z sinc(b) ] x,   a = x (1 + mu), b = x (1 - mu), z = exp(-2 i x)
// (sum of the two one-way links of the arm, PAPER.md:196 Eq. 15, :206 Eq. 17 with N = 0; the common
// factor -i and the Doppler phase of spacecraft 1 are applied outside).  Of the two angles a + b = 2x the
// SMALLER one gets the direct sincos (its sine is divided by the small 1 +- mu and must be relatively
// accurate); the other follows from the angle-difference formulas.  Branch-free.
__device__ __forceinline__ void arm_response(double xq, double c2x, double s2x, double Pm, double Qm,
                                             double rho, double &gr, double &gi)
{
    const bool a_direct = fabs(Pm) <= fabs(Qm);
    double sd, cd;
    sincos_qt(xq * (a_direct ? Pm : Qm), sd, cd);
    const double so = fma(s2x, cd, -c2x * sd);           // sin(2x - d)
    const double co = fma(c2x, cd, s2x * sd);            // cos(2x - d)
    const double sa = a_direct ? sd : so, ca = a_direct ? cd : co, sb = a_direct ? so : sd;
    const double sca = sa * Qm * rho;                    // x sinc(a) = sin(a) / (1 + mu)
    const double scb = sb * Pm * rho;                    // x sinc(b) = sin(b) / (1 - mu)
    const double br = fma(c2x, scb, sca);
    const double bi = -s2x * scb;
    gr = fma(ca, br, sa * bi);
    gi = fma(ca, bi, -sa * br);
}

// The same arm seen from BOTH of its ends (rows f4: Y, Z, A, E, T need the Michelson combinations centred on all three
// spacecraft): gf = g(mu) as above (vertex at the tail of n), gb = g(-mu) = exp(-i b) [ sinc(b) + z sinc(a) ] x (vertex
// at the head), and dop = exp(-i (a - b)) = exp(-2 i x mu), the Doppler phase of the head relative to the tail.
__device__ __forceinline__ void arm_response_both(double xq, double c2x, double s2x, double Pm, double Qm, double rho,
                                                  double &gfr, double &gfi, double &gbr, double &gbi, double &dr,
                                                  double &di)
{
    const bool a_direct = fabs(Pm) <= fabs(Qm);
    double sd, cd;
    sincos_qt(xq * (a_direct ? Pm : Qm), sd, cd);
    const double so = fma(s2x, cd, -c2x * sd);           // sin(2x - d)
    const double co = fma(c2x, cd, s2x * sd);            // cos(2x - d)
    const double sa = a_direct ? sd : so, ca = a_direct ? cd : co, sb = a_direct ? so : sd, cb = a_direct ? co : cd;
    const double sca = sa * Qm * rho;                    // x sinc(a) = sin(a) / (1 + mu)
    const double scb = sb * Pm * rho;                    // x sinc(b) = sin(b) / (1 - mu)
    const double br = fma(c2x, scb, sca), bi = -s2x * scb;
    gfr = fma(ca, br, sa * bi);
    gfi = fma(ca, bi, -sa * br);
    const double cr = fma(c2x, sca, scb), ci = -s2x * sca;
    gbr = fma(cb, cr, sb * ci);
    gbi = fma(cb, ci, -sb * cr);
    dr = fma(ca, cb, sa * sb);
    di = fma(ca, sb, -sa * cb);
}

// a2 and the geometry half of a3 at one frequency: SPA phase (quarter turns) without its linear term, plus the Doppler
// phase of spacecraft 1 (reading A4); k.n, u.n, v.n of the arms 1->2 and 1->3 at t_f.  `row` is a table row (layout
// TabCol), c[] the particle's coefficients.
struct NodeGeom {
    double psi_nl, xq, c2x, s2x;
    double mu2, mu3, un2, un3, vn2, vn3;
};
__device__ __forceinline__ void node_geometry(const double2 *__restrict__ row, const double (&c)[kNCoef],
                                              const OrbitCoef &orb, NodeGeom &g)
{
    const double kx = c[11], ky = c[12], kz = c[13];
    const double ux = c[14], uy = c[15], uz = c[16];
    const double vx = c[17], vy = c[18], vz = c[19];
    const double2 r0 = row[0], r1 = row[1], r2 = row[2], r3 = row[3], r4 = row[4];
    const double2 d0 = row[5], d1 = row[6], d2 = row[7], d3 = row[8];
    const double2 zz = row[9];
    const double f = r0.x;

    // ---- a2: SPA phase (quarter turns) and orbital phase at t_f  (Eq. A3 :404, Eq. 20 :220)
    double psi = fma(c[2], r0.y, c[1]);
    psi = fma(c[3], r1.x, psi);
    psi = fma(c[4], r1.y, psi);
    psi = fma(c[5], r2.x, psi);
    psi = fma(c[6], r2.y, psi);
    psi = fma(c[7], r3.x, psi);
    psi = fma(c[8], r3.y, psi);
    psi = fma(c[9], r4.x, psi);
    g.xq = r4.y;
    g.c2x = zz.x;
    g.s2x = zz.y;
    double alq = fma(c[2], d0.x, c[10]);
    alq = fma(c[3], d0.y, alq);
    alq = fma(c[4], d1.x, alq);
    alq = fma(c[5], d1.y, alq);
    alq = fma(c[6], d2.x, alq);
    alq = fma(c[7], d2.y, alq);
    alq = fma(c[8], d3.x, alq);
    alq = fma(c[9], d3.y, alq);

    // ---- a3: orbit to O(e^2) at t_f (reading A9), arm geometry
    double s1, c1;
    sincos_qt(alq, s1, c1);
    const double c2 = fma(c1, c1, -s1 * s1), s2 = 2.0 * s1 * c1;
    const double c3 = fma(c1, c2, -s1 * s2), s3 = fma(s1, c2, c1 * s2);
    const double p1x = orb7(orb.c[0][0], c1, s1, c2, s2, c3, s3);
    const double p1y = orb7(orb.c[0][1], c1, s1, c2, s2, c3, s3);
    const double p1z = orb5(orb.c[0][2], c1, s1, c2, s2);
    const double n2x = orb7(orb.c[1][0], c1, s1, c2, s2, c3, s3);
    const double n2y = orb7(orb.c[1][1], c1, s1, c2, s2, c3, s3);
    const double n2z = orb5(orb.c[1][2], c1, s1, c2, s2);
    const double n3x = orb7(orb.c[2][0], c1, s1, c2, s2, c3, s3);
    const double n3y = orb7(orb.c[2][1], c1, s1, c2, s2, c3, s3);
    const double n3z = orb5(orb.c[2][2], c1, s1, c2, s2);
    const double kp = fma(kx, p1x, fma(ky, p1y, kz * p1z));        // 4 k.p_1/c
    g.mu2 = fma(kx, n2x, fma(ky, n2y, kz * n2z));
    g.mu3 = fma(kx, n3x, fma(ky, n3y, kz * n3z));
    g.un2 = fma(ux, n2x, fma(uy, n2y, uz * n2z));
    g.un3 = fma(ux, n3x, fma(uy, n3y, uz * n3z));
    g.vn2 = fma(vx, n2x, fma(vy, n2y, vz * n2z));
    g.vn3 = fma(vx, n3x, fma(vy, n3y, vz * n3z));
    g.psi_nl = fma(f, kp, psi);                                     // + Doppler phase of spacecraft 1
}

// The three first-generation Michelson responses X', Y', Z' of one node, both polarisations, all relative to the
// Doppler phase of spacecraft 1: three arms 1->2, 1->3, 2->3 (n_23 = n_13 - n_12), each evaluated once and seen from
// both ends.  xyz[pol][0..5] = (X re, X im, Y re, Y im, Z re, Z im), pol 0 = +, 1 = x.
//   X = xi_13 g(mu_13) - xi_12 g(mu_12);  Y = [xi_12 g(-mu_12) - xi_23 g(mu_23)] exp(-2 i x mu_12);
//   Z = [xi_23 g(-mu_23) - xi_13 g(-mu_13)] exp(-2 i x mu_13)          (cyclic relabelling of reading A7)
__device__ __forceinline__ void michelson_xyz(const NodeGeom &g, double (&xyz)[2][6])
{
    const double mu23 = g.mu3 - g.mu2, un23 = g.un3 - g.un2, vn23 = g.vn3 - g.vn2;
    const double P2 = arm_nonzero(1.0 + g.mu2), Q2 = arm_nonzero(1.0 - g.mu2);
    const double P3 = arm_nonzero(1.0 + g.mu3), Q3 = arm_nonzero(1.0 - g.mu3);
    const double P4 = arm_nonzero(1.0 + mu23), Q4 = arm_nonzero(1.0 - mu23);
    const double den2 = P2 * Q2, den3 = P3 * Q3, den4 = P4 * Q4;
    const double R = rcp_fast(den2 * den3 * den4);
    double f2r, f2i, b2r, b2i, d2r, d2i, f3r, f3i, b3r, b3i, d3r, d3i, f4r, f4i, b4r, b4i, d4r, d4i;
    arm_response_both(g.xq, g.c2x, g.s2x, P2, Q2, den3 * den4 * R, f2r, f2i, b2r, b2i, d2r, d2i);
    arm_response_both(g.xq, g.c2x, g.s2x, P3, Q3, den2 * den4 * R, f3r, f3i, b3r, b3i, d3r, d3i);
    arm_response_both(g.xq, g.c2x, g.s2x, P4, Q4, den2 * den3 * R, f4r, f4i, b4r, b4i, d4r, d4i);
    const double xp2 = fma(g.un2, g.un2, -g.vn2 * g.vn2), xc2 = 2.0 * g.un2 * g.vn2;
    const double xp3 = fma(g.un3, g.un3, -g.vn3 * g.vn3), xc3 = 2.0 * g.un3 * g.vn3;
    const double xp4 = fma(un23, un23, -vn23 * vn23), xc4 = 2.0 * un23 * vn23;
#pragma unroll
    for (int pol = 0; pol < 2; ++pol) {
        const double x2 = pol ? xc2 : xp2, x3 = pol ? xc3 : xp3, x4 = pol ? xc4 : xp4;
        xyz[pol][0] = fma(x3, f3r, -x2 * f2r);
        xyz[pol][1] = fma(x3, f3i, -x2 * f2i);
        const double yr = fma(x2, b2r, -x4 * f4r), yi = fma(x2, b2i, -x4 * f4i);
        const double zr = fma(x4, b4r, -x3 * b3r), zi = fma(x4, b4i, -x3 * b3i);
        xyz[pol][2] = fma(yr, d2r, -yi * d2i);
        xyz[pol][3] = fma(yr, d2i, yi * d2r);
        xyz[pol][4] = fma(zr, d3r, -zi * d3i);
        xyz[pol][5] = fma(zr, d3i, zi * d3r);
    }
}

// a2 + a3 at one frequency.  Returns, in quarter turns, psi_nl (the carrier phase without its linear term c[0] f) and
// T'_+, T'_x with T_P = K_f T'_P, K_f = -i (1 - z^2) folded into the data tables.
// AET = false: first-generation Michelson X (Y, Z through the orbit coefficients of the relabelled constellation).
// AET = true (reading A28): T' = w_X X' + w_Y Y' + w_Z Z' with the weights orb.wch of A = (Z - X)/sqrt 2,
// E = (X - 2Y + Z)/sqrt 6 or T = (X + Y + Z)/sqrt 3; the three Michelson responses share the phase, t_f, the orbit and
// the three arms.
template <bool AET = false>
__device__ __forceinline__ void model_eval(const double2 *__restrict__ row, const double (&c)[kNCoef],
                                           const OrbitCoef &orb, double &psi_nl, double &tpr, double &tpi,
                                           double &tcr, double &tci)
{
    NodeGeom g;
    node_geometry(row, c, orb, g);
    psi_nl = g.psi_nl;
    if (!AET) {
        // two arms
        const double P2 = arm_nonzero(1.0 + g.mu2), Q2 = arm_nonzero(1.0 - g.mu2);
        const double P3 = arm_nonzero(1.0 + g.mu3), Q3 = arm_nonzero(1.0 - g.mu3);
        const double den2 = P2 * Q2, den3 = P3 * Q3;         // either sign (|mu| may exceed 1 by 0.0024), never 0
        const double R = rcp_fast(den2 * den3);
        double g2r, g2i, g3r, g3i;
        arm_response(g.xq, g.c2x, g.s2x, P2, Q2, den3 * R, g2r, g2i);
        arm_response(g.xq, g.c2x, g.s2x, P3, Q3, den2 * R, g3r, g3i);
        const double xp2 = fma(g.un2, g.un2, -g.vn2 * g.vn2), xc2 = 2.0 * g.un2 * g.vn2;   // n.e_+.n, n.e_x.n
        const double xp3 = fma(g.un3, g.un3, -g.vn3 * g.vn3), xc3 = 2.0 * g.un3 * g.vn3;
        // T'_P = xi_P3 g_3 - xi_P2 g_2   (TDI-X: arm 3 minus arm 2, reading A7)
        tpr = fma(xp3, g3r, -xp2 * g2r);
        tpi = fma(xp3, g3i, -xp2 * g2i);
        tcr = fma(xc3, g3r, -xc2 * g2r);
        tci = fma(xc3, g3i, -xc2 * g2i);
    } else {
        double xyz[2][6];
        michelson_xyz(g, xyz);
        const double wx = orb.wch[0], wy = orb.wch[1], wz = orb.wch[2];
        tpr = fma(wx, xyz[0][0], fma(wy, xyz[0][2], wz * xyz[0][4]));
        tpi = fma(wx, xyz[0][1], fma(wy, xyz[0][3], wz * xyz[0][5]));
        tcr = fma(wx, xyz[1][0], fma(wy, xyz[1][2], wz * xyz[1][4]));
        tci = fma(wx, xyz[1][1], fma(wy, xyz[1][3], wz * xyz[1][5]));
    }
}

// The particle-independent columns of a table row at frequency f (phase basis B_j, derivative basis D_j,
// arm phases); the data columns T_DWR, T_DWI, T_W are left to the caller.
__device__ __forceinline__ void fill_basis_row(double f, double L, double *row)
{
    const double lnf = log(f);
    const double cb = cbrt(f);                 // f^(1/3)
    const double icb = 1.0 / cb;               // f^(-1/3)
    const double fm23 = icb * icb;
    const double fm1 = 1.0 / f;
    const double fm53 = fm1 * fm23;
    const double fm349 = pow(f, -34.0 / 9.0);
    const double iyr = 1.0 / kYear;
    row[T_F] = f;
    row[T_LNF] = lnf;
    row[T_FM53] = fm53;
    row[T_FM1] = fm1;
    row[T_FM23] = fm23;
    row[T_FM13] = icb;
    row[T_FP13] = cb;
    row[T_FP13LN] = cb * lnf;
    row[T_FM349] = fm349;
    row[T_XQ] = 2.0 * f * L / kC;
    // D_j = (dB_j/df) / year, same order as B_2..B_9
    row[T_D0 + 0] = fm1 * iyr;                                   // ln f
    row[T_D0 + 1] = (-5.0 / 3.0) * fm53 * fm1 * iyr;              // f^(-5/3)
    row[T_D0 + 2] = -fm1 * fm1 * iyr;                             // f^(-1)
    row[T_D0 + 3] = (-2.0 / 3.0) * fm53 * iyr;                    // f^(-2/3)
    row[T_D0 + 4] = (-1.0 / 3.0) * icb * fm1 * iyr;               // f^(-1/3)
    row[T_D0 + 5] = (1.0 / 3.0) * fm23 * iyr;                     // f^(1/3)
    row[T_D0 + 6] = fm23 * (1.0 + lnf / 3.0) * iyr;               // f^(1/3) ln f
    row[T_D0 + 7] = (-34.0 / 9.0) * fm349 * fm1 * iyr;            // f^(-34/9)
    const double x = kPi * f * L / kC;
    double s2x, c2x;
    sincos(2.0 * x, &s2x, &c2x);
    row[T_C2X] = c2x;
    row[T_S2X] = s2x;
    row[T_X] = x;
}

}  // namespace fstat
