// fstat_fast.cuh -- device pieces shared by the two interpolating kernels (fstat_fast_kernel in fstat_fast.cu:
// CTA-uniform partition edges; fstat_fastband_kernel in fstat_fastband.cu: per-thread partition edges, row f2) and by
// the plan-time Gram builders: the Lagrange basis of a node interval, the Chebyshev-economised cubic, the exact
// reduction of the linear phase term, the Newton-basis coefficients of the running sums.  Product path only.
#pragma once
#include "fstat_device.cuh"
#include "fstat_internal.h"

namespace fstat {

// Lagrange basis of the nodes t = -1, 0, 1, 2 at t
__device__ __forceinline__ void lagrange4(double t, double (&l)[4])
{
    const double tp = t + 1.0, tm = t - 1.0, tm2 = t - 2.0;
    l[0] = -t * tm * tm2 * (1.0 / 6.0);
    l[1] = tp * tm * tm2 * 0.5;
    l[2] = -tp * t * tm2 * 0.5;
    l[3] = tp * t * tm * (1.0 / 6.0);
}

// The cubic carried over a node interval [node m, node m+1] is NOT the Lagrange cubic through four nodes but
// the Chebyshev-economised quintic through the six nodes m-2 .. m+3: the quintic's T_4 and T_5 terms on the
// interval are dropped, which leaves the 4th-order error term 72 times smaller than the centre-interval error
// of the four-node cubic (h^4 f/3072 against 3 h^4 f/128) for the same node evaluations.  Row a of
// kEcon gives the value of that cubic at t = -1, 0, 1, 2 (so that everything downstream -- Newton
// coefficients, Gram matrices in the four-node Lagrange basis -- is unchanged) from the node values at
// t = -2 .. 3; rows sum to 1 exactly (rationals with denominator 61440).
__constant__ double kEcon[4][6] = {
    {-9133.0 / 61440.0, 6371.0 / 4096.0, -4517.0 / 6144.0, 2209.0 / 6144.0, 33.0 / 4096.0, -2407.0 / 61440.0},
    {-11.0 / 61440.0, 7.0 / 12288.0, 2047.0 / 2048.0, -1.0 / 6144.0, 5.0 / 12288.0, -3.0 / 20480.0},
    {-3.0 / 20480.0, 5.0 / 12288.0, -1.0 / 6144.0, 2047.0 / 2048.0, 7.0 / 12288.0, -11.0 / 61440.0},
    {-2407.0 / 61440.0, 33.0 / 4096.0, 2209.0 / 6144.0, -4517.0 / 6144.0, 6371.0 / 4096.0, -9133.0 / 61440.0}};

// v[k] = node values at t = -2 .. 3.  Returns yref = v[2] (node "0") and e[a] = cubic(t_a) - yref, t_a = -1, 0,
// 1, 2, from the DIFFERENCES v[k] - yref (the phase values are ~1e7 quarter turns, their differences ~1e3).
__device__ __forceinline__ void economise(const double (&v)[6], double &yref, double (&e)[4])
{
    yref = v[2];
    const double d0 = v[0] - yref, d1 = v[1] - yref, d3 = v[3] - yref, d4 = v[4] - yref, d5 = v[5] - yref;
#pragma unroll
    for (int a = 0; a < 4; ++a)
        e[a] = fma(kEcon[a][0], d0, fma(kEcon[a][1], d1, fma(kEcon[a][3], d3, fma(kEcon[a][4], d4, kEcon[a][5] * d5))));
}

// The same economised cubic as monomial coefficients in t: y(t) = y(0) + a_1 t + a_2 t^2 + a_3 t^3 on [0, 1], rows y(0),
// a_1, a_2, a_3 from the node values at t = -2 .. 3 (kEcon followed by the 4-point fit; exact rationals; row 0 sums to 1,
// the others to 0).  The sub-block sums of the slow factors T' use it (sub-block_moments), the carrier phase keeps
// economise(): its values are ~1e7 quarter turns and need the differences.
__constant__ double kEconMono[4][6] = {
    {-11.0 / 61440.0, 7.0 / 12288.0, 2047.0 / 2048.0, -1.0 / 6144.0, 5.0 / 12288.0, -3.0 / 20480.0},
    {1721.0 / 30720.0, -3193.0 / 6144.0, -967.0 / 3072.0, 3079.0 / 3072.0, -1607.0 / 6144.0, 1159.0 / 30720.0},
    {-19.0 / 256.0, 199.0 / 256.0, -175.0 / 128.0, 87.0 / 128.0, 1.0 / 256.0, -5.0 / 256.0},
    {7.0 / 384.0, -33.0 / 128.0, 131.0 / 192.0, -131.0 / 192.0, 33.0 / 128.0, -7.0 / 384.0}};

// Plan time: the Gram matrix G (upper triangle g, Lagrange basis of the nodes t = -1, 0, 1, 2) of a sub-block as the
// factor W = L^T E, G = L L^T (Cholesky; G is a sum of w l l^T, positive semi-definite), E = kEcon as a map from the SIX
// node values at t = -2 .. 3 to the four cubic values: for node values v, y = E v and y^T G y' = (W v) . (W v').  A
// sub-block of fewer than four bins has a rank-deficient G: a pivot that vanishes takes its column with it.
__device__ __forceinline__ void gram_to_w(const double (&g)[kNGram], double (&W)[kNW])
{
    double G[4][4];
    {
        int j = 0;
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a; b < 4; ++b) { G[a][b] = g[j]; G[b][a] = g[j]; ++j; }
    }
    double L[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) L[i][j] = 0.0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        double d = G[j][j];
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (k < j) d = fma(-L[j][k], L[j][k], d);
        if (d > 1e-28 * G[j][j] && d > 0.0) {
            const double r = sqrt(d), ir = 1.0 / r;
            L[j][j] = r;
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (i > j) {
                    double x = G[i][j];
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if (k < j) x = fma(-L[i][k], L[j][k], x);
                    L[i][j] = x * ir;
                }
        }
    }
    // E with the column of node "0" taken from the row sums, as economise() applies it (values relative to that node)
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            double x = 0.0;
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (i >= j) {
                    double e = kEcon[i][k];
                    if (k == 2) e = 1.0 - (kEcon[i][0] + kEcon[i][1] + kEcon[i][3] + kEcon[i][4] + kEcon[i][5]);
                    x = fma(L[i][j], e, x);
                }
            W[j * 6 + k] = x;
        }
}

// m_PQ of a sub-block from the node values of T'_+ and of the recentred T'_x (t = -2 .. 3) and the sub-block's W:
// w^X = W v^X (4 x 6), m_pp = |w^+|^2, m_cc = |w^c|^2, m_pc = w^+ . conj(w^c).  128 FP64 instructions.
__device__ __forceinline__ void gram_forms(const double *__restrict__ Wg, const double (&vpr)[6], const double (&vpi)[6],
                                           const double (&vcr)[6], const double (&vci)[6], double &mpp, double &mcc,
                                           double &mre, double &mim)
{
    const double2 *wp = reinterpret_cast<const double2 *>(Wg);
    mpp = 0.0; mcc = 0.0; mre = 0.0; mim = 0.0;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const double2 w01 = wp[3 * r], w23 = wp[3 * r + 1], w45 = wp[3 * r + 2];
        const double w[6] = {w01.x, w01.y, w23.x, w23.y, w45.x, w45.y};
        double ar = w[0] * vpr[0], ai = w[0] * vpi[0], br = w[0] * vcr[0], bi = w[0] * vci[0];
#pragma unroll
        for (int k = 1; k < 6; ++k) {
            ar = fma(w[k], vpr[k], ar);
            ai = fma(w[k], vpi[k], ai);
            br = fma(w[k], vcr[k], br);
            bi = fma(w[k], vci[k], bi);
        }
        mpp = fma(ar, ar, fma(ai, ai, mpp));
        mcc = fma(br, br, fma(bi, bi, mcc));
        mre = fma(ar, br, fma(ai, bi, mre));
        mim = fma(ai, br, fma(-ar, bi, mim));
    }
}

// The sums of a sub-block that ends U bins after node 0, sum_i conj(T'(i)) q_i for a slow factor T' given by its six node
// values v_k, are sum_k conj(v_k) B_k with weights B_k that do not depend on the factor: with the economised cubic
// T'(t) = y0 + a_1 t + a_2 t^2 + a_3 t^3 (rows of kEconMono) and the running sums A_n (binomial weights C(u + n - 1, n)
// counted back from the end of the sub-block), the monomial moments Q_j = sum_i t_i^j q_i are
//   Q_1 = u A_0 - r A_1,   Q_2 = u^2 A_0 - (2 u r + r^2) A_1 + 2 r^2 A_2,
//   Q_3 = u^3 A_0 - (3 u^2 r + 3 u r^2 + r^3) A_1 + (6 u r^2 + 6 r^3) A_2 - 6 r^3 A_3,     r = 1 / S, u = U / S
// (the Newton-basis conversion of newton_coefs, transposed onto the sums), and B_k = E_0k A_0 + sum_j E_jk Q_j.
// A = (A_0 re, im, A_1 re, im, A_2 re, im, A_3 re, im).  78 FP64 instructions, once per sub-block.
__device__ __forceinline__ void subblock_weights(const double (&A)[8], double rS, double U, double (&Br)[6], double (&Bi)[6])
{
    const double u = U * rS, r2 = rS * rS, r3 = r2 * rS, u2 = u * u;
    const double p21 = rS * fma(2.0, u, rS);
    const double p31 = rS * fma(3.0 * u, u + rS, r2);
    const double p32 = 6.0 * r2 * (u + rS);
    const double q1r = fma(u, A[0], -rS * A[2]), q1i = fma(u, A[1], -rS * A[3]);
    const double q2r = fma(u2, A[0], fma(-p21, A[2], 2.0 * r2 * A[4])), q2i = fma(u2, A[1], fma(-p21, A[3], 2.0 * r2 * A[5]));
    const double u3 = u2 * u, s3 = -6.0 * r3;
    const double q3r = fma(u3, A[0], fma(-p31, A[2], fma(p32, A[4], s3 * A[6])));
    const double q3i = fma(u3, A[1], fma(-p31, A[3], fma(p32, A[5], s3 * A[7])));
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        Br[k] = fma(kEconMono[0][k], A[0], fma(kEconMono[1][k], q1r, fma(kEconMono[2][k], q2r, kEconMono[3][k] * q3r)));
        Bi[k] = fma(kEconMono[0][k], A[1], fma(kEconMono[1][k], q1i, fma(kEconMono[2][k], q2i, kEconMono[3][k] * q3i)));
    }
}

// z += sum_k conj(v_k) B_k
__device__ __forceinline__ void z_from_nodes(const double (&vr)[6], const double (&vi)[6], const double (&Br)[6],
                                             const double (&Bi)[6], double &zr, double &zi)
{
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        sr = fma(vr[k], Br[k], fma(vi[k], Bi[k], sr));
        si = fma(vr[k], Bi[k], fma(-vi[k], Br[k], si));
    }
    zr += sr;
    zi += si;
}

// x - 4 rint(x / 4): exact for |x| < 2^51
__device__ __forceinline__ double red4(double x) { return fma(-4.0, rint(0.25 * x), x); }

// (c * f) mod 4 to full precision: the product is split exactly into hi + lo by one FMA
__device__ __forceinline__ double mulmod4(double c, double f)
{
    const double hi = c * f;
    const double lo = fma(c, f, -hi);
    return red4(hi) + lo;
}

// Newton-basis coefficients c_n (basis C(u + n - 1, n), u = j1 - i) of the cubic through the node values
// y0..y3 at t = -1, 0, 1, 2 (t = s / S), for a sub-block that ends U bins after node 0.
__device__ __forceinline__ void newton_coefs(double y0, double y1, double y2, double y3, double rS, double U,
                                             double (&c)[4])
{
    const double d0 = y0 - y1, d2 = y2 - y1, d3 = y3 - y1;
    const double a1 = fma(d0, -1.0 / 3.0, fma(d3, -1.0 / 6.0, d2));
    const double a2 = 0.5 * (d0 + d2);
    const double a3 = fma(d2, -0.5, (d3 - d0) * (1.0 / 6.0));
    const double g1 = a1 * rS, g2 = a2 * rS * rS, g3 = a3 * rS * rS * rS;
    const double e0 = fma(U, fma(U, fma(U, g3, g2), g1), y1);
    const double e1 = -fma(U, fma(3.0 * U, g3, 2.0 * g2), g1);
    const double e2 = fma(3.0 * U, g3, g2);
    const double e3 = -g3;
    c[0] = e0;
    c[1] = e1 - e2 + e3;
    c[2] = fma(-6.0, e3, 2.0 * e2);
    c[3] = 6.0 * e3;
}

__device__ __forceinline__ void load_coef(const double *__restrict__ cf, int64_t P_pad, double (&c)[kNCoef])
{
#pragma unroll
    for (int j = 0; j < kNCoef; ++j) c[j] = cf[(int64_t)j * P_pad];
}

}  // namespace fstat
