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
