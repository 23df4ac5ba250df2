// fstat_device.cuh -- device-side helpers of the sm_100a F-statistic kernels: FP64 sincos of an angle
// given in quarter turns, a fast FP64 reciprocal, and the mbarrier / TMA bulk-copy PTX wrappers.
// Part of the product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fstat {

// ------------------------------------------------------------------------------------------------
// sincos of (pi/2) * t for |t| < 2^50, FP64.  t = n + w with n = rint(t), |w| <= 1/2; the angle
// (pi/2) w lies in [-pi/4, pi/4], where the Taylor polynomials below (sin through w^15, cos through
// w^14) are accurate to 5e-17 / 1e-15 absolute.  No slow path, no table, no divergence: the
// arguments on the hot path (carrier phase, orbital phase, arm phases) are bounded by construction.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sincos_qt(double t, double &s, double &c)
{
    const double MAGIC = 6755399441055744.0;            // 1.5 * 2^52: adding it rounds to nearest int
    const double tm = t + MAGIC;
    const int q = __double2loint(tm);                    // low word holds n (two's complement)
    const double n = tm - MAGIC;
    const double w = t - n;
    const double w2 = w * w;
    double ps = -6.688035109811467232478226e-10;
    ps = fma(ps, w2, 5.692172921967926811775255e-8);
    ps = fma(ps, w2, -3.59884323521208534045854e-6);
    ps = fma(ps, w2, 1.604411847873598218726609e-4);
    ps = fma(ps, w2, -4.681754135318688100685464e-3);
    ps = fma(ps, w2, 7.969262624616704512050555e-2);
    ps = fma(ps, w2, -0.6459640975062462536557566);
    ps = fma(ps, w2, 1.570796326794896619231322);
    ps *= w;
    double pc = -6.386603083791852241089888e-9;
    pc = fma(pc, w2, 4.710874778818171503670277e-7);
    pc = fma(pc, w2, -2.520204237306060548105302e-5);
    pc = fma(pc, w2, 9.192602748394265802417162e-4);
    pc = fma(pc, w2, -2.086348076335296087305164e-2);
    pc = fma(pc, w2, 0.2536695079010480136365634);
    pc = fma(pc, w2, -1.233700550136169827354311);
    pc = fma(pc, w2, 1.0);
    // quadrant: q&3 = 0: (s,c) = (ps,pc); 1: (pc,-ps); 2: (-ps,-pc); 3: (-pc,ps)
    const bool swap = (q & 1) != 0;
    double ss = swap ? pc : ps;
    double cc = swap ? ps : pc;
    const int sflip = (q & 2) << 30;                     // bit 31 of the high word
    const int cflip = ((q + 1) & 2) << 30;
    s = __hiloint2double(__double2hiint(ss) ^ sflip, __double2loint(ss));
    c = __hiloint2double(__double2hiint(cc) ^ cflip, __double2loint(cc));
}

// sincos of (pi/2) t for |t| < 1/64 (the second and third phase differences of the interpolating kernel;
// the stride selection sends work items with larger differences to the direct kernel): Taylor series
// through x^9 / x^8, error < 1e-18.
__device__ __forceinline__ void sincos_qt_small(double t, double &s, double &c)
{
    const double x = 1.570796326794896619231322 * t, x2 = x * x;
    s = x * fma(x2, fma(x2, fma(x2, fma(x2, 1.0 / 362880.0, -1.0 / 5040.0), 1.0 / 120.0), -1.0 / 6.0), 1.0);
    c = fma(x2, fma(x2, fma(x2, fma(x2, 1.0 / 40320.0, -1.0 / 720.0), 1.0 / 24.0), -0.5), 1.0);
}

// 1/x for a normal x of either sign: hardware seed (MUFU.RCP64H, about 2^-20) and one cubic Newton step
// r <- r + r (e + e^2), e = 1 - x r, which leaves a relative error near 2^-60.
__device__ __forceinline__ double rcp_fast(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);
    const double e2 = fma(e, e, e);
    r = fma(r, e2, r);
    const double e3 = fma(-x, r, 1.0);                   // one linear clean-up step: ~2^-100 -> rounding
    return fma(r, e3, r);
}

// ------------------------------------------------------------------------------------------------
// mbarrier + TMA 1-D bulk copy (cp.async.bulk, SASS UBLKCP) wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// global -> shared bulk copy of `bytes` (multiple of 16, both addresses 16-byte aligned), completion
// signalled on `bar` as transaction bytes.
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

}  // namespace fstat
