// fstat_pso.cu -- SURVEY row f1: particle swarm optimisation on the device (Sec. III.A;
// Eq. 13-14 :146-150), driving fstat_eval_batch without a host synchronisation per iteration.
//
// Several independent swarms (PSO runs, :160) are batched: particle gid = swarm * n_particles + i.  Positions
// live in the unit box [0,1]^6 and map to (t_c, M_c, eta, theta, phi, e0) = lo + x (hi - lo).  Per iteration,
// all on the caller's stream:  pso_step_kernel (Eq. 13-14, lbest ring topology, |v| <= v_max, linearly decaying
// inertia, "let them fly": a particle outside the box gets NaN parameters, which fstat_eval_batch turns into
// F = -inf, :158)  ->  fstat_eval_batch  ->  pso_update_best_kernel.  Random numbers come from Philox4x32-10
// (counter = (gid, iteration, draw, 0), key = seed), the same counter-based generator the CPU test oracle
// implements on its own; every floating-point operation is written with explicit round-to-nearest intrinsics in the
// oracle's order, so positions and velocities agree bit for bit given the same fitness values.
#include "../../include/fstat.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <new>
#include <string>
#include <vector>

namespace {

constexpr int kDim = 6;

__host__ __device__ inline void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4])
{
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// 12 uniforms in (0, 1): (x + 0.5) 2^-32, exact in FP64
__device__ inline void draw12(uint32_t gid, uint32_t it, uint64_t seed, double (&u)[12])
{
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        uint32_t o[4];
        philox4x32_10(gid, it, (uint32_t)j, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), o);
#pragma unroll
        for (int q = 0; q < 4; ++q) u[4 * j + q] = __dmul_rn(__dadd_rn((double)o[q], 0.5), 2.3283064365386963e-10);
    }
}

__device__ inline double clampv(double v, double vmax) { return fmin(fmax(v, -vmax), vmax); }

__device__ inline void write_params(const double *x, const double *lo, const double *hi, double *par)
{
    bool inside = true;
#pragma unroll
    for (int d = 0; d < kDim; ++d) inside = inside && (x[d] >= 0.0) && (x[d] <= 1.0);
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int d = 0; d < kDim; ++d)
        par[d] = inside ? __dadd_rn(lo[d], __dmul_rn(x[d], __dsub_rn(hi[d], lo[d]))) : nan;
}

// boxes: [n_swarms][2][kDim] (lo, then hi) on the device: every swarm searches its own box (the hierarchy's stages run
// one swarm set per t_c interval / candidate)

__global__ void pso_init_kernel(int32_t n, int32_t n_particles, uint64_t seed, double vmax,
                                const double *__restrict__ boxes, double *__restrict__ x,
                                double *__restrict__ v, double *__restrict__ params)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n) return;
    double u[12], xx[kDim];
    draw12((uint32_t)g, 0u, seed, u);
#pragma unroll
    for (int d = 0; d < kDim; ++d) {
        xx[d] = u[d];                                            // x ~ U[a, b]          (:158)
        x[g * kDim + d] = xx[d];
        v[g * kDim + d] = clampv(__dsub_rn(u[6 + d], xx[d]), vmax);   // v ~ U[a - x, b - x]  (:158)
    }
    const double *bx = boxes + (g / n_particles) * 2 * kDim;
    write_params(xx, bx, bx + kDim, params + (int64_t)g * kDim);
}

// first evaluation: the personal best is the initial position
__global__ void pso_first_best_kernel(int32_t n, const double *__restrict__ x, const double *__restrict__ F,
                                      double *__restrict__ pbest, double *__restrict__ pbest_f)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n) return;
#pragma unroll
    for (int d = 0; d < kDim; ++d) pbest[g * kDim + d] = x[g * kDim + d];
    pbest_f[g] = F[g];
}

__global__ void pso_step_kernel(int32_t n, int32_t n_particles, uint32_t it, uint64_t seed, double w, double c1,
                                double c2, double vmax, const double *__restrict__ boxes, double *__restrict__ x,
                                double *__restrict__ v,
                                const double *__restrict__ pbest, const double *__restrict__ pbest_f,
                                double *__restrict__ params)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n) return;
    const int64_t sw = g / n_particles;
    const int i = (int)(g - sw * n_particles);
    // lbest: best personal best among the ring neighbours i-1, i, i+1 (first maximum in that order)
    const int64_t left = sw * n_particles + (i + n_particles - 1) % n_particles;
    const int64_t right = sw * n_particles + (i + 1) % n_particles;
    int64_t lb = left;
    double fb = pbest_f[left];
    if (pbest_f[g] > fb) { fb = pbest_f[g]; lb = g; }
    if (pbest_f[right] > fb) { fb = pbest_f[right]; lb = right; }
    double u[12], xx[kDim];
    draw12((uint32_t)g, it, seed, u);
#pragma unroll
    for (int d = 0; d < kDim; ++d) {
        const double xd = x[g * kDim + d], vd = v[g * kDim + d];
        const double t1 = __dmul_rn(__dmul_rn(c1, u[d]), __dsub_rn(pbest[g * kDim + d], xd));
        const double t2 = __dmul_rn(__dmul_rn(c2, u[6 + d]), __dsub_rn(pbest[lb * kDim + d], xd));
        const double vn = clampv(__dadd_rn(__dadd_rn(__dmul_rn(w, vd), t1), t2), vmax);   // Eq. 14 :150
        xx[d] = __dadd_rn(xd, vn);                                                       // Eq. 13 :146
        v[g * kDim + d] = vn;
    }
    // positions are written after every thread of the grid has read its neighbours' pbest (they are not
    // touched here) -- x itself is private to the thread
#pragma unroll
    for (int d = 0; d < kDim; ++d) x[g * kDim + d] = xx[d];
    const double *bx = boxes + sw * 2 * kDim;
    write_params(xx, bx, bx + kDim, params + (int64_t)g * kDim);
}

__global__ void pso_update_best_kernel(int32_t n, const double *__restrict__ x, const double *__restrict__ F,
                                       double *__restrict__ pbest, double *__restrict__ pbest_f)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n) return;
    if (F[g] > pbest_f[g]) {
        pbest_f[g] = F[g];
#pragma unroll
        for (int d = 0; d < kDim; ++d) pbest[g * kDim + d] = x[g * kDim + d];
    }
}

// one block per swarm: arg max of pbest_f (lowest index on ties), mapped to physical parameters
__global__ void __launch_bounds__(128) pso_swarm_best_kernel(int32_t n_particles, const double *__restrict__ boxes,
                                                             const double *__restrict__ pbest,
                                                             const double *__restrict__ pbest_f,
                                                             double *__restrict__ best_params,
                                                             double *__restrict__ best_f)
{
    __shared__ double sf[128];
    __shared__ int si[128];
    const int sw = blockIdx.x, tid = threadIdx.x;
    double f = -INFINITY;
    int idx = 0x7fffffff;
    for (int i = tid; i < n_particles; i += 128) {
        const double fi = pbest_f[(int64_t)sw * n_particles + i];
        if (fi > f || (fi == f && i < idx)) { f = fi; idx = i; }
    }
    sf[tid] = f; si[tid] = idx;
    __syncthreads();
    for (int s = 64; s > 0; s >>= 1) {
        if (tid < s) {
            if (sf[tid + s] > sf[tid] || (sf[tid + s] == sf[tid] && si[tid + s] < si[tid])) {
                sf[tid] = sf[tid + s]; si[tid] = si[tid + s];
            }
        }
        __syncthreads();
    }
    if (tid == 0) {
        const int i = (si[0] == 0x7fffffff) ? 0 : si[0];
        const double *pb = pbest + ((int64_t)sw * n_particles + i) * kDim;
        best_f[sw] = sf[0];
        const double *lo = boxes + (int64_t)sw * 2 * kDim, *hi = lo + kDim;
        for (int d = 0; d < kDim; ++d)
            best_params[(int64_t)sw * kDim + d] = __dadd_rn(lo[d], __dmul_rn(pb[d], __dsub_rn(hi[d], lo[d])));
    }
}

}  // namespace

struct fstat_pso;
static fstat_status pso_fitness(fstat_pso *ps, cudaStream_t st);

struct fstat_pso {
    fstat_plan *plan = nullptr;
    int32_t n_swarms = 0, n_particles = 0, n_iter_total = 0, n = 0;
    uint32_t it_done = 0;
    uint64_t seed = 0;
    fstat_pso_options opt{};
    double *d_boxes = nullptr;            // [n_swarms][2][kDim]
    double *d_x = nullptr, *d_v = nullptr, *d_pbest = nullptr, *d_pbest_f = nullptr, *d_params = nullptr, *d_F = nullptr;
    double *d_best_params = nullptr, *d_best_f = nullptr;
    std::string err;
};

#define PSO_TRY(ps, call)                                                                           \
    do {                                                                                            \
        cudaError_t e__ = (call);                                                                   \
        if (e__ != cudaSuccess) {                                                                   \
            cudaGetLastError();                                                                     \
            (ps)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                        \
            return e__ == cudaErrorMemoryAllocation ? FSTAT_ENOMEM : FSTAT_ECUDA;                   \
        }                                                                                           \
    } while (0)

// the fitness of all particles of all swarms: the plan's fixed partitions, or (rows f1 x f2) per-template bands
static fstat_status pso_fitness(fstat_pso *ps, cudaStream_t st)
{
    if (ps->opt.band_n_seg >= 1)
        return fstat_eval_batch_bands(ps->plan, ps->n, ps->d_params, ps->opt.band_n_seg, ps->opt.band_lattice, ps->d_F,
                                      nullptr, nullptr, (void *)st);
    return fstat_eval_batch(ps->plan, ps->n, ps->d_params, ps->d_F, nullptr, (void *)st);
}

extern "C" {

void fstat_pso_default_options(fstat_pso_options *o)
{
    if (!o) return;
    o->c1 = 2.0; o->c2 = 2.0; o->v_max = 0.5; o->w_start = 0.9; o->w_end = 0.4;
    o->band_n_seg = 0; o->band_lattice = 1;
}

void fstat_pso_destroy(fstat_pso *ps)
{
    if (!ps) return;
    int dev = fstat_plan_device(ps->plan), prev = -1;
    cudaGetDevice(&prev);
    if (dev >= 0) cudaSetDevice(dev);
    cudaFree(ps->d_x); cudaFree(ps->d_v); cudaFree(ps->d_pbest); cudaFree(ps->d_pbest_f); cudaFree(ps->d_params);
    cudaFree(ps->d_F); cudaFree(ps->d_best_params); cudaFree(ps->d_best_f); cudaFree(ps->d_boxes);
    if (prev >= 0) cudaSetDevice(prev);
    delete ps;
}

static fstat_status pso_create_impl(fstat_pso *ps, cudaStream_t st)
{
    const size_t n = (size_t)ps->n;
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_x, n * kDim * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_v, n * kDim * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_pbest, n * kDim * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_pbest_f, n * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_params, n * kDim * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_F, n * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_best_params, (size_t)ps->n_swarms * kDim * sizeof(double)));
    PSO_TRY(ps, cudaMalloc((void **)&ps->d_best_f, (size_t)ps->n_swarms * sizeof(double)));
    const int nt = 128, nb = (ps->n + nt - 1) / nt;
    pso_init_kernel<<<nb, nt, 0, st>>>(ps->n, ps->n_particles, ps->seed, ps->opt.v_max, ps->d_boxes, ps->d_x, ps->d_v,
                                       ps->d_params);
    PSO_TRY(ps, cudaGetLastError());
    fstat_status s = pso_fitness(ps, st);
    if (s != FSTAT_OK) { ps->err = fstat_last_error(ps->plan); return s; }
    pso_first_best_kernel<<<nb, nt, 0, st>>>(ps->n, ps->d_x, ps->d_F, ps->d_pbest, ps->d_pbest_f);
    PSO_TRY(ps, cudaGetLastError());
    return FSTAT_OK;
}

// boxes_h: HOST [n_box][2][kDim]-like input given as lo [n_box][kDim], hi [n_box][kDim]; n_box = 1 (one box for every
// swarm) or n_swarms
static fstat_status pso_create_common(fstat_pso **out, fstat_plan *plan, int32_t n_swarms, int32_t n_particles,
                                      int32_t n_iter_total, const double *lo, const double *hi, int32_t n_box,
                                      uint64_t seed, const fstat_pso_options *opts, void *stream)
{
    if (!out) return FSTAT_EINVAL;
    *out = nullptr;
    if (!plan || !lo || !hi || n_swarms < 1 || n_particles < 1 || n_iter_total < 0 ||
        (int64_t)n_swarms * n_particles > ((int64_t)1 << 30))
        return FSTAT_EINVAL;
    fstat_pso_options o;
    fstat_pso_default_options(&o);
    if (opts) o = *opts;
    if (!(o.v_max > 0.0) || !isfinite(o.c1) || !isfinite(o.c2) || !isfinite(o.w_start) || !isfinite(o.w_end) ||
        o.band_n_seg < 0 || (o.band_n_seg >= 1 && o.band_lattice < 1))
        return FSTAT_EINVAL;
    for (int64_t d = 0; d < (int64_t)n_box * kDim; ++d)
        if (!isfinite(lo[d]) || !isfinite(hi[d]) || !(hi[d] >= lo[d])) return FSTAT_EINVAL;
    fstat_pso *ps = new (std::nothrow) fstat_pso;
    if (!ps) return FSTAT_ENOMEM;
    ps->plan = plan; ps->n_swarms = n_swarms; ps->n_particles = n_particles; ps->n_iter_total = n_iter_total;
    ps->n = n_swarms * n_particles; ps->seed = seed; ps->opt = o;
    std::vector<double> boxes((size_t)n_swarms * 2 * kDim);
    for (int32_t sw = 0; sw < n_swarms; ++sw) {
        const int64_t b = n_box == 1 ? 0 : sw;
        for (int d = 0; d < kDim; ++d) {
            boxes[((size_t)sw * 2 + 0) * kDim + d] = lo[b * kDim + d];
            boxes[((size_t)sw * 2 + 1) * kDim + d] = hi[b * kDim + d];
        }
    }
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(fstat_plan_device(plan));
    fstat_status s = FSTAT_OK;
    if (cudaMalloc((void **)&ps->d_boxes, boxes.size() * sizeof(double)) != cudaSuccess ||
        cudaMemcpy(ps->d_boxes, boxes.data(), boxes.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        s = FSTAT_ECUDA;
    }
    if (s == FSTAT_OK) s = pso_create_impl(ps, (cudaStream_t)stream);
    if (prev >= 0) cudaSetDevice(prev);
    if (s != FSTAT_OK) { fstat_pso_destroy(ps); return s; }
    *out = ps;
    return FSTAT_OK;
}

fstat_status fstat_pso_create(fstat_pso **out, fstat_plan *plan, int32_t n_swarms, int32_t n_particles,
                              int32_t n_iter_total, const double *lo, const double *hi, uint64_t seed,
                              const fstat_pso_options *opts, void *stream)
{
    return pso_create_common(out, plan, n_swarms, n_particles, n_iter_total, lo, hi, 1, seed, opts, stream);
}

fstat_status fstat_pso_create_boxes(fstat_pso **out, fstat_plan *plan, int32_t n_swarms, int32_t n_particles,
                                    int32_t n_iter_total, const double *lo, const double *hi, uint64_t seed,
                                    const fstat_pso_options *opts, void *stream)
{
    return pso_create_common(out, plan, n_swarms, n_particles, n_iter_total, lo, hi, n_swarms, seed, opts, stream);
}

fstat_status fstat_pso_iterate(fstat_pso *ps, int32_t n_iter, void *stream)
{
    if (!ps || n_iter < 0) return FSTAT_EINVAL;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(fstat_plan_device(ps->plan));
    cudaStream_t st = (cudaStream_t)stream;
    const int nt = 128, nb = (ps->n + nt - 1) / nt;
    fstat_status rc = FSTAT_OK;
    for (int32_t k = 0; k < n_iter && rc == FSTAT_OK; ++k) {
        const uint32_t it = ps->it_done + 1;                       // 1-based step number
        const int32_t den = ps->n_iter_total > 1 ? ps->n_iter_total - 1 : 1;
        const double frac = (double)(it - 1) / (double)den;
        const double w = ps->opt.w_start + (ps->opt.w_end - ps->opt.w_start) * (frac < 1.0 ? frac : 1.0);
        pso_step_kernel<<<nb, nt, 0, st>>>(ps->n, ps->n_particles, it, ps->seed, w, ps->opt.c1, ps->opt.c2,
                                           ps->opt.v_max, ps->d_boxes, ps->d_x, ps->d_v, ps->d_pbest, ps->d_pbest_f,
                                           ps->d_params);
        if (cudaGetLastError() != cudaSuccess) { ps->err = "pso_step_kernel launch failed"; rc = FSTAT_ECUDA; break; }
        rc = pso_fitness(ps, st);
        if (rc != FSTAT_OK) { ps->err = fstat_last_error(ps->plan); break; }
        pso_update_best_kernel<<<nb, nt, 0, st>>>(ps->n, ps->d_x, ps->d_F, ps->d_pbest, ps->d_pbest_f);
        if (cudaGetLastError() != cudaSuccess) { ps->err = "pso_update_best_kernel launch failed"; rc = FSTAT_ECUDA; break; }
        ps->it_done = it;
    }
    if (prev >= 0) cudaSetDevice(prev);
    return rc;
}

fstat_status fstat_pso_best(fstat_pso *ps, double *best_params_host, double *best_f_host, void *stream)
{
    if (!ps || !best_params_host || !best_f_host) return FSTAT_EINVAL;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(fstat_plan_device(ps->plan));
    cudaStream_t st = (cudaStream_t)stream;
    fstat_status rc = FSTAT_OK;
    pso_swarm_best_kernel<<<ps->n_swarms, 128, 0, st>>>(ps->n_particles, ps->d_boxes, ps->d_pbest, ps->d_pbest_f,
                                                        ps->d_best_params, ps->d_best_f);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(best_params_host, ps->d_best_params, (size_t)ps->n_swarms * kDim * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(best_f_host, ps->d_best_f, (size_t)ps->n_swarms * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaGetLastError(); ps->err = cudaGetErrorString(e); rc = FSTAT_ECUDA; }
    if (prev >= 0) cudaSetDevice(prev);
    return rc;
}

fstat_status fstat_pso_state(fstat_pso *ps, double *x, double *v, double *pbest, double *pbest_f, double *f_last,
                             void *stream)
{
    if (!ps) return FSTAT_EINVAL;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(fstat_plan_device(ps->plan));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)ps->n;
    cudaError_t e = cudaSuccess;
    if (x && e == cudaSuccess) e = cudaMemcpyAsync(x, ps->d_x, n * kDim * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (v && e == cudaSuccess) e = cudaMemcpyAsync(v, ps->d_v, n * kDim * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (pbest && e == cudaSuccess) e = cudaMemcpyAsync(pbest, ps->d_pbest, n * kDim * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (pbest_f && e == cudaSuccess) e = cudaMemcpyAsync(pbest_f, ps->d_pbest_f, n * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (f_last && e == cudaSuccess) e = cudaMemcpyAsync(f_last, ps->d_F, n * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (prev >= 0) cudaSetDevice(prev);
    if (e != cudaSuccess) { cudaGetLastError(); ps->err = cudaGetErrorString(e); return FSTAT_ECUDA; }
    return FSTAT_OK;
}

int32_t fstat_pso_iterations_done(const fstat_pso *ps) { return ps ? (int32_t)ps->it_done : 0; }

}  // extern "C"
