/*
 * fstat.h -- C ABI of the B200-native batched semi-coherent F-statistic (arXiv 2407.10797).
 *
 * The library evaluates, for P PSO particles at once, the paper's fitness function
 *
 *     F(Theta_I) = sum_{k=1..N_p} F_k ,      F_k = 1/2 N_k^T M_k^-1 N_k            (Eq. 7,
 *                                                                                   :110 Eq. 11, :117 Eq. 12)
 *
 * where N_k^i = <d, A^i>_k and M_k^ij = <A^i, A^j>_k are the noise-weighted inner products
 * (PAPER.md:66 Eq. 4, :89-91 Eq. 8-9) restricted to frequency partition k, and A^1..A^4 are the four
 * basis templates of the linear decomposition h = sum a_i A^i (Eq. 5) built from the
 * restricted-PN stationary-phase waveform h~(f) = A f^(-7/6) exp(-i Psi(f)) (PAPER.md:397-405
 * Eq. A1-A3) times the leading-order frequency-domain LISA TDI-X response T(f) evaluated at
 * t_f = (1/2pi) dPsi/df (Eq. 17-20 with N = 0; orbit :198).  N_p = 1 is the fully
 * coherent statistic.  F is the SUM of the F_k, not the mean of Eq. 11 (DESIGN.md
 * reading A12).  Every step runs in hand-written sm_100a CUDA kernels; no template is written to
 * memory; there is no CPU fallback (calls fail with FSTAT_ECUDA when no usable device exists).
 *
 * Conventions common to all calls
 *   - All floating-point data are IEEE double.  "host" / "device" is stated per pointer.
 *   - Every call returns an fstat_status and never throws or aborts.
 *   - A plan may be used by one host thread at a time, from ONE stream at a time, and has one evaluation in flight
 *     at a time: its workspace (coefficients, partial sums, work lists, the timing ring) lives inside the plan and is
 *     not guarded, so two evaluations of one plan on different streams would race.  Distinct plans are independent.
 *   - Evaluation calls only enqueue work on the caller's stream.  Host-side work happens when something changes: the
 *     first evaluation with a new batch size builds (and caches, per work-segment length) the segment tables and may
 *     grow the workspace (cudaMalloc / cudaFree, which can synchronise the device); the first
 *     fstat_eval_batch_bands call builds its prefix tables.  Repeated calls with batch sizes seen before do neither.
 */
#ifndef FSTAT_H_
#define FSTAT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define FSTAT_API
#else
#define FSTAT_API __attribute__((visibility("default")))
#endif

typedef struct fstat_plan fstat_plan;    /* opaque; created and destroyed by the library */

typedef enum {
    FSTAT_OK = 0,
    FSTAT_EINVAL = 1,        /* an argument violates the contract below (see fstat_last_error)  */
    FSTAT_ENOMEM = 2,        /* host or device allocation failed                                 */
    FSTAT_ECUDA = 3,         /* a CUDA runtime call or kernel launch failed / no device          */
    FSTAT_EUNSUPPORTED = 4   /* valid request outside this build's limits (e.g. n_bins >= 2^31)  */
} fstat_status;

/* TDI combinations the library can template: the first-generation Michelson combinations X, Y, Z
 * (centred on spacecraft 1, 2, 3; reading A7) and A = (Z - X)/sqrt 2, E = (X - 2Y + Z)/sqrt 6,
 * T = (X + Y + Z)/sqrt 3, "that have mutually independent noise of instrumental origin [64]" (reading A28). */
typedef enum {
    FSTAT_TDI_X = 0, FSTAT_TDI_Y = 1, FSTAT_TDI_Z = 2, FSTAT_TDI_A = 3, FSTAT_TDI_E = 4, FSTAT_TDI_T = 5
} fstat_tdi_channel;

/* Options of a plan.  Obtain defaults with fstat_default_options; opts == NULL means defaults. */
typedef struct {
    double f_ref_e0;          /* frequency [Hz] at which e0 is defined; default 0.01      */
    double arm_length_m;      /* LISA arm length L [m]; default 2.5e9                                   */
    double orbit_kappa;       /* initial orbital phase of the constellation centre [rad]; default 0     */
    double orbit_lambda;      /* initial orientation of the constellation [rad]; default 0              */
    int32_t device;           /* CUDA device ordinal; -1 (default) = the calling thread's current one   */
    int32_t inputs_on_device; /* 0 (default): freq/dw/inv_sn are host pointers; 1: device pointers      */
    int32_t max_segment_bins; /* 0 (default) = automatic.  Upper bound on the number of bins one CTA    *
                               * sums before handing its partial sums to the epilogue (tuning / tests)  */
    int32_t force_level;      /* -2 (default): the stride of the interpolating kernel is chosen per (particle      *
                               * group, segment) from an a-priori error bound; -1: direct kernel everywhere       *
                               * (every bin evaluated in full, no interpolation); 0..6: stride 8 << level          *
                               * wherever the segment allows it, regardless of the bound (tests / tuning)          */
    double interp_tol;        /* scale of the interpolation error tolerances; 1.0 (default) = carrier phase        *
                               * 1.5e-7 rad and TDI response 2e-7 relative            */
    int32_t tdi_channel;      /* fstat_tdi_channel: the TDI combination this plan's data and templates are in;     *
                               * default FSTAT_TDI_X, the paper's                                     */
    int32_t no_channel_fusion;/* 0 (default): fstat_eval_batch_channels evaluates two or three plans of the A / E / T  *
                               * family in ONE pass of the interpolating kernel (shared node model and carrier);   *
                               * 1 (read from plans[0]): one pass per channel, as for any other set (tests / tuning)*/
    int32_t min_stride_level; /* smallest stride level 0..6 (stride 8 << level) the plan keeps tables for; -1 (set by      *
                               * fstat_default_options) = automatic: 2 (stride 32), or force_level when that is 0 or 1.  *
                               * Work items whose error bound asks for a smaller stride go to the direct kernel.  The    *
                               * tables of levels 0 and 1 are 3/4 of the per-sub-block tables (36 of 48 bytes per bin);   *
                               * no work item of the paper's band (>= 10 mHz, 2.5 yr) asks for them                       */
} fstat_options;

FSTAT_API void fstat_default_options(fstat_options *opts);

/*
 * fstat_plan_create -- copy one TDI channel's frequency-domain data into the device and fold every
 * particle-independent factor of the template and of the inner product (PAPER.md:66 Eq. 4; :397
 * Eq. A1; :404 Eq. A3) into per-bin tables.
 *
 *   out         [out] receives the plan; set to NULL on failure.
 *   n_bins      number of frequency bins N, 1 <= N < 2^31.
 *   freq_hz     [N] strictly positive, strictly ascending, uniform grid f_k = k/T (df = 1/T is taken
 *               as (f[N-1]-f[0])/(N-1), or f[0] when N == 1).  Non-uniformity > 1e-6 df is EINVAL.
 *   dw_re_im    [N][2] interleaved re, im of  d~(f_k) / S_n(f_k)   (data weighted by the one-sided PSD).
 *   inv_sn      [N] 1 / S_n(f_k), finite and > 0.
 *   n_part      number of partitions N_p >= 1 (N_p = 1: fully coherent).
 *   part_edges  [N_p+1] HOST pointer, bin offsets 0 = e_0 < e_1 < ... < e_{N_p} = N; partition k is the
 *               half-open bin range [e_k, e_{k+1})  (Eq. 12; fixed data-side edges,
 *               DESIGN.md reading A13).
 *   opts        may be NULL.
 *
 * freq_hz, dw_re_im, inv_sn are host or device pointers according to opts->inputs_on_device.  The plan
 * copies everything it needs: the caller may free or overwrite its arrays once the call returns.
 * Errors: EINVAL for NULL pointers, a non-positive / non-ascending / non-uniform grid, non-finite dw or
 * inv_sn, inv_sn <= 0, bad edges, an empty partition; ENOMEM; ECUDA; EUNSUPPORTED.
 */
FSTAT_API fstat_status fstat_plan_create(fstat_plan **out,
                                         int64_t n_bins, const double *freq_hz,
                                         const double *dw_re_im, const double *inv_sn,
                                         int32_t n_part, const int64_t *part_edges,
                                         const fstat_options *opts);

/*
 * fstat_plan_set_partitions -- replace the partition edges of an existing plan (same data, another
 * N_p: the hierarchy stages of PAPER.md:168-174 differ only in N_seg).  Same rules for part_edges
 * (HOST pointer) as in fstat_plan_create.  On error the plan keeps its previous partitions.
 */
FSTAT_API fstat_status fstat_plan_set_partitions(fstat_plan *plan, int32_t n_part,
                                                 const int64_t *part_edges);

/*
 * fstat_eval_batch -- evaluate F and the per-partition F_k for P particles ("the
 * computation of the semi-coherent F-statistic for each particle can be carried out in parallel").
 *
 *   params  [P][6] DEVICE pointer, row-major: t_c [s from the first sample], M_c [solar masses], eta,
 *           theta [rad, ecliptic colatitude], phi [rad, ecliptic longitude], e0 (eta in
 *           place of delta_mu, eta = (1 - delta_mu^2)/4, reading A18).
 *   F       [P] DEVICE pointer, out.
 *   Fk      [P][N_p] DEVICE pointer, row-major, out; may be NULL.
 *   cuda_stream  a cudaStream_t (NULL = the legacy default stream).  The call only enqueues work on
 *           that stream and returns; results are valid once the stream has reached that point.
 *
 * A particle with a non-finite parameter, M_c <= 0, eta outside (0, 0.25] or e0 < 0 is not an error:
 * it gets F = -inf and F_k = -inf (PSO's "let them fly" fitness).  P == 0 is a no-op.
 * Errors: EINVAL (NULL plan/params/F with P > 0, P < 0), ENOMEM (workspace growth), ECUDA.
 */
FSTAT_API fstat_status fstat_eval_batch(fstat_plan *plan, int64_t P,
                                        const double *params, double *F, double *Fk,
                                        void *cuda_stream);

/*
 * fstat_eval_batch_noalloc -- fstat_eval_batch for callers that cannot allocate device memory inside the call (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): same arguments, same kernels, same results
 * bit for bit, but the workspace (coefficients, slot ranking, stride levels, work list, partial sums) is carved from ONE
 * static device array of fstat_noalloc_scratch_bytes() = 32 MiB that every GPU which loads the library holds until the
 * process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *   Limit: the workspace of the batch must fit: about n_work_segments x 10 KiB + 24 KiB per 128 particles (one swarm of
 *   128 particles on a 2.5-yr grid with N_p = 1024: 18 MB; 1024 particles with N_p = 64 on the same grid: 29 MB), and
 *   P <= 16384.  Beyond that: EUNSUPPORTED, with the sizes in fstat_last_error.
 *   Set-up: the plan's segment tables for this batch size are plan state (device memory the plan owns): they exist once
 *   fstat_eval_batch has been called with a batch of this size (number of 128-particle groups) since the last
 *   fstat_plan_create / fstat_plan_set_partitions; without them the call returns EUNSUPPORTED and says so.
 *   Sharing: EVERY call, on any plan and any stream of the device, uses the same array, which keeps the last call's
 *   contents (the call clears what it needs cleared).  Calls that overlap on the GPU -- two streams, two host threads --
 *   RACE: keep them on one stream, or order them with events.  F and Fk are written only by this call's last kernels.
 * Errors: as fstat_eval_batch, plus EUNSUPPORTED as above; never ENOMEM.
 */
FSTAT_API fstat_status fstat_eval_batch_noalloc(fstat_plan *plan, int64_t P, const double *params, double *F, double *Fk,
                                                void *cuda_stream);
FSTAT_API int64_t fstat_noalloc_scratch_bytes(void);

/*
 * fstat_eval_batch_bands -- SURVEY row f2: the semi-coherent F-statistic with the paper's OWN segment
 * limits (the number of segments is the same for all templates; the lowest and highest
 * limits are "the lowest and highest instantaneous frequencies occurring during the observation period
 * in the template").  For every particle the template is windowed to the bins [k_lo, k_hi) of the plan's
 * grid whose stationary time t_f = (1/2pi) dPsi_0/df (Eq. 20 :220) lies in [0, T_obs], T_obs = 1/df
 * (k_lo = number of bins with t_f < 0, k_hi = number with t_f <= T_obs), and that band is cut into n_seg
 * partitions with edges (reading A26)
 *     e_j = min(C (q_lo + floor(j (q_hi - q_lo) / n_seg)), n_bins),  q = floor((k + C/2) / C),  C = edge_lattice,
 * j = 0..n_seg; F_k over [e_j, e_{j+1}) as in fstat_eval_batch, an empty partition gives F_k = 0, F = sum_k F_k.
 * The plan's own partition edges play no role.
 *
 *   params  [P][6] DEVICE pointer as in fstat_eval_batch.
 *   n_seg   >= 1; edge_lattice >= 1 bins (1 = edges at any bin).
 *   F       [P] DEVICE pointer, out.   Fk  [P][n_seg] DEVICE pointer, out; may be NULL.
 *   band    [P][2] int64 DEVICE pointer, out: k_lo, k_hi of every particle; may be NULL.
 * Invalid particles get F = F_k = -inf and band (0, 0).  Asynchronous on cuda_stream.
 * Work: the interpolating kernel with per-THREAD partition edges: all templates of a CTA walk the
 * same bins, each cuts its running sums at its own edges; a partition that lies inside one work segment is finished in
 * the thread, the others are stitched from one head and one tail record per (work segment, template).  Templates with
 * an empty partition or one shorter than 8 bins are evaluated partition by partition with the full model; with
 * options.force_level == -1 (or a grid that starts within 1025 bins of f = 0) so is every in-band bin.
 * Workspace: 160 bytes per (work segment, particle) -- 73 MB for 2048 particles on the 2.5-yr grid -- plus, once per
 * plan, prefix tables of 70 bytes per bin.  X, Y, Z plans only (EUNSUPPORTED for tdi_channel A, E, T).
 * Errors: EINVAL (NULL plan/params/F, n_seg < 1, edge_lattice < 1), ENOMEM, ECUDA, EUNSUPPORTED.
 */
FSTAT_API fstat_status fstat_eval_batch_bands(fstat_plan *plan, int64_t P, const double *params, int32_t n_seg,
                                              int32_t edge_lattice, double *F, double *Fk, int64_t *band,
                                              void *cuda_stream);

/* Rows f2 x f3: the extrinsic amplitudes a = M^-1 N (Eq. 10 :96) of every partition of every template's band, as
 * fstat_eval_amplitudes gives them for the plan's partitions: amp [P][n_seg][4] DEVICE pointer, out (a_1..a_4; NaN
 * for invalid particles, 0 for empty partitions).  n_seg = 1 is the coherent estimate over the template's band
 * that App. B starts from. */
FSTAT_API fstat_status fstat_eval_amplitudes_bands(fstat_plan *plan, int64_t P, const double *params, int32_t n_seg,
                                                   int32_t edge_lattice, double *amp, void *cuda_stream);

/* fstat_eval_batch_bands with HOST buffers (params_host [P][6] in; F_host [P], Fk_host [P][n_seg] or NULL,
 * band_host [P][2] or NULL out): copies inside, returns after the results have landed.  Pinned buffers make the
 * copies asynchronous DMA. */
FSTAT_API fstat_status fstat_eval_batch_bands_host(fstat_plan *plan, int64_t P, const double *params_host,
                                                   int32_t n_seg, int32_t edge_lattice, double *F_host,
                                                   double *Fk_host, int64_t *band_host, void *cuda_stream);

/*
 * fstat_eval_batch_channels -- SURVEY row f4, the channel sum of PAPER.md:62 Eq. 3: with several TDI combinations I
 * of mutually independent noise, Lambda = sum_I [<s^I, h^I>_I - |h^I|_I^2 / 2] and the four amplitudes of Eq. 5 are
 * common to all of them, so N^i = sum_I <d_I, A^i_I>_I, M^ij = sum_I <A^i_I, A^j_I>_I and F_k = N.M^-1.N / 2.
 * One plan per channel: its own data and 1/S_n^I, and its own response through options.tdi_channel.  Eq. 3 ASSUMES
 * independent noise between the channels: that holds for {A, E, T} and NOT for {X, Y, Z}, whose noises
 * are correlated -- the call adds whatever set it is given (the sum over X, Y, Z is then not a likelihood ratio; it
 * is accepted because the paper leaves the choice of combinations open, and tests use it).  All plans must share the
 * device, the grid, the partition edges and the other options.  Two or three plans of the A / E / T family (any
 * order, same orbit and tolerances) go through ONE pass of a fused interpolating kernel: the node model (phase, t_f,
 * orbit, the three arms, X', Y', Z') and the per-bin carrier are evaluated once per template and shared, each channel
 * keeps its own data stream, Gram tables and eight sums (csrc/fstat_fastmulti.cu; 9 + 10 n FP64 instructions per bin
 * against 19 n).  Any other set (X, Y, Z plans, four channels, options.no_channel_fusion) runs the a1-a5 kernels once
 * per channel.  One epilogue adds the channels' sums and solves.
 *
 *   plans   HOST array of n_channels (1..4) plan handles, all different.
 *   params, F, Fk, cuda_stream as in fstat_eval_batch (Fk is [P][N_p]).
 * Errors: EINVAL (NULL, mismatching plans), EUNSUPPORTED (> 4 channels), ENOMEM, ECUDA; the reason is stored in
 * plans[0].
 */
FSTAT_API fstat_status fstat_eval_batch_channels(fstat_plan *const *plans, int32_t n_channels, int64_t P,
                                                 const double *params, double *F, double *Fk, void *cuda_stream);

/*
 * fstat_eval_amplitudes -- the maximum-likelihood extrinsic amplitudes a = M^-1 N of every partition
 * (Eq. 10; a_1..a_4 multiply the basis templates A^1 = u_+, A^2 = u_x, A^3 = i u_+, A^4 = i u_x of
 * Eq. 5 :77, and are the reparameterisation of (D_L, psi, iota, phi_c) of Eq. B1 :413 up to the amplitude
 * constant of Eq. A2 :402, which the templates drop -- DESIGN.md reading A21).  Same kernels as
 * fstat_eval_batch up to the last one; N_p = 1 gives the coherent estimate App. B asks for.
 *
 *   params  [P][6] DEVICE pointer as in fstat_eval_batch.
 *   amp     [P][N_p][4] DEVICE pointer, row-major, out: a_1, a_2, a_3, a_4.  Invalid particles get NaN; a
 *           partition whose M is rank-deficient gets the solution with the degenerate component set to 0.
 * Asynchronous on cuda_stream.  Errors as fstat_eval_batch.
 */
FSTAT_API fstat_status fstat_eval_amplitudes(fstat_plan *plan, int64_t P, const double *params, double *amp,
                                             void *cuda_stream);

/*
 * fstat_extrinsic_from_amplitudes -- App. B (Eq. B2-B3 :426-440): the maximum-likelihood extrinsic
 * parameters from ONE amplitude vector a = M^-1 N (fstat_eval_amplitudes / _bands at the best intrinsic point, N_p = 1).
 * Plain host arithmetic, no device, no plan.
 *   a               HOST [4]: a_1..a_4.
 *   chirp_mass_msun > 0: `a` are the library's amplitudes, whose templates drop the amplitude constant of Eq. A2 (:402,
 *                   reading A21); it is restored and D_L comes out in metres.  <= 0: `a` are the paper's a_i and D_L
 *                   comes out in their inverse units.
 *   out             HOST [4]: D_L, iota, psi, phi_c.  iota in [0, pi]; psi in (-pi/4, pi/4] (the branch of the paper's
 *                   arctan); phi_c in (-pi, pi]: the paper's arctan plus the half-plane that reproduces the sign of the
 *                   amplitudes (reading A25).  All-zero amplitudes give D_L = +inf and zeros.
 * What the four numbers mean physically is fixed by a test, not by convention (pin P20, reading A31): amplitudes
 * estimated from the time-domain TDI signal of a quadrupole-formula binary at a known distance and orientation give back
 * D_L within 5 % (the residual of the paper's N = 0 response) and iota within 0.05 rad; iota is the angle between the
 * orbital angular momentum and the propagation direction (source -> observer), psi = pi/2 - (angle of its sky
 * projection from u towards v) modulo pi/2, and advancing the wave's phase lowers phi_c by as much.
 * Errors: EINVAL (NULL pointer, non-finite input).
 */
FSTAT_API fstat_status fstat_extrinsic_from_amplitudes(const double *a, double chirp_mass_msun, double *out);

/* Eq. B1 (:413-420), the forward map: a_out HOST [4] = a_1..a_4 of (D_L, psi, iota, phi_c), D_L > 0 in the inverse units of
 * the amplitudes.  EINVAL for a NULL pointer, D_L <= 0 or non-finite input. */
FSTAT_API fstat_status fstat_amplitudes_from_extrinsic(double d_l, double psi, double iota, double phi_c, double *a_out);

/*
 * fstat_eval_batch_host -- the same evaluation with HOST buffers: copies params to the device,
 * evaluates, copies F (and Fk when non-NULL) back and waits for completion before returning.
 * Pinned host memory makes the copies asynchronous DMA; pageable memory works too.
 * When the F_k block is large (P N_p 8 B >= 2 MiB) the interpolating kernel is launched as up to 5 ranges of partitions
 * on streams the plan owns (one per CUDA stream priority, the earlier range the higher), and a copy stream runs each
 * range's epilogue and the copy of its F_k columns under the later ranges' kernels; everything is ordered after the
 * work already queued on cuda_stream and joined into it before the call returns.  Same kernels, same sums: the
 * results equal fstat_eval_batch's bit for bit.  Config 1: 5.19 ms against 5.11 ms device-resident (the copy alone
 * is 0.3 ms).
 */
FSTAT_API fstat_status fstat_eval_batch_host(fstat_plan *plan, int64_t P,
                                             const double *params_host, double *F_host,
                                             double *Fk_host, void *cuda_stream);

/*
 * fstat_eval_template -- NOT on the hot path: write the two complex basis templates of ONE parameter
 * vector over the plan's whole grid,
 *     u_P(f_k) = T_P(f_k; t_f) f_k^(-7/6) exp(-i Psi_0(f_k)),  P in {+, x}
 * (PAPER.md:397 Eq. A1 with the amplitude constant of Eq. A2 dropped, reading A21; :206
 * Eq. 17 with N = 0), from which the four real basis templates of PAPER.md:77 Eq. 5 are
 * A^1 = u_+, A^2 = u_x, A^3 = i u_+, A^4 = i u_x.  It runs the same device code as fstat_eval_batch
 * and exists to synthesise injections (h = sum a_i A^i) and for element-wise tests.
 *
 *   params_host  [6] HOST pointer (t_c, M_c, eta, theta, phi, e0); an invalid vector is EINVAL here.
 *   u_plus, u_cross  [N][2] DEVICE pointers, interleaved re, im, out.
 * Synchronous: returns after the stream has finished the work.
 */
FSTAT_API fstat_status fstat_eval_template(fstat_plan *plan, const double *params_host,
                                           double *u_plus, double *u_cross, void *cuda_stream);

/* fstat_plan_destroy -- free a plan and its device memory.  NULL is allowed. */
FSTAT_API void fstat_plan_destroy(fstat_plan *plan);

/* Plan introspection (all NULL-safe; return 0 / -1 for a NULL plan). */
FSTAT_API int64_t fstat_plan_n_bins(const fstat_plan *plan);
FSTAT_API int32_t fstat_plan_n_part(const fstat_plan *plan);
FSTAT_API int32_t fstat_plan_device(const fstat_plan *plan);
/* Number of CTAs the interpolating main kernel launches for P particles: particle groups of 128 x chunks of
 * consecutive segments (a chunk is one segment unless the partitions are short). */
FSTAT_API int64_t fstat_plan_n_ctas(const fstat_plan *plan, int64_t P);
/* Work of the interpolating kernel in the most recent fstat_eval_batch_bands call on this plan, counted per WARP of 32
 * templates (a warp walks the union of its lanes' bands): out HOST [5] = bins, node intervals, node intervals in which
 * some lane had a partition edge, runs (work segments entered), and the internal-invariant flag (0 = fine).
 * Synchronises the device.  For the roofline of the bench line. */
FSTAT_API fstat_status fstat_plan_band_stats(fstat_plan *plan, int64_t *out);
/* Bytes of device memory held by the plan's persistent tables: the folded data and (f, w') (32 bytes per bin), the
 * node rows (192 bytes per 8 bins), the Gram matrices of the current partitions and, after the first
 * fstat_eval_batch_bands call, the prefix Gram tables (70 bytes per bin).  Workspace (grown per batch size) not included. */
FSTAT_API int64_t fstat_plan_table_bytes(const fstat_plan *plan);
/* Number of CUDA kernels the evaluation calls on this plan have launched so far (per fstat_eval_batch: slot keys,
 * ranking, prologue, stride selection, interpolating main kernel, direct main kernel, epilogue, and the chunk sums of
 * F when the partitions are split over several epilogue blocks; a radix sort above 16384 particles counts as one). */
FSTAT_API int64_t fstat_plan_launch_count(const fstat_plan *plan);
/* How the most recent fstat_eval_batch on this plan was split between the direct kernel and the seven
 * strides of the interpolating kernel: bins_out[0] / [1..7] = sum over the (particle group, segment) work
 * items run by the direct kernel / at stride 8, 16, 32, 64, 128, 256, 512 of the segment's bin count
 * (multiply by 128 particles per group for template-bins); subblocks_out[1..7] = number of node intervals
 * those items walked (one full-model node evaluation each).  HOST arrays of 8.  Synchronises the device. */
FSTAT_API fstat_status fstat_plan_level_bins(fstat_plan *plan, int64_t *bins_out, int64_t *subblocks_out);
/* Device time of the main (fused template + inner product) kernels in the most recent evaluations on
 * this plan: CUDA events are recorded on the call's stream around that kernel at every fstat_eval_batch
 * (ring of 128).  Writes the milliseconds of the last min(n_last, 128, evaluations so far) calls, oldest
 * first, to the HOST array ms_out and returns how many were written.  Synchronises on those events. */
FSTAT_API int32_t fstat_plan_main_kernel_ms(fstat_plan *plan, int32_t n_last, double *ms_out);

/*
 * fstat_edges_equal_bins -- "equal-bin partitions": e_j = floor(j * n_bins / n_part), j = 0..n_part,
 * written to the HOST array edges_out[n_part+1].  EINVAL if n_part < 1 or n_part > n_bins.
 */
FSTAT_API fstat_status fstat_edges_equal_bins(int64_t n_bins, int32_t n_part, int64_t *edges_out);

/*
 * fstat_probe_pipe_peak -- measure, on the given device, the sustained rate of a dependent-free stream
 * of FP64 FMA (which = 0), FP32 FMA (which = 1) or MUFU.SIN (which = 2) instructions, in thread-level
 * instructions per second, over roughly `millis` milliseconds.  It is the measured denominator of the
 * "alu" roofline bench.py reports.  which = 3: the FP64 FMA stream with one FP32 FMA after
 * every four FP64 ones, reported as FP64 instructions per second -- the drop against which = 0 is what an instruction
 * of another pipe costs a kernel that is bound by the FP64 pipe (the "dispatch" entry of the roofline).  Also
 * returns the SM count.
 */
FSTAT_API fstat_status fstat_probe_pipe_peak(int32_t device, int32_t which, double millis,
                                             double *inst_per_s, int32_t *n_sm);

/* ------------------------------------------------------------------------------------------------
 * Particle swarm optimisation on the device (Sec. III.A; Eq. 13-14 :146-150).
 *
 * n_swarms independent swarms (PSO runs, :160) of n_particles each are advanced together: every iteration
 * is "update velocities and positions -> ONE fstat_eval_batch over all particles -> update personal bests",
 * enqueued on the caller's stream with no host synchronisation.  Settings as in the paper (:158-162): lbest
 * ring topology (neighbours i-1, i, i+1), x ~ U[lo, hi], v ~ U[lo - x, hi - x] at the start, |v| <= v_max
 * (in box units), inertia falling linearly from w_start to w_end over n_iter_total iterations, "let them
 * fly": a particle outside [lo, hi] keeps moving but gets fitness -inf (its parameters are sent as NaN).
 * Random numbers: Philox4x32-10, counter (particle, iteration, draw, 0), key = seed.
 * ------------------------------------------------------------------------------------------------ */
typedef struct fstat_pso fstat_pso;      /* opaque */
typedef struct {
    double c1, c2;            /* acceleration constants, default 2, 2 (:162)          */
    double v_max;             /* velocity clamp in box units, default 0.5 (:162)      */
    double w_start, w_end;    /* inertia weight at the first / last iteration: 0.9, 0.4 */
    int32_t band_n_seg;       /* 0 (default): fitness = fstat_eval_batch with the plan's partitions;
                                 >= 1: fitness = fstat_eval_batch_bands with this many segments per template
                                 (the paper's own segment limits)                             */
    int32_t band_lattice;     /* edge lattice of that call in bins, default 1 (edges at any bin)          */
} fstat_pso_options;

FSTAT_API void fstat_pso_default_options(fstat_pso_options *opts);

/* Draw the initial swarms and evaluate them (asynchronous on cuda_stream).  lo, hi: HOST [6] box of
 * (t_c, M_c, eta, theta, phi, e0).  The plan must outlive the fstat_pso and is used by it for every
 * evaluation (one evaluation in flight per plan).  EINVAL for bad sizes / box / options. */
FSTAT_API fstat_status fstat_pso_create(fstat_pso **out, fstat_plan *plan, int32_t n_swarms, int32_t n_particles,
                                        int32_t n_iter_total, const double *lo, const double *hi, uint64_t seed,
                                        const fstat_pso_options *opts, void *cuda_stream);
/* The same with one box PER SWARM: lo, hi HOST [n_swarms][6].  The hierarchy of PAPER.md:168-174 runs its PSO runs over
 * different boxes (24 t_c intervals in stage 1, 24 candidate-centred boxes in stage 2): one object and one batched
 * evaluation per iteration serve them all; fstat_pso_best returns the best of every swarm, the best-of-runs per box
 * (:160) is a maximum over the swarms that share a box. */
FSTAT_API fstat_status fstat_pso_create_boxes(fstat_pso **out, fstat_plan *plan, int32_t n_swarms, int32_t n_particles,
                                              int32_t n_iter_total, const double *lo, const double *hi, uint64_t seed,
                                              const fstat_pso_options *opts, void *cuda_stream);
/* Advance all swarms by n_iter iterations; only enqueues work. */
FSTAT_API fstat_status fstat_pso_iterate(fstat_pso *pso, int32_t n_iter, void *cuda_stream);
/* Best position (physical parameters) and fitness of every swarm so far: HOST [n_swarms][6], [n_swarms].
 * Waits for the stream. */
FSTAT_API fstat_status fstat_pso_best(fstat_pso *pso, double *best_params_host, double *best_f_host,
                                      void *cuda_stream);
/* Copy of the swarm state for tests and check-pointing: HOST x, v, pbest [N][6] (unit-box coordinates),
 * pbest_f, f_last [N], N = n_swarms * n_particles; any pointer may be NULL.  Waits for the stream. */
FSTAT_API fstat_status fstat_pso_state(fstat_pso *pso, double *x, double *v, double *pbest, double *pbest_f,
                                       double *f_last, void *cuda_stream);
FSTAT_API int32_t fstat_pso_iterations_done(const fstat_pso *pso);
FSTAT_API void fstat_pso_destroy(fstat_pso *pso);       /* NULL is allowed */

FSTAT_API const char *fstat_status_str(fstat_status s);
/* Human-readable reason of the most recent failing call on this plan; plan == NULL returns the
 * reason of the most recent failing fstat_plan_create on the calling thread.  Never NULL. */
FSTAT_API const char *fstat_last_error(const fstat_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* FSTAT_H_ */
