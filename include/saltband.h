/* saltband.h -- C ABI of the B200-native SALT3 batched band-flux library (libsaltband.so).
 *
 * The operations are those of the JAX-bandflux paper (arXiv 2504.08081; PAPER.md) as fixed by
 * BASELINE.json `north_star` and the readings G0-G15 listed in DESIGN.md:
 *
 *   PAPER.md:19-23  F(p, lam) = x0 [M0(p,lam) + x1 M1(p,lam)] exp(c CL(lam)); free parameters
 *                   x0, x1, t0, c; p is a function of redshift and t - t0
 *   PAPER.md:38-43  bandflux = int F(lam) T(lam) lam/(hc) dlam over the band
 *   PAPER.md:45     "trapezoidal integration along the wavelength dimension"; batching over data
 *                   instances
 *   PAPER.md:47     dedicated interpolation routines for the SALT3 / SALT3-NIR surfaces
 *   north_star      p = (t - t0)/(1+z), lam_rest = lam_obs/(1+z); bicubic interpolation on the
 *                   (phase, wavelength) grid; zero-point normalisation; chi^2 per supernova;
 *                   analytic gradient with respect to (x0, x1, c, t0)
 *
 * One evaluation ("eval") = one (supernova s, parameter sample k, observation i):
 *
 *   m = S_i * x0 * sum_j w_j * [M0(p, l_j) + x1 M1(p, l_j)] * exp(c CL(l_j)) * T_j * lam_j/(hc)
 *       p = (t_i - t0)/(1+z_s),  l_j = lam_j/(1+z_s),  lam_j, T_j = grid/transmission of band b_i,
 *       w_j = trapezoid weights of that grid, S_i = 10^(0.4 zp_i)/ZPAB_b (1 if zp == NULL),
 *       ZPAB_b = the same trapezoid of (3.631e-20 erg/s/cm^2/Hz * c/lam^2) T lam/(hc)        [G7]
 *   M(p, l): separable cubic convolution (Keys a = -1/2) on the uniform model grid, linear in the
 *       first/last cell of each axis, zero outside the closed grid range                [G1-G3]
 *   CL(l): polynomial in (l - cl_wave_b)/(cl_wave_v - cl_wave_b) on [cl_lo, cl_hi], continued
 *       linearly (value and slope) outside                                                 [G5]
 *   Conventions against SNCosmo-style SALT code (readings G5, G6): the exponent is NATURAL, exp(c CL) -- a
 *       colour law given for 10^(-0.4 c CL') is passed as cl_coef[q] = -0.4 ln(10) a'_q; and there is NO
 *       1/(1+z) flux-dilution factor -- the x0 of this library is such a code's x0/(1+z).
 *
 * Conventions
 *   - Loaders take HOST pointers and copy; compute calls take DEVICE pointers owned by the caller
 *     (e.g. torch tensors) and a cudaStream_t passed as void*.  Compute calls only enqueue work on
 *     that stream: no host synchronisation, no retained pointers, no allocation visible to the
 *     caller.  A call with sb_batch.pack set touches no memory but its arguments.  A call without a
 *     pack needs a few hundred KB of scratch (redshift order of the batch); it lives in a workspace
 *     owned by the sb_bands handle, one per stream, allocated (cudaMalloc) by the first call on that
 *     stream or when a larger batch arrives, never by later calls -- so a warmed-up call can be
 *     captured into a CUDA graph -- and released by sb_free_bands.
 *   - dtype selects the element type of every floating-point array of a compute call (inputs and
 *     outputs): SB_F32 (production: per-sample arithmetic in fp32) or SB_F64 (verification).
 *   - All functions return SB_OK (0) or a negative sb_status; sb_strerror() names it.  Device data
 *     are not validated (that would need a sync): a band index outside [0, n_bands) gives NaN for
 *     that evaluation; fluxerr <= 0 propagates inf/NaN into chi^2; a phase or wavelength outside
 *     the model grid is not an error and contributes zero flux [G3].
 *   - No global mutable state.  Model, band and pack tables are immutable after creation;
 *     concurrent compute calls from several host threads on distinct streams with the same handles
 *     are allowed (the per-stream workspaces above are the only thing a call may create, under a
 *     lock).  Handles belong to the device that was current when they were created: a compute call
 *     made with another current device returns SB_EINVAL.
 *   - There is no CPU fallback: without a CUDA device every compute call returns SB_ECUDA.
 */
#ifndef SALTBAND_H
#define SALTBAND_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sb_model sb_model; /* opaque: device-resident M0, M1 tables and the colour law */
typedef struct sb_bands sb_bands; /* opaque: device-resident band tables, folded weights, ZPAB */
typedef struct sb_pack sb_pack;   /* opaque: theta-independent precompute of one batch (optional) */

typedef enum { SB_F32 = 0, SB_F64 = 1 } sb_dtype;

/* Formulation bits, OR-ed into sb_batch.dtype (optional; 0 = the library picks the fastest that
 * applies).  Both formulations compute the same sums for every evaluation; they differ in what is
 * shared between evaluations (G_geom / G_col):
 *   SB_FORM_DIRECT   one warp per evaluation, geometry and colour factor recomputed per evaluation
 *                    (G = 1); any band grid, fp32 or fp64, forward or gradient.
 *   SB_FORM_GROUPED  the observations of a unit that share a band are integrated together, sharing
 *                    the rest-frame geometry and the colour factor; fp32 forward calls with uniform
 *                    band grids only -- a call that demands it where it does not apply returns
 *                    SB_ELIMIT.
 *   SB_FORM_TILED    the node-weight kernel (csrc/sb_nw.cuh): as SB_FORM_GROUPED, and the observations
 *                    of a group of units that are neighbours in redshift are ordered by phase so
 *                    that the model rows they read stay in registers; fp32
 *                    forward AND gradient calls, uniform or non-uniform band grids, at most 64 bands;
 *                    same error behaviour.  The only formulation that uses sb_batch.pack. */
enum { SB_FORM_DIRECT = 0x100, SB_FORM_GROUPED = 0x200, SB_FORM_TILED = 0x400 };

typedef enum {
    SB_OK = 0,
    SB_EINVAL = -1, /* NULL pointer, bad count, non-uniform / non-increasing grid, non-finite table */
    SB_ENOMEM = -2, /* host or device allocation failed */
    SB_ECUDA = -3,  /* no device, or a copy / launch failed (see sb_last_cuda_error) */
    SB_ELIMIT = -4  /* a table exceeds what the kernels stage on chip */
} sb_status;

/* sb_load_model -- PAPER.md:19-23, 47 (the M0/M1 surfaces and CL of the SALT model).
 *   phase[n_phase], wave[n_wave]  HOST, uniform (|spacing deviation| <= 1e-9 relative), strictly
 *                                 increasing, n_phase >= 2, n_wave >= 2 (days; Angstrom, rest frame)
 *   m0, m1                        HOST, row-major [n_phase][n_wave], wavelength fastest, finite
 *   cl_coef[n_cl]                 HOST, CL(l) = sum_q cl_coef[q] r^q, r = (l - cl_wave_b)/(cl_wave_v -
 *                                 cl_wave_b); 1 <= n_cl <= 8; natural exponent exp(c*CL)    [G5]
 *   cl_lo < cl_hi                 range (Angstrom, rest frame) outside which CL continues linearly
 *   out                           receives the handle; free with sb_free_model.
 * Copies everything (fp64 and fp32 device tables); the caller keeps ownership of its arrays. */
int sb_load_model(const double *phase, int32_t n_phase, const double *wave, int32_t n_wave,
                  const double *m0, const double *m1, const double *cl_coef, int32_t n_cl,
                  double cl_wave_b, double cl_wave_v, double cl_lo, double cl_hi, sb_model **out);

/* sb_load_bandpasses -- PAPER.md:38-43, 47 (tabulated transmission T(lam) per filter).
 *   CSR-packed HOST arrays: band b owns [offset[b], offset[b+1]) of wave/trans; each band has
 *   >= 2 points, wave strictly increasing (observer frame, Angstrom; uniform spacing not
 *   required), trans finite.  Precomputes in fp64 the trapezoid weights w_j, the
 *   folded weights w_j T_j lam_j/(hc) and ZPAB_b [G7].  Copies; caller keeps ownership. */
int sb_load_bandpasses(int32_t n_bands, const int64_t *offset, const double *wave,
                       const double *trans, sb_bands **out);

void sb_free_model(sb_model *m); /* NULL is allowed */
void sb_free_bands(sb_bands *b); /* NULL is allowed */

/* One batch of evaluations.  Every pointer is a DEVICE pointer owned by the caller.
 * "unit" u = s*n_samples + k is one (supernova, parameter sample). */
typedef struct {
    int32_t dtype;             /* sb_dtype of time, zp, z, x0, x1, c, t0 and of all outputs,
                                  optionally OR-ed with one SB_FORM_* bit */
    int32_t n_sn;              /* supernovae, >= 0 */
    int32_t n_samples;         /* parameter samples per supernova, >= 1 */
    int32_t n_obs_total;       /* = obs_offset[n_sn] (host copy, so no sync is needed) */
    const int32_t *obs_offset; /* [n_sn+1] CSR into the observation arrays; ragged allowed */
    const void *time;          /* [n_obs_total] observer-frame time t_i (days) */
    const int32_t *band;       /* [n_obs_total] index into sb_bands */
    const void *zp;            /* [n_obs_total] zero point, or NULL => S_i = 1 (raw photon flux) */
    const void *z;             /* [n_sn] redshift, > -1 */
    const void *x0, *x1, *c, *t0; /* [n_sn*n_samples], sample fastest */
    const sb_pack *pack;       /* NULL, or the pack built by sb_pack_observations from this batch's
                                  n_sn and z (same model and bands); DEVICE calls only */
} sb_batch;

/* sb_pack_observations -- optional: everything the hot path needs that does not depend on the
 * free parameters (in a fit or a sampling run the observations and redshifts are
 * fixed over thousands of calls, only x0, x1, c, t0 change).  Holds the redshift order of the
 * supernovae (stable sort: neighbours in z share their window of the model surfaces) and, per
 * (supernova, band), the rest-frame geometry of the band integral (in-range samples decided in
 * fp64 [G9], model cells spanned, colour-law regime).  Reads batch->n_sn, batch->dtype (SB_F32
 * only) and the DEVICE array batch->z; the other fields are ignored.  Allocates the pack's device
 * memory and enqueues its build on `stream` (no host synchronisation: use the pack on the same
 * stream, or synchronise first).  A compute call whose batch points to the pack must pass the
 * same n_sn, model and bands and the same device array z it was built from (else SB_EINVAL: the
 * pack holds geometry computed from those redshifts; the pointer is compared, the values are not, so do
 * not overwrite z in place between the build and the last use).  Kernels that do not use a pack (fp64,
 * SB_FORM_DIRECT, SB_FORM_GROUPED) ignore it.  SB_ELIMIT when the band set is one the node-weight kernel
 * does not handle (more than 64 bands); non-uniform band grids are fine. */
int sb_pack_observations(const sb_model *m, const sb_bands *b, const sb_batch *batch, void *stream,
                         sb_pack **out);
void sb_free_pack(sb_pack *p); /* NULL is allowed; free after the work that uses it has finished */

/* sb_bandflux -- the band flux m of every evaluation.
 *   out_flux  DEVICE [n_obs_total*n_samples]: supernova s occupies the block starting at
 *             obs_offset[s]*n_samples, laid out [n_samples][n_obs(s)], observation fastest. */
int sb_bandflux(const sb_model *m, const sb_bands *b, const sb_batch *batch, void *out_flux,
                void *stream);

/* sb_chi2 -- chi^2 per unit: sum_i ((flux_i - m_i)/fluxerr_i)^2 over the supernova's observations
 * (north_star; reading G10: diagonal, data errors only).  Summation order is fixed, so repeated
 * calls are bit-identical.
 *   flux, fluxerr  DEVICE [n_obs_total] measured flux and its 1-sigma error
 *   out_chi2       DEVICE [n_sn*n_samples]
 *   out_flux       DEVICE, layout as in sb_bandflux, or NULL */
int sb_chi2(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
            const void *fluxerr, void *out_chi2, void *out_flux, void *stream);

/* sb_bandflux_grad -- forward plus analytic gradient with respect to (x0, x1, c, t0), in that
 * order (north_star; "fully differentiable").
 *   out_flux   DEVICE, layout as in sb_bandflux, or NULL
 *   out_dflux  DEVICE [n_obs_total*n_samples][4] d m / d(x0, x1, c, t0), same eval order, or NULL;
 *              out_dflux and out_dchi2 must be aligned to 4 elements (16 bytes in fp32): they are
 *              written as vectors (SB_EINVAL otherwise)
 *   flux, fluxerr  DEVICE [n_obs_total], required iff out_chi2 or out_dchi2 is non-NULL
 *   out_chi2   DEVICE [n_sn*n_samples] or NULL
 *   out_dchi2  DEVICE [n_sn*n_samples][4] = -2 sum_i (flux_i - m_i)/fluxerr_i^2 * dm_i, or NULL
 * The derivative with respect to t0 is that of the interpolation cell selected by the phase
 * (reading G11); it is zero outside the grid. */
int sb_bandflux_grad(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                     const void *fluxerr, void *out_flux, void *out_dflux, void *out_chi2,
                     void *out_dchi2, void *stream);

/* sb_chi2_host / sb_bandflux_grad_host -- the same operations for data that lives in HOST memory
 * (the end-to-end path of a fit driver that keeps its light curves on the host).  Every pointer of
 * `batch`, flux, fluxerr and every output is a HOST pointer with the layout of the device call;
 * pinned (page-locked) buffers give the full PCIe rate, pageable ones work.  The library cuts the
 * supernovae into chunks, stages each chunk through device buffers owned by the sb_bands handle
 * (one set per concurrent host call, grown on demand, released by sb_free_bands) and overlaps
 * host->device copies, kernels and device->host copies of consecutive chunks on internal streams;
 * batch->pack must be NULL.  Results are those of the device call on each
 * chunk: identical to the whole-batch device call in the direct formulation, and within rounding
 * (the parity tolerance) in the tiled one, whose summation order depends on which supernovae share
 * a group.  The call returns when all outputs are complete (it synchronises its streams);
 * sb_last_launch_count() then reports the kernels of all chunks.  Errors as for the device calls. */
int sb_chi2_host(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                 const void *fluxerr, void *out_chi2, void *out_flux);
int sb_bandflux_grad_host(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                          const void *fluxerr, void *out_flux, void *out_dflux, void *out_chi2,
                          void *out_dchi2);

/* sb_chi2_noalloc -- sb_chi2 (same arguments, same outputs, same error codes) for callers that must not
 * allocate device memory.  Two kinds of caller are meant: a process whose GPU memory has been handed, all of
 * it, to another component's pool at start-up (an inference server, a framework's caching allocator with the
 * device filled), so that a cudaMalloc issued from inside this library would fail; and a latency-bound loop
 * that cannot afford the device-wide synchronisation a cudaMalloc may imply.  sb_chi2 keeps its scratch (the
 * redshift order of the batch, a few hundred KB) in a workspace it allocates on the first call per stream;
 * this call keeps the same scratch in a fixed array that is part of the library image instead, so it never
 * calls cudaMalloc, cudaFree or any allocating library routine.
 *   Limits       SB_F32 batches only, node-weight formulation only (SB_FORM_TILED is implied; another
 *                formulation bit -> SB_EINVAL; calls of fewer than 4096 evaluations run the direct kernel,
 *                which has no scratch, as they do in sb_chi2), batch->pack must be NULL (SB_EINVAL: a pack already makes
 *                sb_chi2 allocation-free), and batch->n_sn <= SB_NOALLOC_MAX_SN -- a larger batch is refused
 *                with SB_ELIMIT before anything is enqueued (cut it into several calls).  A model or band set
 *                the node-weight kernel does not take (more than 64 bands, ...) also gives SB_ELIMIT: there
 *                is no fall-back to a kernel that would allocate.
 *   Cost         the array (about 1 MB for SB_NOALLOC_MAX_SN = 131072) is reserved on every GPU on which the
 *                process loads this library, from load until the process exits, whether or not the call is
 *                ever made.
 *   First call   the first call on each device looks up the array's device address (with that device
 *                current) and remembers it; make that first call during set-up, before starting any stream
 *                capture.  Later calls on that device do no set-up.
 *   Sharing      every call on a device uses the SAME array, whatever its stream or host thread, and the
 *                array keeps what the previous call left in it (the call clears the part that must start at
 *                zero itself).  Two calls whose GPU work can overlap -- distinct streams with no dependency
 *                between them -- race on it and give wrong results; order them (same stream, or an event). */
#define SB_NOALLOC_MAX_SN 131072
int sb_chi2_noalloc(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                    const void *fluxerr, void *out_chi2, void *out_flux, void *stream);

/* sb_fit_lbfgs -- device-resident batched fit of (x0, x1, c, t0): every unit (supernova, parameter sample)
 * is one optimiser LANE that minimises its own chi^2 ("fmin_bfgs.py ... optimisation via
 * L-BFGS-B" is one of the paper's two workloads; the paper gives no algorithmic detail, the algorithm is
 * reading G16 of DESIGN.md).  Limited-memory BFGS (two-loop recursion, `memory` curvature pairs) with a
 * backtracking Armijo line search (c1 = 1e-4, step halved on rejection, at most 30 halvings) and an
 * optional box (trial points are projected on it).  Lanes work in scaled variables u = theta / s,
 * s = (x0 of the start point, 1, 1, 1).  One STEP = one batched evaluation of chi^2 and its gradient at
 * every running lane's trial point (the kernels of sb_bandflux_grad, through batch->pack when given)
 * plus one lane-update kernel; the call enqueues exactly max_eval steps on `stream` and returns: there
 * is NO host synchronisation and no device-to-host copy.  Stopped lanes are skipped by the evaluation
 * kernels, and steps after the last lane has stopped return at once.
 *   batch          as for sb_bandflux_grad; x0, x1, c, t0 are the START point of every lane (not modified)
 *   flux, fluxerr  DEVICE [n_obs_total], required
 *   opts           see sb_fit_opts; all fields must be set (sb_fit_default_opts fills the defaults)
 *   result         DEVICE outputs, written when a lane stops (all lanes have stopped when the call's work
 *                  is complete): theta [n_units][4] = (x0, x1, c, t0) of the last accepted point and chi2
 *                  [n_units], both of the batch's element type; optional int32 status (0 running -- never
 *                  seen after completion, 1 converged, 2 line search stalled, 3 budget exhausted), n_iter
 *                  (accepted steps), n_eval (evaluations) [n_units]; optional trace [trace_len][n_units]
 *                  fp64: chi^2 after i accepted steps (row 0: start point; NaN where not reached).
 * A lane converges when an accepted step lowers chi^2 by <= ftol * max(|chi2_old|, |chi2_new|, 1) or
 * when max_k |d chi^2 / d u_k| <= gtol.  In SB_F32 batches every trial point is rounded to fp32 (the
 * kernels take fp32 parameters) and chi^2 comes back in fp32, so a decrease below a few fp32 ulps cannot be
 * observed: there a positive ftol below 2^-21 (4.8e-7) is raised to 2^-21 (the default 1e-12 included);
 * ftol = 0 switches the test off in either precision.  Lane state and all optimiser arithmetic are fp64.
 * With a box, every evaluated and every returned theta satisfies lo <= theta <= hi exactly in the batch's
 * element type (the point is clamped again after scaling and rounding).  Lane state lives in a
 * workspace owned by the sb_bands handle (one per stream, as for the compute calls; ~0.7 KB per lane).
 * Errors as for the compute calls; SB_EINVAL for out-of-range options. */
typedef struct {
    int32_t memory;    /* curvature pairs kept per lane, 1..8 (default 8) */
    int32_t max_eval;  /* evaluations per lane = steps enqueued, >= 1 (default 60) */
    int32_t max_iter;  /* accepted steps per lane, >= 1 (default 1000) */
    int32_t trace_len; /* rows of result->trace (0: no trace) */
    double ftol, gtol; /* >= 0 (defaults 1e-12, 0; SB_F32 batches: see the ftol floor above) */
    const double *lo, *hi; /* HOST [4] box on (x0, x1, c, t0) in theta units, or NULL: no bound on that side */
} sb_fit_opts;

typedef struct {
    void *theta, *chi2;                /* [n_units][4], [n_units], element type of the batch; required */
    int32_t *status, *n_iter, *n_eval; /* [n_units] each, or NULL */
    double *trace;                     /* [trace_len][n_units] or NULL (required iff trace_len > 0) */
} sb_fit_result;

void sb_fit_default_opts(sb_fit_opts *opts);
int sb_fit_lbfgs(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                 const void *fluxerr, const sb_fit_opts *opts, const sb_fit_result *result, void *stream);
/* The same fit for data in HOST memory (every pointer of batch, flux, fluxerr and result is a HOST
 * pointer): copies the batch to a device buffer owned by the sb_bands handle, builds a pack, runs the
 * fit, copies the results back and returns when they are complete.  batch->pack must be NULL. */
int sb_fit_lbfgs_host(const sb_model *m, const sb_bands *b, const sb_batch *batch, const void *flux,
                      const void *fluxerr, const sb_fit_opts *opts, const sb_fit_result *result);

/* Introspection (host side, cheap). */
int32_t sb_bands_count(const sb_bands *b);
/* ZPAB_b as computed at load (fp64), or NaN for a bad index. */
double sb_bands_zpab(const sb_bands *b, int32_t band);
/* Number of kernels launched by the calling thread's most recent compute call (0 if it failed). */
int32_t sb_last_launch_count(void);
/* SB_FORM_* bit of the formulation that the calling thread's most recent compute call ran (0 if it
 * failed or launched nothing). */
int32_t sb_last_form(void);
/* cudaError_t of the calling thread's most recent failing CUDA call (0 if none). */
int32_t sb_last_cuda_error(void);
const char *sb_strerror(int status);
const char *sb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SALTBAND_H */
