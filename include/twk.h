/* twk.h -- C ABI of the B200-native finite-source binary-lens magnification library (libtwk.so).
 *
 * The operation: for every source centre zeta_c in a batch, the magnification mu = (total area of all images of
 * the uniform disk |zeta - zeta_c| <= rho under the binary-lens map, Eq.(1)) / (pi rho^2)
 * (PAPER.md:35), computed by contour integration: sample the source boundary, build the
 * quintic with the cancellation-free coefficients of Eq.(6), solve it in FP64, drop ghost roots
 * with the residual detector, link images of adjacent samples incl. creation/annihilation at caustic
 * crossings, sum the Stokes area with trapezium + parabolic corrections (Eq.(8)-(11)),
 * estimate the error (Eq.(17)-(18)) and refine the boundary by error-weighted inverse-transform
 * sampling until the estimate meets the requested relative accuracy.
 *
 * Conventions
 *  - Coordinates: the paper's centre-of-mass frame, Einstein-radius units (Eq.(2)): primary at
 *    z1 = -q s/(1+q), secondary at z2 = +s/(1+q), both on the real axis; q = m2/m1.
 *  - "DEVICE" pointers are CUDA device pointers owned by the caller (e.g. torch tensors); the library never
 *    frees, reallocates or retains them.  "HOST" pointers are ordinary host memory.
 *  - complex arrays are interleaved (re, im) doubles.
 *  - Device-pointer calls are asynchronous on `stream` and perform no host synchronisation.
 *  - A context owns ONE workspace: its calls must be issued on one stream at a time (stream order serialises them);
 *    use one context per stream for concurrent batches.  One context per device; create it with that device current.
 *  - Return value: TWK_OK or a negative TWK_E* code from synchronous argument validation / CUDA runtime errors.
 *    Device-side problems never abort a call: they set per-source status bits (TWK_ST_*).
 *  - There is no CPU fallback: every entry point that computes needs a CUDA device.
 */
#ifndef TWK_H_
#define TWK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TWK_OK 0
#define TWK_EINVAL (-1) /* null required pointer, N < 4, rel_tol <= 0, bad options, n_sources > max_sources */
#define TWK_ENOMEM (-2) /* workspace allocation failed */
#define TWK_ECUDA (-3)  /* a CUDA runtime call failed; twk_strerror gives the CUDA text of the last one */
#define TWK_ELIMIT (-4) /* twk_magnify_static: n_sources > TWK_STATIC_MAX_SOURCES (its scratch has a fixed size) */

/* per-source status bits (out_status) */
#define TWK_ST_CONVERGED 1u  /* error estimate <= rel_tol * |A|                                       */
#define TWK_ST_CAP 2u        /* sample cap reached: value and estimated error returned as the paper does */
#define TWK_ST_REPAIRED 4u   /* a sample's parity sum was not -1 and was repaired (reading G-5)        */
#define TWK_ST_DOMAIN 8u     /* s, q outside the validated domain 0.1<=s<=10, q>=1e-9: still computed;   */
                             /* non-finite / non-positive s, q, rho or non-finite zeta: out_mu = NaN             */
#define TWK_ST_NUMERIC 16u   /* a boundary sample sat on a lens and was moved off it by 1e-14 s (reading B-1; mu is */
                             /* finite and accurate), or a non-finite value appeared in the solve (mu = NaN)         */
#define TWK_ST_SLOPE 32u     /* the slope detector re-judged a real image pair as ghosts (reading G-4) */
#define TWK_ST_POINT 64u     /* point-source adequacy tests passed: out_mu = point-source magnification +   */
                             /* quadrupole term, no contour was integrated, out_nsamples = 0                        */

typedef struct twk_ctx twk_ctx; /* opaque; owns only its device scratch workspace */

/* Not options of this build: the 64 new boundary samples (= quantiles) per refinement iteration ("the
 * number is adjustable") and the 64 uniform samples of the first iteration.  One thread solves one new sample and
 * two warps own one source; every shared-memory tile, scan and compaction of the kernels is laid out for that width, so
 * it is a compile-time constant (kThreads in csrc/twk_kernels.cuh), not a run-time field. */
typedef struct {
  int max_samples;      /* sample cap per source, default 4096; 64 <= max_samples <= 4096                  */
  int subtract_avg_tol; /* 1 = subtract the average tolerance from every interval error before sampling */
  int64_t handoff_slots; /* slots of the hand-over arena through which the first iteration (64 records, interval     */
                        /* pieces, seeds; 14,720 B per slot) of an unfinished source passes to the refinement stages */
                        /* (the first refinement iteration in a kernel of its own, all in shared memory, then the     */
                        /* 512-sample stage) instead of being recomputed there.  -1 = default min(max_sources, 524288); 0 = none.      */
                        /* Sources beyond the slots are still refined (their first iteration is recomputed).  A context */
                        /* with slots also gets 1024 carry-over slots (120 KB each) through which a source that fills */
                        /* the 512-sample refinement stage takes its whole state to the 4096-sample stage; with 0     */
                        /* (or beyond 1024 such sources per call) that stage recomputes the source from its first     */
                        /* sample.                                                                                    */
  double slope_gate;    /* slope detector: at a change of the image count between adjacent samples the    */
                        /* new real pair must be perpendicular (within 45 deg) to the neighbouring ghost pair, else    */
                        /* it is re-judged as ghosts.  Applied only when both pairs are closer than slope_gate         */
                        /* (Einstein radii; "works only for the point sources near caustics").  Default 1e-5;  */
                        /* 0 switches the detector off.  Adaptive mode only.                                           */
  double slope_cos;     /* largest |cos| of the angle between the two pairs still counted as perpendicular; default    */
                        /* cos 45 deg (reading G-4).  0 <= slope_cos <= 1.                                             */
  int point_source_test; /* 1 = before the contour integration, test whether the point-source magnification plus its   */
                        /* quadrupole (finite-source) term is accurate to rel_tol: quadrupole test + ghost-image test  */
                        /* (formulas derived in DESIGN.md, readings N1-a..c).  Sources that pass get that value  */
                        /* (status TWK_ST_POINT, out_err = relative size of the quadrupole term, out_nsamples = 0) and  */
                        /* skip the contour.  Default 0: every source takes the contour path.                           */
  int hidden_crossing_guard; /* 1 = add the hidden-crossing term to the interval error estimates: an EXTENSION of the paper's */
                        /* Eq.(17) (reading L-4), default 0.  A source boundary that dips into a caustic and  */
                        /* out again between two adjacent samples is invisible to Eq.(17); the ghost pair's separation  */
                        /* at the two samples and their neighbours predicts it, and the area it would hide is added to   */
                        /* the interval's estimate.  Changes ~1 source in 50,000 (those it is for) and no other result;   */
                        /* the kernels with the guard are separate instances and slower (config 3 of the bench: 107 M   */
                        /* instead of 147 M magnifications/s on a B200).                                                */
  int frame;            /* frame of the zeta passed in: 0 = centre of mass (the paper's, Eq.(2)); 1 = primary lens at   */
                        /* the origin (z1 = -q s/(1+q) is added to every zeta; BASELINE configs 1 and 2 are stated so)  */
} twk_options;

/* Fill *opt with the defaults above. */
void twk_default_options(twk_options* opt);

/* Create a context able to process up to max_sources sources per call on the current CUDA device.
 * opt == NULL means defaults.  Allocates the device workspace (twk_workspace_bytes) once; no allocation happens
 * inside twk_magnify / twk_images_fixed.  *ctx is set to NULL on failure. */
int twk_create(twk_ctx** ctx, const twk_options* opt, size_t max_sources);
int twk_destroy(twk_ctx* ctx);

/* Bytes of device workspace twk_create would allocate (host-side arithmetic only; needs no GPU). */
size_t twk_workspace_bytes(const twk_options* opt, size_t max_sources);

/* Adaptive mode (the hot path; BASELINE configs 2-5).
 *   s, q, rho   DEVICE double[n_models]   lens separation, mass ratio, source radius per model
 *   model_id    DEVICE int32[n_sources] or NULL; NULL means n_models == 1 (shared) or n_models == n_sources (identity)
 *   zeta        DEVICE double[n_sources][2]  source centres (re, im)
 *   rel_tol     requested relative accuracy of mu: stop when sum e_i <= rel_tol * |A|
 *   out_mu      DEVICE double[n_sources]    required
 *   out_err     DEVICE double[n_sources]    optional (NULL): estimated relative error sum e_i / |A|
 *   out_nsamples DEVICE int32[n_sources]    optional: boundary samples used
 *   out_status  DEVICE uint32[n_sources]    optional: TWK_ST_* bits
 * n_sources == 0 is a no-op returning TWK_OK. */
int twk_magnify(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho, size_t n_sources,
                const int32_t* model_id, const double* zeta, double rel_tol, double* out_mu, double* out_err,
                int32_t* out_nsamples, uint32_t* out_status, void* stream /* cudaStream_t */);

/* Light-curve front end: as twk_magnify, but the source centres are computed on the device from the
 * epochs and each model's straight-line trajectory, zeta(t) = -(tau + i u0) e^{i alpha}, tau = (t - t0) / tE (the sign
 * with which the source passes the origin on the planet's side for u0 > 0, alpha in (0, pi); centre-of-mass frame, or
 * primary at the origin with options.frame = 1).  Input traffic drops from 20 to 12 bytes per source.
 *   t0, u0, tE, alpha   DEVICE double[n_models]
 *   t                   DEVICE double[n_sources]   epochs (same unit as t0, tE)                                        */
int twk_magnify_lightcurve(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                           const double* t0, const double* u0, const double* tE, const double* alpha, size_t n_sources,
                           const int32_t* model_id, const double* t, double rel_tol, double* out_mu, double* out_err,
                           int32_t* out_nsamples, uint32_t* out_status, void* stream);

/* Light-curve front end with lens ORBITAL MOTION (contour integration is "particularly suitable
 * for modeling lens orbital motion" because every epoch may have its own lens -- nothing is precomputed per lens).  As
 * twk_magnify_lightcurve, with the lens of each epoch moved to first order in time (the paper gives no parametrisation;
 * this is the usual two-rate one):
 *     s(t) = s + ds_dt (t - t0),      alpha(t) = alpha + dalpha_dt (t - t0),
 * q, rho, u0, tE unchanged.  An epoch whose s(t) leaves (0, inf) gives NaN with TWK_ST_DOMAIN, like any invalid parameter.
 *   ds_dt, dalpha_dt    DEVICE double[n_models]   rates per unit of t (required; zeros reproduce twk_magnify_lightcurve) */
int twk_magnify_lightcurve_orbital(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                                   const double* t0, const double* u0, const double* tE, const double* alpha,
                                   const double* ds_dt, const double* dalpha_dt, size_t n_sources, const int32_t* model_id,
                                   const double* t, double rel_tol, double* out_mu, double* out_err, int32_t* out_nsamples,
                                   uint32_t* out_status, void* stream);

/* Fixed-sampling mode (BASELINE config 1 and the parity harness): theta_j = 2 pi j / N, no adaptivity.
 *   out_z       DEVICE double[n_sources][N][5][2]  optional: all five roots, CM frame, order unspecified
 *   out_kind    DEVICE int8[n_sources][N][5]       optional: 0 ghost, +1 / -1 real image of that parity
 *   out_count   DEVICE int8[n_sources][N]          optional: number of real images (3 or 5)
 *   out_mu      DEVICE double[n_sources]           optional: fixed-N area sum / (pi rho^2)
 *   out_err     DEVICE double[n_sources]           optional: fixed-N error estimate / |A|
 * N >= 4. */
int twk_images_fixed(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                     size_t n_sources, const int32_t* model_id, const double* zeta, int N, double* out_z,
                     int8_t* out_kind, int8_t* out_count, double* out_mu, double* out_err, void* stream);

/* Diagnostics for the parity harness: fixed sampling with the solver of the ADAPTIVE kernels.  As twk_images_fixed, but
 * every boundary sample is solved the way twk_magnify solves it: the point source at the
 * source centre is solved once, its five roots and their first-order response predict the roots of every boundary
 * sample, which are refined by Newton on the undeflated (monic) quintic -- four chains, the fifth root from Vieta's sum --,
 * verified by Vieta's product (and sum), recovered through Vieta's
 * formulas when two chains merge, with the cold Laguerre solver as last resort.
 *   out_diag   DEVICE uint32[4] or NULL: {point solves, Vieta recoveries, cold-solver fallbacks, lens-guard hits} */
int twk_images_fixed_seeded(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                            size_t n_sources, const int32_t* model_id, const double* zeta, int N, double* out_z,
                            int8_t* out_kind, int8_t* out_count, double* out_mu, double* out_err, uint32_t* out_diag,
                            void* stream);

/* Diagnostics for the parity harness: the sample records of the FIRST iteration (64 uniform samples theta_j = 2 pi j / 64,
 * P:318) exactly as the stage-1 kernel of twk_magnify computes them (same kernel, a dump switched on).
 *   out_records DEVICE double[n_sources][26][64]: element e of sample j of source i at [i][e][j]; per sample
 *               e = 0..4 Re z, 5..9 Im z of slots 0..4 (slots 0,1 positive-parity images, 2,3,4 negative-parity images;
 *               a sample with 3 real images keeps them in slots 0, 2, 3 and its ghost pair's positions in slots 1 and 4),
 *               10..14 Re z', 15..19 Im z', 20..24 z'^z'' (real images only), 25 = (number of real images + 8 * flags)
 *               as the raw bits of an int64.  Sources with invalid parameters are left untouched.
 *   out_diag    DEVICE uint32[4] or NULL: as above */
int twk_stage1_records(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho, size_t n_sources,
                       const int32_t* model_id, const double* zeta, double* out_records, uint32_t* out_diag, void* stream);

/* Diagnostics for the parity harness (SURVEY T-1): the Eq.(6) coefficients c0..c5 of the point source at zeta,
 * exactly as the device builder of the kernels computes them (planet frame; before the monic normalisation).
 *   out_c   DEVICE double[n_sources][6][2]  (re, im) of c0..c5.  Same batch arguments as twk_magnify (rho is not read). */
int twk_coeffs_eq6(twk_ctx* ctx, size_t n_models, const double* s, const double* q, size_t n_sources, const int32_t* model_id,
                   const double* zeta, double* out_c, void* stream);

/* End-to-end convenience with HOST buffers (same meaning as twk_magnify): copies the inputs host->device into the
 * context's staging area, runs twk_magnify on `stream`, copies the outputs device->host and synchronises the
 * stream before returning.  Optional outputs may be NULL.  A batch of 2,097,152 sources or more goes through in chunks
 * of about that size (the sources are independent): the kernels of every chunk run on `stream` in order, the
 * copies of the neighbouring chunks run beside them on two copy streams the context creates on first use (pinned host
 * buffers make them asynchronous; pageable ones work, without the overlap).  Per-source results do not depend on the
 * chunking; twk_last_stats / twk_last_stage_ms then describe the last chunk (n_launches: all of them). */
int twk_magnify_host(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                     size_t n_sources, const int32_t* model_id, const double* zeta, double rel_tol, double* out_mu,
                     double* out_err, int32_t* out_nsamples, uint32_t* out_status, void* stream);

/* The adaptive mode for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): twk_magnify without a context.  Same kernels, same arguments and results as twk_magnify on a
 * context created with default options and handoff_slots = 0 (every refinement starts again from the source's first
 * sample; results agree with the default context's within the tolerance, most of them bit for bit); all pointers DEVICE,
 * asynchronous on `stream`.  The call and everything under it calls no cudaMalloc, cudaFree or allocating library routine:
 * its workspace (counters, worklists, seed blocks, the refinement stages' record arena) is a fixed array in the library's
 * device image, TWK_STATIC_SCRATCH_BYTES per GPU, held by every GPU that loads the library until the process exits.
 *   - Limit: n_sources <= TWK_STATIC_MAX_SOURCES, else TWK_ELIMIT (nothing is launched); split larger batches or use a
 *     context.  The refinement stages run on 128 and 16 CTAs here (their record arena is what the scratch mostly is),
 *     so a batch in which most sources refine is slower than on a context.
 *   - Every call on a device shares the one array, which keeps the previous call's contents.  The call clears the work
 *     counters itself (on `stream`); everything else is written before it is read.  Calls that OVERLAP on the GPU (two
 *     streams, two host threads) race on it: keep calls on one device in stream order.
 *   - The first call on each device looks the array's device address up (cudaGetSymbolAddress, with that device current)
 *     and sets a function attribute; make that call outside a graph capture. */
#define TWK_STATIC_MAX_SOURCES 16384
#define TWK_STATIC_SCRATCH_BYTES (18u << 20) /* 18 MiB: 256 B counters + 3 x 64 KiB lists + 3.9 MiB seed blocks + 13 MiB arena */
int twk_magnify_static(size_t n_models, const double* s, const double* q, const double* rho, size_t n_sources,
                       const int32_t* model_id, const double* zeta, double rel_tol, double* out_mu, double* out_err,
                       int32_t* out_nsamples, uint32_t* out_status, void* stream);

/* Diagnostics of the last twk_magnify on this context (synchronises `stream`): number of sources the first iteration
 * left unfinished (*n_stage2: the worklist of the refinement stages 1.5 and 2), number that filled the 512-sample stage
 * and went on to the last one (*n_stage3), and the number of kernels the call launched (5 with hand-over slots: centre
 * solves, first iteration, first refinement iteration in shared memory, 512-sample stage, max_samples stage; 4 without:
 * the third is then not launched).  Any pointer may be NULL. */
int twk_last_stats(twk_ctx* ctx, int64_t* n_stage2, int64_t* n_stage3, int* n_launches, void* stream);

/* Per-stage device timing of twk_magnify for measurement: when enabled, CUDA events are recorded on the call's
 * stream around each stage.  twk_last_stage_ms waits for the last recorded event and writes the durations (ms)
 * of {stage-0 (centre solves), stage-1, stage-1.5 + stage-2, stage-3 kernel} of the last twk_magnify on this context
 * (0 for absent stages) into ms4[4]. */
int twk_enable_stage_timing(twk_ctx* ctx, int on);
int twk_last_stage_ms(twk_ctx* ctx, float* ms4);

/* FP64 FMA throughput probe used for the ALU roofline denominator: runs `iters` dependent-chain DFMAs per thread
 * (8 independent chains per thread, a full persistent grid) and returns the measured TFLOP/s (2 flop per DFMA) in
 * *out_tflops.  Synchronous. */
int twk_fp64_peak_probe(int iters, double* out_tflops);

/* Debug build only (libtwk_debug.so, compiled with -DTWK_DEBUG; twk_version() says so): the kernels count violations of
 * their own invariants instead of trapping -- out12 (12 values, caller-owned host memory) = {record id out of range, sample
 * angles not strictly increasing, sorted list not a permutation of the sample ids, two writers to one record in one
 * re-judging phase, worklist / hand-over slot out of range, new angle outside its interval, sources checked, iterations
 * checked, and four event counts of stage 1.5: entries taken up, entries whose new samples were solved, sources finished
 * there, entries passed on unread}.  Synchronises the device;
 * reset != 0 clears the counters.  Returns TWK_EINVAL in the release build.  Stands in for compute-sanitizer, which this
 * pool does not offer. */
int twk_debug_counters(uint32_t* out12, int reset);

const char* twk_strerror(int code);
const char* twk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TWK_H_ */
