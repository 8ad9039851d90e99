/* galario_b200.h — C ABI of the B200-native GALARIO hot path (arXiv:1709.06999).
 *
 * What the library computes (citations are lines of the paper text, PAPER.md):
 *   model image (or radial profile swept into an inclined image)
 *     -> centre shift + 2-D real-to-complex FFT + shift along v
 *     -> rotation of the (u, v) points by PA                                (Eq. 11-12)
 *     -> bilinear interpolation of the half-plane spectrum
 *     -> phase ramp for (dRA, dDec)
 *     -> weighted chi-square against observed visibilities                  (Eq. 10, 718)
 * The executable definition followed is the paper's Appendix D listing;
 * the readings taken where it is silent or garbled are listed in DESIGN.md (A1..A20).
 *
 * Conventions
 *   - Every array pointer is a DEVICE pointer unless the function name ends in `_host_*`, in which case
 *     every array pointer is a HOST pointer (pinned or pageable) and the call copies in, computes, copies
 *     the result out and synchronises the stream before returning (the paper's own calling convention:
 *     inputs start in host memory).
 *   - The caller owns every buffer.  Inputs are const and never modified.  The plan owns its twiddle
 *     tables, the half-plane spectrum workspace, the reduction scratch and (for `_host_` calls) its
 *     device staging buffers.
 *   - Device-pointer calls are asynchronous on `stream` (a cudaStream_t passed as void*, NULL = the
 *     legacy default stream), never synchronise the host, and leave their results in device memory.
 *   - A plan is bound to one device and is not safe for concurrent use from several streams/threads.
 *   - Suffix _f64 / _f32 = storage and FFT precision of every array.  In _f32 the index and phase
 *     arithmetic of the sampling stage is still carried in double (reading A14).
 *   - Units: dxy, dRA, dDec, Rmin, dR, inc, PA in radians; u, v in wavelengths; images in Jy/pixel;
 *     profiles in Jy/sr.  dRA > 0 moves the source East, dDec > 0 North, PA is
 *     measured East of North.
 *   - Image layout: row-major [nxy][nxy], row 0 = North, column 0 = East, origin at pixel
 *     [nxy/2][nxy/2].  nxy must be a power of two in [8, 16384] (the paper's range).
 *   - Alignment: images must be 16-byte aligned, visibility / spectrum outputs aligned to one complex value (16 bytes
 *     in _f64, 8 in _f32) — the kernels move them as complex pairs and bulk copies; anything else returns
 *     GAL_ERR_INVALID_ARGUMENT (allocations always qualify; a sub-view at an odd element offset does not).  The
 *     per-point arrays u, v, re_obs, im_obs, w may have any alignment (16-byte aligned ones take the TMA path).
 *   - Visibilities out: complex interleaved (re, im), 2*M reals.  Observations in:
 *     separate re_obs[M], im_obs[M], w[M].
 *   - (u, v) points whose interpolation cell leaves the half-plane grid are NOT clamped: the spectrum is
 *     extended to the whole plane by its own periodicity and Hermitian symmetry (reading A6); the number
 *     of such points in the last call is available from gal_last_oob_count().
 *   - Return value: 0 = GAL_OK, negative = error (see below).  No exception crosses this boundary.
 *     M == 0 is valid: chi2 = 0, nothing written to vis_out.
 */
#ifndef GALARIO_B200_H
#define GALARIO_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GAL_OK 0
#define GAL_ERR_INVALID_ARGUMENT (-1) /* null pointer, bad nxy, M < 0, nr < 2, dR <= 0, dxy <= 0, |inc| >= pi/2, C > plan batch, wrong precision */
#define GAL_ERR_ALLOC (-2)            /* device or host allocation failed */
#define GAL_ERR_CUDA (-3)             /* a CUDA call failed; see gal_last_cuda_error() */
#define GAL_ERR_UNSUPPORTED (-4)      /* a power-of-two nxy above 16384; M >= 2^32 in gal_plan_bind_obs */
#define GAL_ERR_BINDING_VIOLATED (-5) /* an earlier call found a bound (u, v) set changed: that call's results are invalid; the binding is dropped */
#define GAL_ERR_TOO_LARGE (-6)        /* gal_chi2_profile_hankel_noalloc_f64 only: M > GAL_NOALLOC_MAX_POINTS, its fixed scratch cannot hold the partial sums */

typedef struct gal_plan gal_plan;

/* Create a plan for images of nxy x nxy pixels, up to `batch` images per call (1 for everything but
 * the batched cube), precision_bits = 64 or 32, on CUDA device `device`.  Allocates the twiddle table
 * and the workspace (3 * batch * nxy * (nxy/2+1) complex numbers: the row-transformed image and the spectrum
 * as column pairs, plus reduction scratch). */
int gal_plan_create(gal_plan** out, int nxy, int batch, int precision_bits, int device);
int gal_plan_destroy(gal_plan* plan);
/* Bytes of device memory the plan owns (workspace + tables + staging). */
size_t gal_plan_workspace_bytes(const gal_plan* plan);
/* Points of the most recent sample/chi2 call that fell outside the half-plane grid (synchronises the
 * stream of that call).  Returns -1 on error. */
int64_t gal_last_oob_count(gal_plan* plan);
/* cudaError_t of the most recent failing CUDA call made through this plan (0 if none). */
int gal_last_cuda_error(const gal_plan* plan);
const char* gal_strerror(int code);
/* Number of kernels the plan has launched since it was created (for launch accounting). */
int64_t gal_plan_launch_count(const gal_plan* plan);

/* Pruned transform (not in the paper, changes no result).  The bilinear gather only
 * reads the part of the half plane the (u, v) set reaches (Eq. 19 of the paper, keeps it
 * inside a quarter of the grid).  With pruning on, a call first reduces the point set to its extent
 * {largest column ku, first and last shifted row kvs} with the sampler's own index arithmetic, and the FFT
 * passes neither form nor write what lies outside it.  mode 0 = never, 1 = automatic (default: prune when
 * re-reading u and v costs less than a quarter of the three spectrum passes it can save), 2 = always.
 * A point whose cell leaves the grid (reading A6) makes the extent the whole half plane.
 * In mode 1, image calls at nxy = 2048 / 4096 on 16-byte aligned arrays of 32 MB of (u, v) or more do not run the
 * uv-extent kernel from the second call on: the transform is pruned to the extent the call before derived from the
 * largest baseline length of ITS points (valid for any PA), the sampling kernel verifies every point of this call
 * against it, and if a point lies outside, the call repeats itself on the device on the extent of its own points
 * (one conditional kernel, no host synchronisation).  Results do not depend on this: a repeated call may differ
 * from an unrepeated one in the last bits of the transform only.  Mode 2 always computes the exact extent. */
int gal_plan_set_pruning(gal_plan* plan, int mode);
/* Tuning options of a plan.  The library reads NO environment variable; these are the only switches.  They choose
 * among kernel forms and launch geometries that compute the same thing (results agree bit for bit, except where a
 * different row-pass kernel is selected: last bits of the transform), and their defaults are the measured optimum
 * on B200 — they exist for measurements and for tests that must reach a particular kernel at a small size.
 * Takes effect from the next call.  GAL_ERR_INVALID_ARGUMENT for an unknown option or a value out of range. */
#define GAL_OPT_ROW_MODE 1        /* nxy 1024..4096: -1 per-size default, 0 plain row pass, 1 register untangle with plain loads, 2 its persistent TMA-ring form, 3 one row per CTA */
#define GAL_OPT_BATCH_CHUNK 2     /* channels per chunk of a batched call; 0 (default) = all in one chunk */
#define GAL_OPT_SPECULATE 3       /* 1 (default) = speculative extent in pruning mode 1 (see above); 0 = always run the uv-extent kernel */
#define GAL_OPT_SPEC_MIN_BYTES 4  /* smallest volume of (u, v), in bytes, the speculative extent is used for (default 32e6) */
#define GAL_OPT_BATCH_CONC 5      /* channels in flight in the batched sampler (default 12) */
#define GAL_OPT_ROW_PREFETCH 6    /* scale of the L2 prefetch distance of the FFT passes (default 1; 0 = no prefetch) */
#define GAL_OPT_ROW_X2_ONE_CTA 7  /* nxy = 16384: 1 = one CTA per row instead of a cluster of two (default 0) */
int gal_plan_set_option(gal_plan* plan, int option, double value);
/* extent[3] (host) = {kumax, kvs_min, kvs_max} used by the most recent sample/chi2 call (the whole half plane
 * {nxy/2, 0, nxy-1} if that call did not prune).  Synchronises the stream of that call. */
int gal_last_uv_extent(gal_plan* plan, int* extent);

/* Bound uv set (not in the paper; the use it serves is the paper's own: one observation, many model evaluations,
 * PAPER.md:39-49).  gal_plan_bind_uv declares that the C x M device arrays u and v will keep their contents
 * until the binding is replaced or removed.  It reduces them once to their largest baseline length r_max
 * (one kernel, synchronises `stream`).  Later sample/chi2 calls that pass the same u, v, M (and C) skip the
 * per-call uv-extent kernel: rotation by any PA leaves abs(u'), abs(v') <= r_max, so the extent is the square
 * of half-width r_max / du + 2 cells about the centre, a few per cent larger than the exact one; results are
 * bit-identical.  The sampler verifies every point against that extent: gal_last_extent_violations() returns
 * the number of points of the most recent call that fell outside (0 unless the promise was broken, in which
 * case that call's results are invalid).  Pruning mode 0 ignores the binding.  The first call on a binding, and
 * the first with a new dxy, synchronise the stream once (the extent is uploaded); all later calls are
 * asynchronous as usual. */
int gal_plan_bind_uv_f64(gal_plan* plan, const double* u, const double* v, int64_t M, int C, void* stream);
int gal_plan_bind_uv_f32(gal_plan* plan, const float* u, const float* v, int64_t M, int C, void* stream);
int gal_plan_unbind_uv(gal_plan* plan);
int64_t gal_last_extent_violations(gal_plan* plan);

/* Bound observation set (same use case: the observations of a fit never change).  gal_plan_bind_obs declares that
 * the C x M device arrays u, v, re_obs, im_obs, w keep their contents.  The plan makes a PRIVATE copy of the five
 * arrays reordered along a space-filling (Morton) curve of the uv plane folded to u >= 0, so that the 32 points of
 * a warp fall into a few neighbouring cells of the spectrum for any PA and the bilinear gather
 * is served from L1 instead of L2 (hand-written stable radix sort, a few kernels, synchronises `stream`; the copy
 * costs 5 C M reals of device memory).  It also binds (u, v) as gal_plan_bind_uv does.  Later chi2* calls
 * (gal_chi2_image_*, gal_chi2_profile_*, gal_chi2_image_batch_*) that pass these very five pointers with the same M
 * and C sample the private copy and skip the uv-extent kernel: chi2 is a sum over the points (Eq. 10)
 * and does not depend on their order beyond rounding (the reduction stays deterministic: the permutation is the
 * unique order by (Morton key, original index)).  Changing the contents of the arrays afterwards has NO effect on
 * those calls until the set is bound again.  sample* calls and chi2 calls with other observation pointers use the
 * (u, v) binding only.  gal_plan_unbind_obs (= gal_plan_unbind_uv) drops both.
 * Sticky error: a sample/chi2 call on a bound (u, v) set whose points left the bound extent (the promise was broken)
 * sets a flag; the next sample/chi2 call on the plan after that call has finished returns
 * GAL_ERR_BINDING_VIOLATED without launching anything and drops the binding.  Results of the offending call are
 * undefined.  Errors: as gal_plan_bind_uv; GAL_ERR_UNSUPPORTED for M >= 2^32. */
int gal_plan_bind_obs_f64(gal_plan* plan, const double* u, const double* v, const double* re_obs, const double* im_obs,
                          const double* w, int64_t M, int C, void* stream);
int gal_plan_bind_obs_f32(gal_plan* plan, const float* u, const float* v, const float* re_obs, const float* im_obs,
                          const float* w, int64_t M, int C, void* stream);
int gal_plan_unbind_obs(gal_plan* plan);

/* ---- get_image_size (Eq. 19-24; host only, no device is touched): image size N_lm (rounded
 *      up to a power of two) and pixel size (radians) for the uv coverage u[M], v[M] (HOST pointers,
 *      wavelengths).  With q_min / q_max the shortest / longest baseline sqrt(u^2 + v^2):
 *        PB <= 0 (criterion iia): duv = q_min / (Gamma f_min) (Eq. 21, Gamma = 0.6 as for ALMA) and
 *                 N = 2 f_max q_max / duv (Eq. 19; Eq. 22 as printed drops f_max, Table 1 is only reproduced
 *                 with it);
 *        PB  > 0 (criterion iib): the field of view is the primary beam, duv = 1 / PB (Eq. 23), N as above.
 *      dxy = 1 / (N duv) (Eq. 16).  The paper's Table 1 uses f_min = 5, f_max = 2.5 (pass <= 0 for these defaults).
 *      Errors: GAL_ERR_INVALID_ARGUMENT for null pointers, M < 1, a zero or non-finite baseline. ---- */
int gal_get_image_size(const double* u, const double* v, int64_t M, double PB, double f_min, double f_max,
                       int* nxy_out, double* dxy_out);

/* Diagnostic per-kernel timing.  After gal_plan_timing_enable(plan, n) the next n sample/chi2 calls record a
 * CUDA event on their stream before the first kernel, between the kernels and after the sampling kernel
 * (n = 0 switches it off and frees the events).  gal_plan_timing_read synchronises those events and returns
 * the average duration in milliseconds of the uv-extent kernel (0 when the call did not prune), the row
 * pass, the column pass and the sampling kernel (ms_per_kernel[4]) over the calls recorded so far (*calls,
 * may be null). */
int gal_plan_timing_enable(gal_plan* plan, int max_calls);
int gal_plan_timing_read(gal_plan* plan, double* ms_per_kernel, int64_t* calls);

/* ---- sweep: image_out[nxy][nxy] = dxy^2 * lerp(I, (r - Rmin)/dR),
 *      r = sqrt((x/cos inc)^2 + y^2), 0 outside [Rmin, Rmin + (nr-1) dR]. ---- */
int gal_sweep_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, double dxy, double inc,
                  double* image_out, void* stream);
int gal_sweep_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, double dxy, double inc,
                  float* image_out, void* stream);

/* ---- the transform alone: spectrum_out[nxy][nxy/2+1] complex interleaved =
 *      fftshift(rfft2(fftshift(image)), axes=0), in the paper's layout (for tests and inspection;
 *      the sampling calls use an internal u-major copy and never materialise this one). ---- */
int gal_fft2_shifted_f64(gal_plan* plan, const double* image, double* spectrum_out, void* stream);
int gal_fft2_shifted_f32(gal_plan* plan, const float* image, float* spectrum_out, void* stream);

/* ---- sampleImage: vis_out[2M]. ---- */
int gal_sample_image_f64(gal_plan* plan, const double* image, double dxy, const double* u, const double* v,
                         int64_t M, double dRA, double dDec, double PA, double* vis_out, void* stream);
int gal_sample_image_f32(gal_plan* plan, const float* image, double dxy, const float* u, const float* v,
                         int64_t M, double dRA, double dDec, double PA, float* vis_out, void* stream);

/* ---- chi2Image: chi2_out[1] (device, always double). ---- */
int gal_chi2_image_f64(gal_plan* plan, const double* image, double dxy, const double* u, const double* v,
                       const double* re_obs, const double* im_obs, const double* w, int64_t M, double dRA,
                       double dDec, double PA, double* chi2_out, void* stream);
int gal_chi2_image_f32(gal_plan* plan, const float* image, double dxy, const float* u, const float* v,
                       const float* re_obs, const float* im_obs, const float* w, int64_t M, double dRA,
                       double dDec, double PA, double* chi2_out, void* stream);

/* ---- sampleProfile / chi2Profile: the image is swept from the profile
 *      inside the first FFT pass and never written to memory; nxy comes from the plan. ---- */
int gal_sample_profile_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, double dxy,
                           const double* u, const double* v, int64_t M, double dRA, double dDec, double PA,
                           double inc, double* vis_out, void* stream);
int gal_sample_profile_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, double dxy,
                           const float* u, const float* v, int64_t M, double dRA, double dDec, double PA,
                           double inc, float* vis_out, void* stream);
int gal_chi2_profile_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, double dxy,
                         const double* u, const double* v, const double* re_obs, const double* im_obs,
                         const double* w, int64_t M, double dRA, double dDec, double PA, double inc,
                         double* chi2_out, void* stream);
int gal_chi2_profile_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, double dxy,
                         const float* u, const float* v, const float* re_obs, const float* im_obs,
                         const float* w, int64_t M, double dRA, double dDec, double PA, double inc,
                         double* chi2_out, void* stream);

/* ---- sampleProfile / chi2Profile by the DIRECT HANKEL TRANSFORM of the profile (Eq. 25:
 *      V(rho) = 2 pi int I(r) J0(2 pi rho r) r dr, the analytic result the paper validates sampleProfile against,
 *      PAPER.md:370-404).  An alternative evaluation for axisymmetric models: no image, no
 *      FFT, no interpolation error; cost O(M nr).  Composite trapezoid rule on the profile grid R_k = Rmin + k dR
 *      (profile zero outside, as in the sweep); inclination as in the sweep (East-West axis
 *      stretched by 1/cos inc): V = cos(inc) V(rho), rho = sqrt((u' cos inc)^2 + v'^2) with (u', v')
 *      rotated by PA; phase exp(+2 pi i (u dRA + v dDec)).  There is no dxy and no nxy: the plan only lends its
 *      reduction scratch.  Agrees with gal_sample_profile_* to the FFT route's own accuracy (1e-5 of the peak at
 *      the nodes of the uv grid; the bilinear interpolation error elsewhere).  Arguments as gal_sample_profile_* /
 *      gal_chi2_profile_* without dxy. ---- */
int gal_sample_profile_hankel_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, const double* u,
                                  const double* v, int64_t M, double dRA, double dDec, double PA, double inc,
                                  double* vis_out, void* stream);
int gal_sample_profile_hankel_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, const float* u,
                                  const float* v, int64_t M, double dRA, double dDec, double PA, double inc,
                                  float* vis_out, void* stream);
int gal_chi2_profile_hankel_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, const double* u,
                                const double* v, const double* re_obs, const double* im_obs, const double* w,
                                int64_t M, double dRA, double dDec, double PA, double inc, double* chi2_out,
                                void* stream);
int gal_chi2_profile_hankel_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, const float* u,
                                const float* v, const float* re_obs, const float* im_obs, const float* w,
                                int64_t M, double dRA, double dDec, double PA, double inc, double* chi2_out,
                                void* stream);

/* ---- batched spectral cube (not in the paper; motivated at PAPER.md:45; reading A17):
 *      C <= plan batch independent chi2Image problems sharing (nxy, dxy, dRA, dDec, PA, M).
 *      images [C][nxy][nxy]; u, v, re_obs, im_obs, w each [C][M]; chi2_per_channel[C] and
 *      chi2_total[1] (device, double; the total is summed in channel order). ---- */
int gal_chi2_image_batch_f64(gal_plan* plan, const double* images, int C, double dxy, const double* u,
                             const double* v, const double* re_obs, const double* im_obs, const double* w,
                             int64_t M, double dRA, double dDec, double PA, double* chi2_per_channel,
                             double* chi2_total, void* stream);
int gal_chi2_image_batch_f32(gal_plan* plan, const float* images, int C, double dxy, const float* u,
                             const float* v, const float* re_obs, const float* im_obs, const float* w,
                             int64_t M, double dRA, double dDec, double PA, double* chi2_per_channel,
                             double* chi2_total, void* stream);

/* ---- K observation sets against ONE model image in one call ("fit simultaneously several observations";
 *      PAPER.md:212, second alternative): chi2_per_set[k] = chi2Image(image; set k), for
 *      K <= plan batch sets of M points each sharing (dxy, dRA, dDec, PA).  ONE transform of the image — pruned, when
 *      pruning is on, to the union of the sets' uv extents — then one sampling launch whose grid.y runs over the sets,
 *      all reading the one spectrum: K sets cost one FFT + K samplings, not K calls.  image [nxy][nxy]; u, v, re_obs,
 *      im_obs, w each [K][M] (device); chi2_per_set[K] and chi2_total[1] (device, double; chi2_total may be NULL; it
 *      is the sum in set order).  K is limited by the plan's batch because the reduction scratch is sized by it (the
 *      plan's spectrum workspace for batch > 1 is not used by this call).  Sets of different lengths: pad the
 *      shorter ones with points of weight 0 at u = v = 0.  gal_last_oob_count() is summed over the sets. ---- */
int gal_chi2_image_sets_f64(gal_plan* plan, const double* image, int K, double dxy, const double* u, const double* v,
                            const double* re_obs, const double* im_obs, const double* w, int64_t M, double dRA,
                            double dDec, double PA, double* chi2_per_set, double* chi2_total, void* stream);
int gal_chi2_image_sets_f32(gal_plan* plan, const float* image, int K, double dxy, const float* u, const float* v,
                            const float* re_obs, const float* im_obs, const float* w, int64_t M, double dRA,
                            double dDec, double PA, double* chi2_per_set, double* chi2_total, void* stream);

/* ---- multi-source composition ("summing up the visibilities of each single source ... applying a
 *      different complex phase"): one model image placed S times,
 *        V(u, v) = sum_s scale[s] * sampleImage(image; dRA[s], dDec[s], PA[s])(u, v),
 *      with ONE transform of the image.  dRA, dDec, PA, scale are HOST arrays of S doubles (scale may be NULL:
 *      all 1); every other array is a device array as in the single-source calls.  chi2 compares the summed
 *      visibilities with the observations.  gal_last_oob_count() is summed over the sources. ---- */
int gal_sample_image_multi_f64(gal_plan* plan, const double* image, double dxy, const double* u, const double* v,
                               int64_t M, int S, const double* dRA, const double* dDec, const double* PA,
                               const double* scale, double* vis_out, void* stream);
int gal_sample_image_multi_f32(gal_plan* plan, const float* image, double dxy, const float* u, const float* v,
                               int64_t M, int S, const double* dRA, const double* dDec, const double* PA,
                               const double* scale, float* vis_out, void* stream);
int gal_chi2_image_multi_f64(gal_plan* plan, const double* image, double dxy, const double* u, const double* v,
                             const double* re_obs, const double* im_obs, const double* w, int64_t M, int S,
                             const double* dRA, const double* dDec, const double* PA, const double* scale,
                             double* chi2_out, void* stream);
int gal_chi2_image_multi_f32(gal_plan* plan, const float* image, double dxy, const float* u, const float* v,
                             const float* re_obs, const float* im_obs, const float* w, int64_t M, int S,
                             const double* dRA, const double* dDec, const double* PA, const double* scale,
                             double* chi2_out, void* stream);

/* ---- HOST-pointer entry points (the paper's calling convention): every array is in
 *      host memory; the call stages it through plan-owned device buffers on `stream`, runs the same
 *      kernels, copies the result back and synchronises `stream`.  chi2_out / vis_out are host. ---- */
int gal_chi2_image_host_f64(gal_plan* plan, const double* image, double dxy, const double* u, const double* v,
                            const double* re_obs, const double* im_obs, const double* w, int64_t M, double dRA,
                            double dDec, double PA, double* chi2_out, void* stream);
int gal_chi2_image_host_f32(gal_plan* plan, const float* image, double dxy, const float* u, const float* v,
                            const float* re_obs, const float* im_obs, const float* w, int64_t M, double dRA,
                            double dDec, double PA, double* chi2_out, void* stream);
int gal_sample_image_host_f64(gal_plan* plan, const double* image, double dxy, const double* u, const double* v,
                              int64_t M, double dRA, double dDec, double PA, double* vis_out, void* stream);
int gal_sample_image_host_f32(gal_plan* plan, const float* image, double dxy, const float* u, const float* v,
                              int64_t M, double dRA, double dDec, double PA, float* vis_out, void* stream);
int gal_chi2_profile_host_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, double dxy,
                              const double* u, const double* v, const double* re_obs, const double* im_obs,
                              const double* w, int64_t M, double dRA, double dDec, double PA, double inc,
                              double* chi2_out, void* stream);
int gal_chi2_profile_host_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, double dxy,
                              const float* u, const float* v, const float* re_obs, const float* im_obs,
                              const float* w, int64_t M, double dRA, double dDec, double PA, double inc,
                              double* chi2_out, void* stream);
int gal_sample_profile_host_f64(gal_plan* plan, const double* I, int nr, double Rmin, double dR, double dxy,
                                const double* u, const double* v, int64_t M, double dRA, double dDec, double PA,
                                double inc, double* vis_out, void* stream);
int gal_sample_profile_host_f32(gal_plan* plan, const float* I, int nr, double Rmin, double dR, double dxy,
                                const float* u, const float* v, int64_t M, double dRA, double dDec, double PA,
                                double inc, float* vis_out, void* stream);

/* ---- measurement helper (not part of the method): the FP64 fused-multiply-add rate of `device`, measured with
 *      independent DFMA chains on every SM (a few launches of a few ms each, CUDA-event timed, best of five;
 *      synchronises the device; allocates and frees 8 bytes).  *tflops_out = 2 flop x DFMA/s / 1e12 (host);
 *      ms_out (host, may be NULL) = duration of the best launch.  bench.py divides the FP64 instruction rate of each
 *      kernel by this to report an ALU fraction beside the HBM fraction. ---- */
int gal_measure_fp64_fma_peak(int device, double* tflops_out, double* ms_out);

/* ---- chi2Profile WITHOUT A PLAN AND WITHOUT ANY ALLOCATION (direct Hankel transform, Eq. 25 and Eq. 10:
 *      PAPER.md:366-368, 194-198, 718; same mathematics and same arguments as gal_chi2_profile_hankel_f64).
 *
 *      Why it exists.  Every other call needs a gal_plan, and gal_plan_create takes its workspace with cudaMalloc.
 *      That rules the library out for two kinds of caller: (1) code that runs inside a fixed device-memory budget —
 *      an application that partitions the GPU once at start-up and hands each component its slice, a memory-capped
 *      MPS client, a GPU already filled by the rest of the fit — where one more cudaMalloc fails or eats memory
 *      promised to somebody else; (2) latency-critical loops, because cudaMalloc / cudaFree synchronise the whole
 *      device and serialise on the driver's allocator lock.  This entry point never calls cudaMalloc, cudaFree,
 *      cudaMallocAsync or an allocating library routine, at set-up or later.
 *
 *      How.  Its reduction scratch (one double per CTA of 128 points, one ticket counter) is a file-scope
 *      `static __device__` array of gal_noalloc_scratch_bytes() = 65 792 bytes (64 KiB + 256 B), part of the
 *      library image: every GPU that loads the library holds it until the process exits, whether this call is
 *      used or not.  The array's size fixes the limit: M <= GAL_NOALLOC_MAX_POINTS (1 048 576 = 8192 CTAs x 128
 *      points); a larger M returns GAL_ERR_TOO_LARGE and launches nothing (split the set — chi2 is a sum over
 *      points — or use a plan).  nr is not limited.
 *
 *      Arguments.  `device`: the CUDA device the pointers live on (0 <= device < 64); it is made current for
 *      the duration of the call and the previous device restored.  I[nr], u, v, re_obs, im_obs, w [M]: DEVICE
 *      arrays of doubles, owned by the caller, never modified, any alignment.  chi2_out: DEVICE double[1].
 *      `stream`: cudaStream_t as void* (NULL = legacy default stream); the call is asynchronous on it and never
 *      synchronises the host.  M == 0 is valid (chi2 = 0).  Errors: GAL_ERR_INVALID_ARGUMENT as for
 *      gal_chi2_profile_hankel_f64 (null pointer, nr < 2, dR <= 0, |inc| >= pi/2, M < 0, non-finite scalars, bad
 *      device); GAL_ERR_TOO_LARGE; GAL_ERR_CUDA with the cudaError_t in gal_noalloc_last_cuda_error().
 *
 *      First call on a device.  It looks up the device address of the scratch array (cudaGetSymbolAddress, once
 *      per device, cached) and thereby loads this library's device code on that GPU.  Make one call — M = 1 will
 *      do — during start-up, before any stream capture begins and before the time-critical part of the program.
 *
 *      Shared state.  All calls on one GPU use the same array.  The ticket is zeroed on `stream` in front of every
 *      launch and every partial sum is written before it is read, so nothing leaks from one call into the next;
 *      the array simply keeps the last call's partial sums.  Calls that may OVERLAP on the same GPU (two streams,
 *      two threads) race on it and return wrong sums: keep them on one stream or order them with events.
 *
 *      Result.  Per-point arithmetic identical to gal_chi2_profile_hankel_f64; the sum runs over fixed 128-point
 *      tiles in tile order, so the value is bit-reproducible from run to run and across GPU models, and agrees
 *      with the plan-based call to rounding (a few ulp; the tests allow 1e-12 relative). ---- */
#define GAL_NOALLOC_MAX_POINTS 1048576
int gal_chi2_profile_hankel_noalloc_f64(int device, const double* I, int nr, double Rmin, double dR, const double* u,
                                        const double* v, const double* re_obs, const double* im_obs, const double* w,
                                        int64_t M, double dRA, double dDec, double PA, double inc, double* chi2_out,
                                        void* stream);
/* Bytes of the static scratch array each GPU holds for the call above (65 792). */
size_t gal_noalloc_scratch_bytes(void);
/* cudaError_t of the most recent failing CUDA call made by gal_chi2_profile_hankel_noalloc_f64 (0 if none). */
int gal_noalloc_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GALARIO_B200_H */
