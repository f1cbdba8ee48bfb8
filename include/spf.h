/*
 * spf.h -- C ABI of libspf: the M-TIP slicing + orientation-matching hot path on one B200.
 *
 * What the calls compute is fixed by the paper's problem statement (arxiv 2109.05339,
 * /root/reference/PAPER.md; citations "PAPER.md:<line>"), the call names by
 * BASELINE.json:north_star, and everything the paper leaves open by the readings in
 * DESIGN.md ("Readings", s1..s15 of SURVEY.md section 8(c)).
 *
 *   spf_prepare_model  -- once per model update: deapodise, zero-pad to the upsampled grid,
 *                         3-D FFT (steps a1-a2 of a type-2 NUFFT, refs [8],[15]).
 *   spf_slice          -- M model images: rotate the detector pixels' q-vectors by each
 *                         reference orientation and interpolate the upsampled grid there with
 *                         the exponential-of-semicircle kernel (steps a3-a5).
 *   spf_match          -- every image against every model image by squared Euclidean distance,
 *                         argmin orientation per image (steps a6-a8).
 *   spf_orientation_match_host -- the same three steps behind HOST buffers (what a user with
 *                         NumPy arrays calls; bench.py's end-to-end number).
 *
 * Conventions
 *   - Pointers marked [dev] are DEVICE pointers owned by the caller (allocate them with
 *     PyTorch or cudaMalloc); [host] are host pointers.  Inputs are never modified, outputs are
 *     fully overwritten.  The library owns only what lives inside its context (the fine grid,
 *     deapodisation tables, cuFFT plan, tensor maps).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *     calls enqueue on it and return without synchronising, except where stated.
 *   - Return value: SPF_OK (0) or a negative spf_status; spf_last_error() gives the text (for
 *     SPF_ECUDA the CUDA error string).  No exception or abort crosses the ABI.
 *   - There is no CPU fallback: without a CUDA device every call except spf_version /
 *     spf_status_string / spf_plan_* fails with SPF_ECUDA.
 *   - Layouts are C-order (last index fastest).  Model axes (x,y,z) = (i1,i2,i3); voxel
 *     [i1][i2][i3] sits at integer position n = (i1,i2,i3) - floor(N/2)   (reading s1/s13).
 *   - Quaternions are (w,x,y,z), Hamilton, active: x = R(quat) q; they are normalised inside
 *     (reading s2).  q and -q give the same slice.
 *   - Pixel q-vectors are in radians per voxel, |component| <= pi (values outside are folded
 *     by 2 pi, the transform being 2 pi-periodic)   (reading s4).
 */
#ifndef SPF_H_
#define SPF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define SPF_API __attribute__((visibility("default")))
#else
#define SPF_API
#endif

typedef enum {
    SPF_OK = 0,
    SPF_EINVAL = -1, /* bad size, null pointer, unsupported parameter (checked on host-side arguments only) */
    SPF_ENOMEM = -2, /* host or device allocation failed */
    SPF_ECUDA = -3,  /* a CUDA / cuFFT / driver call failed; text in spf_last_error */
    SPF_ESTATE = -4, /* call order: spf_slice before spf_prepare_model */
    SPF_EFAULT = -5  /* a kernel's pipeline watchdog gave up (see spf_check_fault); results of that call are invalid */
} spf_status;

typedef struct spf_ctx spf_ctx; /* opaque */

typedef struct {
    int32_t n;        /* model edge N >= 2 (odd or even) */
    double eps;       /* NUFFT tolerance in (0, 1e-1]; sets the kernel width w = min(ceil(log10(1/eps)) + 2, 10): 8 at 1e-6 (reading s10b) */
    double upsampfac; /* sigma >= 2.0 (the kernel constants are those of sigma = 2)        (reading s10) */
    int32_t n_fine;   /* 0: smallest even 2-3-5-7-smooth integer >= upsampfac * n; else an explicit fine-grid edge >= 2n */
    int32_t device;   /* CUDA device ordinal */
} spf_params;

typedef struct {
    int32_t n, n_fine, w;   /* model edge, fine-grid edge actually used, kernel width in fine cells */
    double beta;            /* exponential-of-semicircle shape parameter, 2.30 * w */
    int32_t n_padded;       /* edge of the stored, centred fine grid including its periodic halo */
    int32_t grid_is_real;   /* 1 after spf_prepare_model saw a real EVEN model (fine grid real; fp32 grid is gathered) */
    int32_t prepared;       /* 1 once spf_prepare_model has run */
    int32_t sm_count;       /* multiprocessors of the device */
} spf_info;

SPF_API const char *spf_version(void);
SPF_API const char *spf_status_string(int status);

/* Host-only planning helpers (no device needed): kernel width for eps, default fine-grid edge. */
SPF_API int32_t spf_plan_kernel_width(double eps);
SPF_API int32_t spf_plan_n_fine(int32_t n, double upsampfac);

/*
 * Create a context on p->device: allocates the fine grids (n_padded^3 complex64 + fp32),
 * plans cuFFT, computes the deapodisation factors p(n) = 2 / (w phihat(pi w n / n_fine)) on the
 * host in fp64 by Gauss-Legendre quadrature.  Synchronises the device.  *out = NULL on error
 * (then spf_last_error(NULL) holds the text).
 */
SPF_API int spf_create(spf_ctx **out, const spf_params *p);
SPF_API void spf_destroy(spf_ctx *ctx);
SPF_API int spf_get_info(const spf_ctx *ctx, spf_info *out);
SPF_API const char *spf_last_error(const spf_ctx *ctx); /* ctx may be NULL: error of the last failed spf_create */

/*
 * Optional layout promise that lets spf_slice bin points without a sort: the pixel array given
 * to spf_slice is [n_panels][rows][cols][3], each panel a regular lattice (PAPER.md:124:
 * "128 x 128 pixels").  Thread blocks then take compact lattice patches whose fine-grid
 * bounding box is staged in shared memory.  Without the promise (n_panels = 0) blocks take
 * runs of consecutive pixels: same results, lower locality.  Host-only state; returns EINVAL
 * for non-positive sizes.
 */
SPF_API int spf_set_detector_layout(spf_ctx *ctx, int32_t n_panels, int32_t rows, int32_t cols);

/*
 * Steps a1-a2.  model [dev]: [n][n][n] real fp32.  Multiplies by the separable deapodisation
 * factors, scatters into the zeroed n_fine^3 complex grid at index n mod n_fine, runs one
 * forward (exponent -i, reading s1) 3-D cuFFT, and re-lays the result out centred with a
 * periodic halo of ceil(w/2)+1 cells.  Also tests whether the model is exactly even
 * (A[n] == A[-n]); if so the imaginary part of the grid is identically zero up to round-off and
 * a real fp32 copy is what spf_slice gathers.  SYNCHRONISES `stream` once to read that flag
 * back (this call is once per model update and is timed separately).
 */
SPF_API int spf_prepare_model(spf_ctx *ctx, const float *model, void *stream);

#define SPF_OUT_COMPLEX 0   /* out: complex64 [M][P] (re, im interleaved), c_{m,j} */
#define SPF_OUT_INTENSITY 1 /* out: fp32 [M][P], scale * Re c_{m,j}   (reading s3: a model image is Re c) */

/*
 * Steps a3-a5.  quats [dev] [M][4] fp32, pix_q [dev] [P][3] fp32, out [dev] per out_kind.
 *   c_{m,j} ~= sum_n A[n] exp(-i n . R(quat_m) q_j)   to the NUFFT tolerance eps.
 * M, P >= 0 (zero sizes are a no-op).  SPF_ESTATE before spf_prepare_model.
 */
SPF_API int spf_slice(spf_ctx *ctx, const float *quats, int64_t M, const float *pix_q, int64_t P, int32_t out_kind,
                      float scale, void *out, void *stream);

/*
 * Steps a6-a8.  images [dev] [n_img][P] fp32, slices [dev] [M][P] fp32, mask [dev] [P] bytes
 * (1 = use, 0 = leave the pixel out of every sum; NULL = all used; reading s8),
 * best_idx [dev] [n_img] int32, best_dist [dev] [n_img] fp32,
 * workspace [dev]: at least spf_match_workspace_bytes(n_img, M, P) bytes, 1024-byte aligned.
 *   d_{i,m} = sum_{j: mask_j} (I_ij - S_mj)^2,  best_idx[i] = argmin_m d_{i,m} (lowest m on
 *   exact ties of the computed fp32 distances), best_dist[i] = that distance.
 * With option match_impl = 0 (the tcgen05 matcher): evaluated as the conditioned expansion
 *   d = ||I - c||^2 + sum S'(S' + 2c) - 2 I.S',  S' = S - c,  c = the mean of up to 1,024 evenly spaced slices
 * (identical to the definition in exact arithmetic for any c), the cross term I.S' on the tensor
 * cores from two-term fp16 splits of both operands (fp32-equivalent products, fp32 accumulation), the three terms
 * added in fp64.  That decides the argmin; best_dist is then recomputed for the winner as the sum of squared
 * differences (fp64 sum, rounded once), so it is within fp32 round-off of the definition in every case.  Values must
 * satisfy |x| < 2^100 (they are rescaled by powers of two into fp16 range).  Two slices whose true distances to an
 * image differ by less than about 1e-6 (||I - c||^2 + ||S'||^2) can be ranked either way by the tensor-core pass
 * (reading s16); on the Poisson configurations that is far below the 1e-4 d near-tie window.
 * With match_impl = 1 (the library's starting value): the sum of squared differences as
 * written, in fp32 on the CUDA cores.  Either way the distance matrix is never written to
 * memory.  Requires M >= 1 when n_img >= 1.
 */
SPF_API int spf_match(spf_ctx *ctx, const float *images, int64_t n_img, const float *slices, int64_t M, int64_t P,
                      const uint8_t *mask, int32_t *best_idx, float *best_dist, void *workspace,
                      size_t workspace_bytes, void *stream);
SPF_API size_t spf_match_workspace_bytes(int64_t n_img, int64_t M, int64_t P);

/*
 * Steps a3-a8 fused at the a5 / a7 seam: the M orientations are sliced chunk_M at a time into a
 * buffer inside the workspace and each chunk is matched at once, the running (distance, index) keys merging across
 * chunks -- the [M][P] slice array never exists (26 GB at Matching-heavy; 79 GB for the paper's 1.2 M orientations x
 * 16,384 pixels).  Same result as spf_slice into an [M][P] array followed by spf_match, with one
 * difference on the tensor-core path: the common vector c of the conditioned expansion is the mean of the FIRST chunk's
 * slices (any c gives the same distances in exact arithmetic), and the winners are sliced once more (n_img x P points)
 * for the difference-form refinement of best_dist.  quats [dev] [M][4], pix_q [dev] [P][3], images [dev] [n_img][P],
 * mask [dev] [P] or NULL, best_idx / best_dist [dev] [n_img], workspace [dev] >= spf_slice_match_workspace_bytes(n_img,
 * min(chunk_M, M), P) bytes, 1024-byte aligned.  SPF_ESTATE before spf_prepare_model.
 */
SPF_API int spf_slice_match(spf_ctx *ctx, const float *quats, int64_t M, const float *pix_q, int64_t P, float scale,
                            const float *images, int64_t n_img, const uint8_t *mask, int64_t chunk_M, int32_t *best_idx,
                            float *best_dist, void *workspace, size_t workspace_bytes, void *stream);
SPF_API size_t spf_slice_match_workspace_bytes(int64_t n_img, int64_t chunk_M, int64_t P);

/*
 * Debug variant of spf_match for tests: additionally writes the full distance matrix
 * dist [dev] [n_img][M] fp32 with a plain CUDA-core kernel (one block per pair, difference form
 * accumulated in fp64, rounded once) -- used to check the matchers from a second, independent
 * GPU computation.  n_img * M < 2^31: small sizes only.
 */
SPF_API int spf_match_reference(spf_ctx *ctx, const float *images, int64_t n_img, const float *slices, int64_t M,
                                int64_t P, const uint8_t *mask, int32_t *best_idx, float *best_dist, float *dist,
                                void *stream);

/*
 * The whole path behind HOST buffers (all pointers [host]; pinned memory makes the copies
 * asynchronous): uploads model / quats / pix_q / images / mask, runs prepare -> slice -> match,
 * downloads best_idx / best_dist, synchronises.  The image upload runs on a second stream
 * underneath slicing.  slices_out [host] may be NULL; if not, the fp32 intensity slices
 * [M][P] are downloaded too.  Device buffers are cached inside ctx between calls.
 */
SPF_API int spf_orientation_match_host(spf_ctx *ctx, const float *model, const float *quats, int64_t M,
                                       const float *pix_q, int64_t P, float scale, const float *images,
                                       int64_t n_img, const uint8_t *mask, int32_t *best_idx, float *best_dist,
                                       float *slices_out);

/*
 * Inspection for tests (steps a1-a2 parity): copies the deapodisation factors (n doubles,
 * index i <-> n = i - floor(N/2)) to a [host] array, and the fine grid in natural FFT order
 * ([n_fine]^3 complex64, index l mod n_fine) to a [dev] array.  The latter synchronises.
 */
SPF_API int spf_debug_deapodisation(const spf_ctx *ctx, double *out_host);
SPF_API int spf_debug_fine_grid(spf_ctx *ctx, float *out_dev_complex, void *stream);

/*
 * Kernel variants and test/benchmark knobs (defaults in brackets):
 *   "slice_impl":  [1] = plain global-memory gather, one thread per point (the reference form);
 *                  2 = a warp per point, tile staged in shared memory by TMA: 32 lanes read an 8 x 8 window per x-plane
 *                      with no bank conflicts and a shuffle butterfly adds the partial sums (w <= 8; blocks whose box
 *                      does not fit the tile, and every block at w = 10, run as 3);
 *                  3 = the warp-per-point gather straight from global memory (no TMA, mbarrier or tile;
 *                      8 x 8 window at w = 8, 16-cell window at w = 10);
 *                  4 = as 2, the tile staged by cp.async (16-byte pieces copied by every thread, block barrier) instead of
 *                      TMA: classic CUDA only, the staged gather for a device on which the TMA path is not cleared
 *   "force_complex_grid": [0]; 1 = gather the complex grid even for an even model
 *   "match_impl":  0 = tcgen05 / TMEM / TMA split-fp16 GEMM with the fused a_i + b_m - 2 G + argmin epilogue (the product);
 *                  [1] = CUDA-core matcher: the difference form sum (I - S)^2 in fp32, register-tiled, same fused
 *                      argmin -- about 20x slower at Paper-scale, no tensor-core, TMA or mbarrier machinery;
 *                  2 = the same conditioned split-precision contraction on the warp-level tensor-core path (cp.async
 *                      pipeline, ldmatrix, mma.sync m16n8k16, fp32 accumulators in registers): classic CUDA only, the
 *                      tensor-core matcher for a device on which the tcgen05 kernel has not been cleared (legacy path:
 *                      it cannot reach tcgen05 throughput)
 *   "match_cta_group": CTAs per tcgen05 MMA (match_impl 0): 2 = cta_group::2 pairs (UMMA 256 x 256), [1] = single CTA (128 x 256)
 *   "match_chunk_kblocks": [32] 64-pixel K blocks accumulated inside TMEM before the epilogue warps add the chunk to
 *                  their fp32 registers with round-to-nearest adds; 0 = all of K in TMEM (spf_match_math.cuh)
 *   "match_condition": [1] = subtract the common vector c from the slices before the contraction; 0 = c = 0 (the plain
 *                  expansion ||I||^2 + ||S||^2 - 2 I.S)
 *   "match_refine": [1] = recompute the winner's distance in the difference form; 0 = return the epilogue's own value
 * The defaults are the variants with the least machinery (classic CUDA: no TMA, mbarrier or tcgen05).  The others
 * have not yet run on hardware and are opt-in: the caller switches them on once they have been
 * checked on the device at hand: spf_selftest (below) checks one and switches it on; the Python binding's
 * SpfContext.spf_autotune runs the same call in a child process first.
 *   "selftest_small": [0]; 1 = spf_selftest runs its small cases (a few hundred image-slice pairs): quick checks
 *   "record_events": [0]; 1 = spf_slice / spf_match record CUDA events on their stream around the
 *                    dominant kernels, read back with spf_last_kernel_ms
 * Returns SPF_EINVAL for an unknown key or value.
 */
SPF_API int spf_set_option(spf_ctx *ctx, const char *key, int64_t value);
SPF_API int spf_get_option(const spf_ctx *ctx, const char *key, int64_t *value);   /* value [host]; SPF_EINVAL for an unknown key */

/*
 * Device self-check of one kernel variant against this library's reference kernels, and the switch that turns a verified
 * variant on.  variant: "slice_gcoop" (slice_impl 3), "slice_coop_ld" (slice_impl 4), "slice_coop" (slice_impl 2), "match_mma" (match_impl 2), "match_cg1", "match_cg2" (the tcgen05
 * matcher on single CTAs / CTA pairs).  Slicing variants slice the caller's own prepared model (read-only; SPF_ESTATE
 * before spf_prepare_model) at 64 seeded orientations x 16,384 pixels with the reference gather and with the variant
 * (bar: relative L2 <= 3e-6, all finite); matcher variants run two seeded cases, with and without a mask, against
 * spf_match_reference (bar: distances within 1e-4 d; without the refinement 1e-4 d + 2e-6 of the norms; argmin equal
 * outside near-ties).  A consistency check between two CUDA paths, not parity (tests/ hold every variant to the oracle).
 * On success (report->passed = 1) the variant becomes the context's choice -- for slicers only if it was also the
 * fastest verified so far, the tcgen05 matcher supersedes the mma.sync one, pairs supersede single CTAs -- so a C caller reaches the TMA / tcgen05 kernels
 * with spf_create + spf_prepare_model + spf_selftest, no other option set.  Returns SPF_OK when the check RAN (passed or
 * not), another status when it could not (SPF_EFAULT: the variant's watchdog gave up).  Synchronises.  Runs in the
 * calling process: a variant that raises an SM exception takes the caller's CUDA context with it; callers that need
 * containment run it in a child process first (the Python binding's spf_autotune does).  report [host].
 */
typedef struct {
    int32_t passed;      /* 1 = the variant agrees with the reference kernels */
    float ms_variant;    /* device time of the variant on the check's timing case (CUDA events) */
    float ms_reference;  /* the same for the reference kernel */
    double worst_rel;    /* slicers: relative L2 difference; matchers: worst relative distance error (refined result) */
    char detail[192];    /* one line of text */
} spf_selftest_report;
SPF_API int spf_selftest(spf_ctx *ctx, const char *variant, spf_selftest_report *report, void *stream);

/*
 * Measures one of the device figures the rooflines divide by (the SM-side peaks must be
 * microbenchmarked, not taken from a data sheet).  what: "lds32" / "lds128" -- aggregate shared-memory load bandwidth with
 * conflict-free 4-byte / 16-byte loads (all SMs, 4 blocks of 512 threads each); "l2" -- L2 -> SM read bandwidth (a 48 MB
 * buffer streamed 20 times with L1-bypassing loads); "hbm_read" / "hbm_copy" -- 1 GB read twice / copied once.  Best of
 * three timed repetitions after a warm-up, CUDA events on `stream`.  gb_per_s [host].  Synchronises.
 */
SPF_API int spf_microbench(spf_ctx *ctx, const char *what, double *gb_per_s, void *stream);

/*
 * Watchdog.  Every wait on a hardware barrier inside the slicing and matching kernels is bounded
 * (about two seconds of SM clocks): a pipeline that stalls makes its block record a fault, raise the
 * context's device-global abort flag (every other block gives up at its next poll, blocks that start
 * later return at entry: one time-out per launch, not one per block), let its in-flight asynchronous
 * copies and MMAs land, and leave through the normal teardown instead of spinning for ever.  spf_check_fault synchronises
 * `stream`, and returns SPF_EFAULT (text: which kernel, role, block and tile) if any kernel
 * launched through this context since the last check recorded one, else SPF_OK.  The fault is
 * cleared by the call.  spf_orientation_match_host checks it itself before returning.
 */
SPF_API int spf_check_fault(spf_ctx *ctx, void *stream);

/*
 * Number of launches of this library's OWN kernels since the context was created (cuFFT's kernels
 * and memsets are not counted), so that the harness can report gpu_launches.
 */
SPF_API int64_t spf_launch_count(const spf_ctx *ctx);

/*
 * Device time in milliseconds (CUDA events recorded on the stream the kernel was launched on,
 * SURVEY.md section 8(d)) of the last call made with option "record_events" = 1:
 *   which = 0: the interpolation kernel of the last spf_slice   (steps a3-a5, one launch)
 *   which = 1: the contraction of the last spf_match            (steps a7-a8: both tcgen05 instantiations, or k_match_simt)
 *   which = 2: the operand preparation of the last spf_match    (step a6: abs-max, split, norms)
 * ms [host].  Synchronises on the closing event.  SPF_ESTATE when nothing was recorded.
 */
SPF_API int spf_last_kernel_ms(spf_ctx *ctx, int32_t which, float *ms);

/*
 * Number of fp16 operand products the last spf_match issued per K step: 2 when every image value
 * was exact in one fp16 term (photon counts), else 3; 0 when that call ran the CUDA-core matcher
 * (match_impl 1).  products [host].  Synchronises the stream of that call and reads one word of its
 * workspace, which must still be allocated.
 */
SPF_API int spf_last_match_products(spf_ctx *ctx, int32_t *products);

#ifdef __cplusplus
}
#endif
#endif /* SPF_H_ */
