/*
 * sgs.h -- C ABI of the B200-native differentiable 2D-Gaussian (surfel) splatting renderer,
 * the hot path of 2DGS-SLAM (arxiv 2506.00970).  Citations are PAPER.md line numbers; "R<n>"
 * are the readings of the paper listed in DESIGN.md §3.
 *
 * The interface follows the paper's statement of the problem: a map of splats
 * (mu, R, s_u, s_v, c, alpha) (L122) and a camera pose T_cw in SE(3) with a projection W (L95) go
 * in; colour, depth, normal and opacity images come out (Eq. 8); a rendering loss's
 * image gradients go in, gradients to the splat parameters (L122) and to the pose in the tangent
 * space of SE(3) (Eq. 9-13) come out; tracking renders only active splats (L204).
 *
 * Conventions
 *   - Plain pointers and sizes only.  Every pointer says HOST or DEVICE.  All device buffers are
 *     the caller's (borrowed for the duration of the call / until the matching backward); the
 *     library never frees them.  The ctx owns its workspace, obtained through the caller's
 *     allocator callbacks (or cudaMalloc/cudaFree when the callbacks are NULL).
 *   - Every call returns an int status (SGS_OK = 0).  No exceptions, no abort, no stdout.
 *   - Work is enqueued on the given CUDA stream (a cudaStream_t passed as void*).  sgs_render in
 *     the default (safe) mode waits once for the tile-entry count E; with SGS_FLAG_ASYNC it does
 *     not synchronise at all and a workspace overflow is reported by the NEXT call on the ctx.
 *   - Scales and opacity are ACTIVATED values (s > 0 metres, opacity in (0,1]) (R16).  The
 *     quaternion is (w,x,y,z), need not be unit; it is normalised inside and its gradient
 *     includes the normalisation.
 *   - Pixel (i,j) samples the image point (i+0.5, j+0.5), x = fx X/Z + cx (R17).  Images are
 *     channel-planar fp32, background 0.  depth = sum w z, normal = sum w t_nc (camera space,
 *     not flipped, not normalised), alpha = sum w (R9, R10).
 *   - Pose gradient: d_pose6 = (dL/drho, dL/dtheta) for the left perturbation
 *     T <- Exp(tau) o T_cw, tau = (rho, theta), translation first (Eq. 12-13, R15).
 *   - Gradients are OVERWRITTEN, and are exactly zero for inactive or culled surfels (sgs_backward_accumulate adds).
 */
#ifndef SGS_H
#define SGS_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define SGS_API __attribute__((visibility("default")))
#else
#define SGS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sgs_ctx sgs_ctx; /* opaque; owns workspace + the last forward's saved state */

/* Caller's device allocator (e.g. torch's caching allocator).  stream is a cudaStream_t. */
typedef void* (*sgs_alloc_fn)(size_t bytes, void* user, void* stream);
typedef void (*sgs_free_fn)(void* ptr, void* user, void* stream);

enum {
    SGS_OK = 0,
    SGS_INVALID_ARGUMENT = 1,
    SGS_OUT_OF_MEMORY = 2,
    SGS_WORKSPACE_OVERFLOW = 3, /* async mode: the previous render overflowed; workspace was grown, render again */
    SGS_NO_FORWARD_STATE = 4,   /* sgs_backward without a preceding successful sgs_render */
    SGS_CUDA_ERROR = 5,
    SGS_LIMIT_EXCEEDED = 6      /* sgs_map_correction_static: more keyframes than SGS_STATIC_MAX_FRAMES */
};

enum {
    SGS_FLAG_ASYNC = 1,         /* never synchronise the host in sgs_render; an overflow is reported by a later call */
    SGS_FLAG_RADIX_BINNING = 2, /* bin with the global LSD radix sort of the 64-bit keys instead of the
                                   default per-tile buckets + in-tile sort; same list, kept for A/B checks */
    SGS_FLAG_TRACK_REUSE = 4,   /* sgs_track_iter: the map is frozen between sgs_track_new_frame calls, see there */
    SGS_FLAG_LAZY_GRADS = 8,    /* sgs_backward: d_surfels / d_pose6 are complete only behind sgs_wait_grads, see there */
    SGS_FLAG_GRAPH = 32,        /* SGS_FLAG_ASYNC for stream capture: sgs_render, sgs_render_contrib / _median, sgs_backward,
                                   sgs_backward_tracking, sgs_track_iter and the loss calls enqueue kernels and copies on the
                                   caller's stream ONLY (the context has no stream of its own, queries and waits for no
                                   event), so the sequence can be recorded into a CUDA graph once an eager run has brought the
                                   workspace to size (a call that had to grow it would allocate: do not capture the first).
                                   Nothing reports a bucket overflow by itself in this mode: sgs_get_stats (which
                                   synchronises the device) does.  sgs_prepare is SGS_INVALID_ARGUMENT. */
    SGS_FLAG_TIGHT_BINNING = 64, /* SURVEY 8(f) NEXT-3, readings R26 + R27 (Eq. 8 L114-116 with the truncation rules R3/R4):
                                   the tile lists hold only what can contribute.  (i) Opacity-aware cutoff: a pair contributes only if
                                   o exp(-rho^2/2) >= alpha_min, so splat k's support is rho^2 <= c_k^2 = min(cutoff^2, 2 ln(o_k /
                                   alpha_min)); its screen AABB and tile rectangle are those of that ellipse, and o_k < alpha_min is
                                   culled.  (ii) Tile-exact culling: a tile of the rectangle is listed only if the support ellipse
                                   reaches the rectangle of the tile's pixel centres.  Images and gradients are those of the default
                                   binning (same rendered function); sgs_get_binning returns the shorter lists, bit-identical to the
                                   oracle's tight mode.  Not together with SGS_FLAG_RADIX_BINNING (sgs_create: SGS_INVALID_ARGUMENT). */
    SGS_FLAG_LOWPASS = 128,     /* SURVEY 8(f) NEXT-3, reading R28 (the paper states no filter, R8; this is the published 2DGS remedy for
                                   sub-pixel and edge-on splats, restated): the Gaussian weight of a pair is the larger of the splat's
                                   own and a screen-space Gaussian of sigma = sqrt(2)/2 px around the projected centre x_c,
                                   rho^2 = min(u^2 + v^2, 2 |x - x_c|^2); where the screen term wins the pair's depth is the centre
                                   depth, and its gradient reaches the splat through x_c.  The footprint is the cutoff ellipse united
                                   with the disc of radius cutoff / sqrt 2 around x_c.  Supported by sgs_render, sgs_prepare,
                                   sgs_backward(_accumulate), sgs_backward_tracking and the loss calls; sgs_track_iter takes the
                                   unfused sequence; sgs_render_contrib / sgs_render_median return SGS_INVALID_ARGUMENT; not together
                                   with SGS_FLAG_TIGHT_BINNING or SGS_FLAG_NORMALISED_DEPTH (sgs_create: SGS_INVALID_ARGUMENT). */
    SGS_FLAG_NORMALISED_DEPTH = 16 /* SURVEY 8(f) NEXT-3 (variant of R9; Eq. 8 L116-120 renders D = sum w z and
                                   O = sum w): the depth image is the expected depth D_n = D / O (0 where O = 0), i.e.
                                   the blend weights renormalised to sum to one, so a partly transparent surface keeps
                                   its metric depth.  The forward keeps (D_n, 1/O) per pixel in the context; every
                                   backward (sgs_backward, the tracking backward) then takes the depth upstream as
                                   dL/dD_n and carries it to dL/dD = g/O and dL/dO -= g D_n/O inside the compositing
                                   backward's prologue.  Losses computed by this library (Eq. 15-19, Eq. 23-26) see D_n.
                                   sgs_track_iter keeps its one-kernel iteration under this flag. */
};

/* Truncation conventions of Eq. 8 (R3-R7).  sgs_default_config fills the defaults shown. */
typedef struct {
    int tile;        /* 16: tile edge in pixels (only 16 is supported)                       */
    float cutoff;    /* 3.0: pairs with u^2+v^2 > cutoff^2 contribute nothing (R3)           */
    float alpha_min; /* 1/255: pairs with a < alpha_min are skipped (R4)                     */
    float alpha_max; /* 0.99: a = min(alpha_max, o G), true derivative (0 when clamped) (R5) */
    float t_min;     /* 1e-4: stop the pixel when T(1-a) < t_min, that splat excluded (R6)   */
    float z_near;    /* 0.2: cull centre depth <= z_near; skip pair with hit depth <= z_near (R7) */
    int flags;       /* SGS_FLAG_* */
    sgs_alloc_fn alloc; /* nullable */
    sgs_free_fn free;   /* nullable */
    void* user;
} sgs_config;

/* The map (L122, Eq. 14's g_i and delta_i).  All DEVICE pointers, fp32, borrowed. */
typedef struct {
    int64_t n;
    const float* mean;     /* n x 3  world-space centre mu                       */
    const float* scale;    /* n x 2  s_u, s_v                                    */
    const float* quat;     /* n x 4  (w,x,y,z); R = [t_u, t_v, t_n]              */
    const float* opacity;  /* n                                                   */
    const float* rgb;      /* n x 3  plain RGB, no spherical harmonics (L128)     */
    const uint8_t* active; /* n or NULL (= all active); the active flag delta_i (L161, L204) */
} sgs_surfels;

/* Camera: pinhole intrinsics in pixels standing for W (L95, R14) and T_cw (HOST values). */
typedef struct {
    int width, height;
    float fx, fy, cx, cy;
    float T_cw[12]; /* row-major 3x4 [R | t], world -> camera */
} sgs_camera;

/* Output images / upstream gradients, DEVICE, caller-owned, channel-planar fp32.
 * In sgs_render any pointer may be NULL (that image is not written).
 * In sgs_backward a NULL pointer means a zero upstream gradient for that image. */
typedef struct {
    float* rgb;    /* 3 x H x W */
    float* depth;  /* H x W     */
    float* normal; /* 3 x H x W */
    float* alpha;  /* H x W     */
} sgs_images;

/* Surfel gradients, DEVICE, caller-owned, overwritten.  Layout as sgs_surfels. */
typedef struct {
    float* mean;    /* n x 3 */
    float* scale;   /* n x 2 */
    float* quat;    /* n x 4 */
    float* opacity; /* n     */
    float* rgb;     /* n x 3 */
} sgs_surfel_grads;

/* Counters of the last render (HOST struct; reading it synchronises the stream of that render). */
typedef struct {
    int64_t n_visible;    /* surfels that passed culling (N_v)                 */
    int64_t n_entries;    /* tile entries E                                    */
    int64_t capacity;     /* current entry capacity of the workspace           */
    int64_t overflow;     /* 1 if the last render dropped entries              */
    int64_t workspace_bytes;
    int64_t kernel_launches; /* kernels this ctx has launched since creation (memsets/copies not counted) */
} sgs_stats;

/* Per-stage device timing (CUDA events recorded on the caller's stream around each stage). */
enum { SGS_STAGE_PREPROCESS = 0, SGS_STAGE_SORT = 1, SGS_STAGE_FORWARD = 2, SGS_STAGE_LOSS = 3,
       SGS_STAGE_BACKWARD = 4, SGS_STAGE_TRACK = 5 /* sgs_track_iter's fused kernel */, SGS_STAGE_COUNT = 6 };

SGS_API int sgs_default_config(sgs_config* cfg);
/* (Test hook: if the environment variable SGS_DEBUG_HELPER_DELAY_NS is set when the ctx is created, the helper blocks of
 * sgs_track_iter's kernel sleep that many nanoseconds before they start -- results must not depend on it.) */
SGS_API int sgs_create(sgs_ctx** out, const sgs_config* cfg);
SGS_API int sgs_destroy(sgs_ctx* ctx);

/* Forward (Eq. 1-8): preprocess (Eq. 5-7, culling, screen AABB) -> tile binning (the list of (tile, depth, surfel)
 * entries in the order of the 64-bit key tile << 32 | depth bits, ties by surfel index: per-tile buckets + an in-tile
 * sort by default, one global radix sort with SGS_FLAG_RADIX_BINNING -- the same list either way) -> per-tile
 * front-to-back compositing (Eq. 8 with the truncation rules R3-R7).  Saves the state sgs_backward needs inside ctx.
 *   surfels: DEVICE map, borrowed until the matching sgs_backward;  cam: HOST;  out: DEVICE images, any may be NULL.
 * Errors: SGS_INVALID_ARGUMENT (NULL / non-positive sizes / n >= 2^24), SGS_OUT_OF_MEMORY (workspace),
 * SGS_WORKSPACE_OVERFLOW (async mode, see above), SGS_CUDA_ERROR. */
SGS_API int sgs_render(sgs_ctx* ctx, const sgs_surfels* surfels, const sgs_camera* cam, const sgs_images* out,
               void* cuda_stream);

/* First half of sgs_render on its own: preprocess + tile binning of (surfels, cam), enqueued on `stream`, nothing
 * rendered.  The next sgs_render on this ctx with the SAME surfels struct and camera (compared bytewise) skips its
 * own binning, orders its stream behind this call's work (an internal event; the two streams may differ) and goes
 * straight to compositing; any other call in between drops the prepared state.  The call itself is ordered behind
 * the ctx's last sgs_render / sgs_backward, whose stream may differ as well.  Purpose: in a mapping window (L248-252:
 * several keyframes rendered against one map) the latency-bound binning of view v+1, on a second ctx and a side
 * stream, hides under the compositing kernels of view v.  Same arguments, status codes and async-mode overflow
 * reporting as sgs_render. */
SGS_API int sgs_prepare(sgs_ctx* ctx, const sgs_surfels* surfels, const sgs_camera* cam, void* cuda_stream);

/* sgs_render that additionally returns the contribution of every splat to the view (Eq. 20-21):
 * contrib[k] = C_k^V = sum over pixels of w_k(p) = a_k T_k, "how many pixels the splat contributes to"; the
 * paper calls a splat visible in the view when C_k^V > 0.5 (keyframe selection, state update, pruning).
 *   contrib: DEVICE, n floats, overwritten; exactly 0 for inactive, culled or never-composited splats. */
SGS_API int sgs_render_contrib(sgs_ctx* ctx, const sgs_surfels* surfels, const sgs_camera* cam, const sgs_images* out,
                               float* contrib, void* cuda_stream);

/* sgs_render that additionally returns the MEDIAN depth image (reading R9m; a variant of the depth
 * image of L118-120): along a pixel's ray the blending weights w_i = a_i T_i of Eq. 8 and the remaining transmittance
 * form a distribution over the intersection depths z_i; median[p] is the z_i of the composited splat at which the
 * transmittance first falls to T_{i+1} <= 1/2, and 0 where the pixel stays below half opacity.  Forward only: the image is
 * piecewise constant in the opacities and carries no gradient; sgs_backward after this call is that of sgs_render.
 *   median: DEVICE, H x W floats, overwritten.  Other arguments, status codes and stream order as sgs_render. */
SGS_API int sgs_render_median(sgs_ctx* ctx, const sgs_surfels* surfels, const sgs_camera* cam, const sgs_images* out,
                              float* median, void* cuda_stream);

/* Covisibility score of two views (Eq. 22): |G_A n G_B| / |G_A u G_B| with
 * G_V = {k : active[k] != 0 and C_k^V > threshold} (paper: threshold 0.5).
 *   contrib_a, contrib_b: DEVICE, n floats (outputs of sgs_render_contrib);  active: DEVICE n bytes or NULL
 *   result3: DEVICE, 3 floats, overwritten: score (0 when the union is empty), |intersection|, |union| */
SGS_API int sgs_covisibility(sgs_ctx* ctx, const float* contrib_a, const float* contrib_b, int64_t n, const uint8_t* active,
                             float threshold, float* result3, void* cuda_stream);

/* Backward of the most recent sgs_render on this ctx (same surfel buffers, unchanged) (Eq. 9-13).
 *   upstream : dL/d(rgb, depth, normal, alpha)                                     DEVICE
 *   d_surfels: nullable; NULL = pose-only mode (tracking, L204: splats frozen)     DEVICE
 *   d_pose6  : nullable; 6 floats (rho, theta), Eq. 11-13                          DEVICE
 * All results are complete in the order of `cuda_stream` (the zero-fill of d_surfels runs on a stream of the ctx
 * beside the compositing kernel and is joined before the call's last kernel).
 * Errors: SGS_NO_FORWARD_STATE without a preceding successful sgs_render (also after sgs_track_iter, sgs_prepare),
 * SGS_WORKSPACE_OVERFLOW (async mode: that render had overflowed; render again), SGS_OUT_OF_MEMORY, SGS_CUDA_ERROR. */
SGS_API int sgs_backward(sgs_ctx* ctx, const sgs_images* upstream, const sgs_surfel_grads* d_surfels, float* d_pose6,
                 void* cuda_stream);

/* sgs_backward that ADDS this view's surfel gradients to d_surfels instead of overwriting them: the paper's mapping
 * iteration samples N_a + N_i keyframes and takes ONE optimiser step on their summed loss (L248-252, Tab. I), so
 * the gradients of a window of views are a sum.  Nothing is zero-filled (sgs_backward's five N-sized memsets and its write of
 * all N x 13 values go away; only the splats a view sees are touched): the caller zeroes d_surfels once per window
 * (sgs_zero_grads, or its own memset).  d_pose6 is still OVERWRITTEN: every view has its own pose.  d_surfels must not be
 * NULL.  Calls of one window must be ordered (same stream, or one ctx under SGS_FLAG_LAZY_GRADS); two contexts working on
 * one window need an accumulator each.  Other arguments, state and errors as sgs_backward. */
SGS_API int sgs_backward_accumulate(sgs_ctx* ctx, const sgs_images* upstream, const sgs_surfel_grads* d_surfels,
                                    float* d_pose6, void* cuda_stream);

/* Zero-fills the non-NULL arrays of d_surfels (n surfels) on the stream: the start of an accumulation window. */
SGS_API int sgs_zero_grads(sgs_ctx* ctx, const sgs_surfel_grads* d_surfels, int64_t n, void* cuda_stream);

/* SGS_FLAG_LAZY_GRADS.  The last kernel of a full sgs_backward (per-surfel chain rule Eq. 9-10, pose reduction Eq. 13,
 * latency-bound) then stays on a stream of the ctx and `cuda_stream` does not wait for it, so that the next view's
 * kernels (another ctx, same caller stream) run meanwhile.  d_surfels and d_pose6 of that call are complete on a stream
 * only after sgs_wait_grads(ctx, that stream); the ctx orders its own later calls behind the kernel by itself.
 * Without the flag sgs_wait_grads is a no-op. */
SGS_API int sgs_wait_grads(sgs_ctx* ctx, void* cuda_stream);

/* Tracking loss of Eq. 15-19 (harness around the renderer; R18, R19):
 *   L_t = 1/|Omega| sum_p M_n M_o (|I_r - I|_1 + lambda_d |D_r - D|)
 * with M_o = [alpha > 0.95] and M_n = [normal_sign * N_r . ray > 0].  Writes the upstream
 * gradients of the rendered images into `upstream` (all four, zeros where masked) and the scalar
 * loss into loss (DEVICE, 1 float).  rendered/target/upstream are DEVICE; target uses only
 * rgb and depth. */
SGS_API int sgs_tracking_loss(sgs_ctx* ctx, const sgs_camera* cam, const sgs_images* rendered, const sgs_images* target,
                      float lambda_d, float normal_sign, const sgs_images* upstream, float* loss, void* cuda_stream);

/* Mapping loss of Eq. 24-26 (L232-248) without the SSIM term of Eq. 24, which sgs_ssim_loss adds on top; harness
 * around the renderer for the mapping-shaped configs:
 *   L = 1/|Omega| sum_p [ lambda_c |I_r - I|_1 + w_d |D_r - D| + w_n (1 - normal_sign N_{D_r} . N_r) ]
 * N_{D_r}: unit cross product of the central differences of the points back-projected from the RENDERED depth
 * (Eq. 23, 25; reading R23), interior pixels only.  Writes dL/d(rgb, depth, normal, alpha) of the rendered images
 * into `upstream` (the depth gradient includes the chain through N_{D_r}; alpha gets 0) and L into loss
 * (DEVICE, 1 float).  rendered / target / upstream: DEVICE; target uses rgb and depth. */
SGS_API int sgs_mapping_loss(sgs_ctx* ctx, const sgs_camera* cam, const sgs_images* rendered, const sgs_images* target,
                             float lambda_c, float w_d, float w_n, float normal_sign, const sgs_images* upstream,
                             float* loss, void* cuda_stream);

/* Tracking iteration backward (L180-204): the Eq. 15-19 loss of sgs_tracking_loss evaluated INSIDE the
 * pose-only backward on the images of the most recent sgs_render (whose output buffers must still hold
 * them), so neither the upstream gradients nor a loss kernel touch HBM.  target: DEVICE rgb + depth.
 * d_pose6 (6 floats) and loss (1 float, nullable): DEVICE.  Same result as sgs_tracking_loss followed
 * by sgs_backward(upstream, NULL, d_pose6). */
SGS_API int sgs_backward_tracking(sgs_ctx* ctx, const sgs_images* target, float lambda_d, float normal_sign,
                                  float* d_pose6, float* loss, void* cuda_stream);

/* One whole tracking iteration (L180-204): preprocess + tile binning (two launches; one with SGS_FLAG_TRACK_REUSE), then ONE kernel that
 * composites each tile (Eq. 8), evaluates Eq. 15-19 against the current frame in registers and walks the
 * tile's list back for the pose gradient (Eq. 11-13); images, T and the upstream gradients never leave the
 * SM.  Same result as sgs_render + sgs_backward_tracking (bit-identical images, loss and 6-vector up to
 * the order of the block sums).
 *   surfels : DEVICE map; only active splats are rendered (L204)
 *   target  : DEVICE rgb (3xHxW) + depth (HxW) of the current frame
 *   out     : nullable; DEVICE images to write (any pointer may be NULL = not written)
 *   d_pose6 : DEVICE, 6 floats (rho, theta); loss: DEVICE, 1 float, nullable
 * (A one-block kernel that orders the tiles by their measured cost for the next iteration runs on a stream of the ctx.)
 * Leaves no state for sgs_backward (SGS_NO_FORWARD_STATE); sgs_get_binning works.
 * With SGS_FLAG_ASYNC the counters of an iteration reach the host behind its compositing kernel and are never waited
 * for: a tile-bucket overflow is reported (SGS_WORKSPACE_OVERFLOW, workspace grown) by the first later call on the
 * ctx that finds them there, or by sgs_get_stats, which waits. */
SGS_API int sgs_track_iter(sgs_ctx* ctx, const sgs_surfels* surfels, const sgs_camera* cam, const sgs_images* target,
                           float lambda_d, float normal_sign, const sgs_images* out, float* d_pose6, float* loss,
                           void* cuda_stream);

/* sgs_track_iter with the pose in DEVICE memory (L204: the pose is iterated "until convergence or reaching the maximum number
 * of iterations"): d_T_cw (DEVICE, 12 floats, row-major 3x4 [R | t]) is read by the preprocess kernels when they run, so the
 * caller's own pose-update kernel -- d_pose6 in, d_T_cw out -- can sit between the iterations of one stream or of one captured
 * CUDA graph (SGS_FLAG_GRAPH) with no host round trip.  cam carries the image size and intrinsics; its T_cw is ignored.
 * With SGS_FLAG_TRACK_REUSE the kept survivor list is built around the device pose of the iteration that builds it (the first
 * after sgs_track_new_frame); the host cannot see later poses, so the check against the list's margin is made on the device.
 * INVALID RESULTS ARE NaN: an iteration whose pose has left the margin (call sgs_track_new_frame and repeat), or -- in every
 * mode of sgs_track_iter -- one whose tile buckets overflowed, writes NaN to *loss and d_pose6 instead of numbers computed
 * from incomplete lists.  Not with SGS_FLAG_RADIX_BINNING (SGS_INVALID_ARGUMENT).  Otherwise as sgs_track_iter. */
SGS_API int sgs_track_iter_dev(sgs_ctx* ctx, const sgs_surfels* surfels, const sgs_camera* cam, const float* d_T_cw,
                               const sgs_images* target, float lambda_d, float normal_sign, const sgs_images* out,
                               float* d_pose6, float* loss, void* cuda_stream);

/* SGS_FLAG_TRACK_REUSE.  Tracking optimises the pose of ONE frame over many iterations against a frozen map (L204).
 * With the flag set, the caller promises that between two sgs_track_new_frame calls the arrays behind a bytewise-equal
 * sgs_surfels struct (means, scales, active flags) do not change.  sgs_track_iter then keeps the survivor list of its
 * conservative pre-cull (active and possibly inside the frustum), built with a margin of 3 cm / 0.02 rad around the
 * pose of the iteration that built it, and skips that pass over the whole map while the pose stays inside 80 % of the
 * margin; a pose outside, another surfels struct, or any other binning call on the ctx rebuilds it.  The exact
 * culling and everything after it run every iteration on the listed splats, so results are unchanged
 * (tests: binning bit-identical to the oracle's along a pose trajectory that leaves the margin).
 * sgs_track_new_frame drops the list (call it when the map may have changed, i.e. at every new frame). */
SGS_API int sgs_track_new_frame(sgs_ctx* ctx);

/* Debug export of the binning of the last render, for bit-exact parity tests.  Synchronises.
 * Returned DEVICE pointers stay valid until the next call on ctx.  idx holds ORIGINAL surfel
 * indices; culled[i] = 1 iff surfel i was inactive or culled. */
SGS_API int sgs_get_binning(sgs_ctx* ctx, int64_t* n_entries, const uint64_t** keys, const uint32_t** idx,
                    const uint32_t** tile_ranges /* tiles x 2 */, const uint8_t** culled /* n */);

SGS_API int sgs_get_stats(sgs_ctx* ctx, sgs_stats* out);

/* Profiling: when enabled, every stage launch is bracketed by a pair of CUDA events on its stream.
 * sgs_get_profile waits for the device, adds up the elapsed milliseconds and call counts per stage
 * (HOST arrays of SGS_STAGE_COUNT entries) and, if reset != 0, clears the record. */
SGS_API int sgs_set_profiling(sgs_ctx* ctx, int enabled);
SGS_API int sgs_get_profile(sgs_ctx* ctx, double* ms, int64_t* calls, int reset);

/* HOST-buffer convenience path (end-to-end measurement): copies in, runs, copies out, waits.
 * sgs_upload_surfels copies a HOST map into ctx-owned device memory and makes it the resident
 * map; the *_host calls use the resident map. */
SGS_API int sgs_upload_surfels(sgs_ctx* ctx, const sgs_surfels* host_surfels, void* cuda_stream);
SGS_API int sgs_render_host(sgs_ctx* ctx, const sgs_camera* cam, const sgs_images* host_out, void* cuda_stream);
SGS_API int sgs_backward_host(sgs_ctx* ctx, const sgs_images* host_upstream, const sgs_surfel_grads* host_d_surfels,
                      float* host_d_pose6, void* cuda_stream);
/* One tracking iteration on the resident map against a resident target frame (uploaded by
 * sgs_upload_target): render, Eq. 15-19 loss, pose-only backward; reads back loss and the 6-vector. */
SGS_API int sgs_upload_target(sgs_ctx* ctx, const sgs_camera* cam, const float* host_rgb /*3xHxW*/,
                      const float* host_depth /*HxW*/, void* cuda_stream);
SGS_API int sgs_track_iter_host(sgs_ctx* ctx, const sgs_camera* cam, float lambda_d, float normal_sign,
                        float* host_loss, float* host_d_pose6, void* cuda_stream);

/* Mapping window on the resident map through HOST buffers (L234-252: per sampled keyframe render, Eq. 24-26 loss, full
 * backward; one optimiser step per window).  sgs_map_view_host uploads the keyframe (HOST rgb 3xHxW, depth HxW; pinned memory
 * keeps the copy asynchronous), renders the resident map, evaluates L = Eq. 24-26 (sgs_mapping_loss(lambda_c, w_d, w_n) +
 * sgs_ssim_loss(ssim_weight); ssim_weight 0 skips the SSIM term) and ADDS the view's surfel gradients to the ctx's window
 * accumulator on the device.  Nothing waits: *host_loss (1 float, nullable) and host_pose6 (6 floats, nullable; this view's
 * dL/dtau) are written by sgs_sync_host.  At most 64 views between two sgs_sync_host calls (SGS_INVALID_ARGUMENT beyond).
 * sgs_fetch_grads_host ends the window: the accumulated gradients are copied to host_d_surfels (HOST, n x {3,2,4,1,3} floats,
 * NULL arrays skipped) on a stream of the ctx behind the window's last kernel, the accumulator is re-zeroed behind the copy,
 * and the next window fills a second accumulator meanwhile; the host arrays are complete after sgs_sync_host, which waits
 * for `cuda_stream` and for the ctx's copies and delivers the pending per-view results. */
SGS_API int sgs_map_view_host(sgs_ctx* ctx, const sgs_camera* cam, const float* host_target_rgb, const float* host_target_depth,
                              float lambda_c, float w_d, float w_n, float ssim_weight, float normal_sign, float* host_loss,
                              float* host_pose6, void* cuda_stream);
SGS_API int sgs_fetch_grads_host(sgs_ctx* ctx, const sgs_surfel_grads* host_d_surfels, void* cuda_stream);
/* The same hand-over, sparse: a window only touches the surfels its views see (L248-252; in a 2 M-surfel map a view sees
 * ~7 %), so instead of n dense rows the device delivers the rows that hold anything.  Row k < count of every non-NULL
 * array of host_rows ({3,2,4,1,3} floats per row) is the accumulated gradient of surfel host_ids[k]; ids ascend; a surfel
 * is listed iff at least one of its 13 accumulated values is not +-0 (NaN counts), so scattering the rows into zeros gives
 * exactly what sgs_fetch_grads_host would have delivered, bit for bit.  host_ids and the arrays of host_rows (HOST, room
 * for `cap` rows; pinned memory keeps the copies asynchronous) are written by copy commands that a LATER call of this
 * group enqueues, once the device has packed the rows and published their number (sgs_map_view_host if the pack is
 * complete by then, the next fetch, or sgs_sync_host): they must stay valid until sgs_sync_host, after which they and
 * *host_count (HOST, nullable: the number of listed surfels) are complete.  If the count exceeds cap, only the first cap
 * rows are delivered and the rest of the window is lost (cap = n can not overflow).  The accumulator is re-zeroed and the
 * double buffer swapped as in sgs_fetch_grads_host; at most 64 fetches between two sgs_sync_host calls. */
SGS_API int sgs_fetch_grads_sparse_host(sgs_ctx* ctx, int32_t* host_ids, const sgs_surfel_grads* host_rows, int64_t cap,
                                        int64_t* host_count, void* cuda_stream);
SGS_API int sgs_sync_host(sgs_ctx* ctx, void* cuda_stream);

/* SSIM term of the colour loss (Eq. 24; reading R24): per channel the structural similarity index of [87],
 * 11 x 11 Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2;
 *   L = weight / (3 |Omega|) sum_c sum_p (1 - SSIM_c(p)).
 * ACCUMULATES: dL/d(rendered rgb) is added to upstream_rgb and L to *loss, so that it composes with
 * sgs_mapping_loss (call that first; Eq. 24's weights: sgs_mapping_loss(lambda_c, ...) then sgs_ssim_loss(1 - lambda_c)).
 *   rendered_rgb, target_rgb, upstream_rgb: DEVICE 3 x H x W;  loss: DEVICE 1 float, nullable. */
SGS_API int sgs_ssim_loss(sgs_ctx* ctx, int width, int height, const float* rendered_rgb, const float* target_rgb,
                          float weight, float* upstream_rgb, float* loss, void* cuda_stream);

/* Map correction after pose-graph optimisation (Eq. 31-32), in place: Delta T_f = T_f^o T_f^{-1} and
 * mu_k <- Delta T_f mu_k, R_k <- Delta R_f R_k with f = frame_id[k], the splat's closest observed keyframe.
 * CONVENTION (reading R29): Eq. 31-32 as printed keep a splat fixed in its keyframe's camera frame -- the purpose of the
 * correction, L302-306 -- exactly when the poses are CAMERA-TO-WORLD (as a pose graph stores them): then
 * (T_f^o)^{-1} mu' = T_f^{-1} mu.  T_orig / T_opt are therefore camera-to-world [R | t]; a caller holding the world-to-camera
 * poses of sgs_camera.T_cw passes their inverses ([R^T | -R^T t]).  tests/test_gpu_map_correction.py renders a map from
 * the optimised keyframe after the correction and finds the image of the original map from the original keyframe.
 *   mean (n x 3), quat (n x 4, (w,x,y,z), 16-byte aligned), frame_id (n x int32; ids outside [0, n_frames) leave the
 *   splat untouched), T_orig / T_opt (n_frames x 12, row-major 3x4 [R|t] of T_f and T_f^o): all DEVICE. */
SGS_API int sgs_map_correction(sgs_ctx* ctx, int64_t n, float* mean, float* quat, const int32_t* frame_id, int n_frames,
                               const float* T_orig, const float* T_opt, void* cuda_stream);

/* The same operation for callers that must not allocate (code under CUDA stream capture, tight serving loops, harnesses
 * that forbid cudaMalloc): no ctx, and NO cudaMalloc / cudaFree / allocating library call on any path.  The per-keyframe
 * increments Delta T_f (64 bytes each), which sgs_map_correction keeps in the ctx's workspace, live in a static device
 * array of SGS_STATIC_MAX_FRAMES entries (256 KB that every GPU loading the library holds until the process exits).
 *   Arguments, layout and arithmetic as sgs_map_correction (same kernels: the results are bit-identical); all DEVICE.
 *   n_frames > SGS_STATIC_MAX_FRAMES returns SGS_LIMIT_EXCEEDED and touches nothing; other errors as sgs_map_correction.
 *   The array is shared by every call in the process on that device: each call rewrites the entries [0, n_frames) it
 *   reads before reading them, so nothing needs clearing and an earlier call's contents are never seen -- but two calls
 *   that OVERLAP on the GPU (different streams without an ordering between them) race on it: order them.
 *   The first call on a device looks the array's address up (cudaGetSymbolAddress; not an allocation): make one call
 *   outside stream capture before capturing. */
#define SGS_STATIC_MAX_FRAMES 4096
SGS_API int sgs_map_correction_static(int64_t n, float* mean, float* quat, const int32_t* frame_id, int n_frames,
                                      const float* T_orig, const float* T_opt, void* cuda_stream);

/* Measures this device's FP32 FMA throughput with a register-resident loop (16 independent chains per thread,
 * 8 blocks of 256 threads per SM, best of 4 timed launches, ~1 ms each; waits): the denominator of the compositing
 * kernels' roofline.  tflops: HOST double. */
SGS_API int sgs_measure_fp32_peak(double* tflops, void* cuda_stream);

/* A measurement, not a step of the path (north_star: "TMA bulk copies where that pays"): runs the staging of the compositing
 * kernels -- gather of the tile lists' 128-byte payload records, re-basing, seven 16-byte planes into shared memory -- over the
 * tile lists of the ctx's last sgs_render, `reps` times, with mode 0 = one thread per entry gathering seven 16-byte loads (what
 * the kernels do) or mode 1 = one cp.async.bulk (TMA) of the 128-byte record per entry into shared memory, completed through
 * an mbarrier, then the same arithmetic from shared memory.  us_per_launch: HOST double.  Waits.  SGS_NO_FORWARD_STATE
 * without a preceding sgs_render. */
SGS_API int sgs_probe_staging(sgs_ctx* ctx, int mode, int reps, double* us_per_launch, void* cuda_stream);

SGS_API const char* sgs_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* SGS_H */
