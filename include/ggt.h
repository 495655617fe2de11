/* ggt.h — C ABI of the B200-native geometry-guidance hot path of arxiv/paper_2505_18932
 * ("Geometry-guided Online 3D Video Synthesis with Multi-View Temporal Consistency").
 *
 * Three calls follow the paper's statement of the problem (PAPER.md:59 inputs, :96 output):
 *   ggt_refine_depth   colour-difference-mask temporal refinement of ONE input depth map
 *                      (Eq. 1-2)
 *   ggt_integrate      target camera + V input cameras / depth maps -> TSDF + weight volume laid out in
 *                      the target view's image space (pixel u,v x depth bin), overwrite or persistent
 *                      (Eq. 9-12; persistence: analogue of Eq. 13-14)
 *   ggt_extract_depth  volume -> per-pixel zero-crossing depth + confidence
 * plus ggt_raymarch_depth, the paper's own volume-free schedule (adaptive advance 0.8 s, sign change, three
 * bisection steps: PAPER.md:75, 348) on the same inputs.
 *
 * Conventions
 *   - every call returns int: GGT_OK (0) or a negative GGT_ERR_*; ggt_last_error() gives the text.
 *   - arguments named dev_* are DEVICE pointers owned by the caller (e.g. torch tensors); the library
 *     never frees them.  Camera structs, descriptor structs and pointer arrays are HOST memory, copied
 *     at call time.  Arguments named host_* are host pointers (pinned memory makes the copies async).
 *   - `stream` is the caller's cudaStream_t passed as void* (NULL = legacy default stream).  Calls
 *     validate host-side arguments synchronously, enqueue kernels on `stream` and return WITHOUT
 *     synchronising.  No exception crosses the ABI.
 *   - there is no CPU fallback: without a CUDA device every compute call returns GGT_ERR_CUDA.
 *   - stream capture: the compute calls only launch kernels on `stream` (arguments travel as kernel parameters), so a
 *     frame can be captured into a CUDA graph and replayed, provided nothing has to grow during capture: reserve the
 *     {depth, omega} workspace first (ggt_set_workspace, or one eager call of the same shape), refine with
 *     ggt_refine_depth_static (or after one eager ggt_refine_depth* call of the same shape), leave stage profiling off,
 *     and keep ggt_volume_bind, ggt_splat_reserve and ggt_frame_host (which owns streams and events) outside the capture.
 *   - depth maps hold z-depth in metres (the quantity Eq. 9 compares with z_k); <= 0 means invalid.
 *   - pixel (i, j) has its centre at (i + 0.5, j + 0.5); images are row-major, row 0 on top.
 *   - arithmetic is IEEE fp32 in a fixed operation order (P14), so
 *     results are bit-reproducible and comparable with the oracle on the discrete decisions.
 */
#ifndef GGT_H_
#define GGT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GGT_OK 0
#define GGT_ERR_INVALID_ARG (-1)
#define GGT_ERR_SHAPE (-2)
#define GGT_ERR_UNSUPPORTED (-3)
#define GGT_ERR_CUDA (-4)

#define GGT_F32 0          /* volume storage: {T, W} as 2 x fp32 = 8 B / voxel */
#define GGT_F16 1          /* volume storage: {T, W} as 2 x fp16 = 4 B / voxel (RNE on store) */

#define GGT_OVERWRITE 0u   /* T = sum(w c)/sum(w), W = sum(w)  (Eq. 10, normalised: reading P2) */
#define GGT_ACCUMULATE 1u  /* running average against the stored {T, W} with decay and cap (P9) */

#define GGT_FRAME_RESULTS_ASYNC 0x100u /* ggt_frame_host only, OR-ed into flags: result copies on the context's own stream */

#define GGT_MAX_VIEWS 16
#define GGT_REFINE_STATIC_MAX_CELLS 262144 /* ggt_refine_depth_static: ceil(W/4) * ceil(H/4) at most (e.g. 2048 x 2048) */
#define GGT_MAX_BINS 1024

/* Pinhole camera, no skew / distortion.  x_cam = R p_world + t. */
typedef struct ggt_camera {
    float fx, fy, cx, cy;
    float R[9];            /* row-major */
    float t[3];
    int32_t width, height;
} ggt_camera;

/* Eq. 1 parameters.  Paper: lambda_t = 0.7, beta = 0.6, theta = 0;
 * BASELINE.json:configs[2] adds the dead zone theta = 8/255 (reading P6).
 * Only downscale = 4 and pool = 3 (the paper's values) are implemented: others -> GGT_ERR_UNSUPPORTED. */
typedef struct ggt_refine_params {
    float lambda_t, beta, theta;
    int32_t downscale, pool;
} ggt_refine_params;

/* Volume descriptor.  tau_j = trunc_bins x local bin spacing (reading P3) unless trunc_metric > 0
 * (paper: 0.02 m).  w_window = 7, w_sigma0 = 0.001, w_clip = 0.02 are Eq. 11-12's
 * constants; w_window = 0 gives omega = 1 on valid pixels.  weight_cap / decay: persistent mode. */
typedef struct ggt_volume_desc {
    int32_t width, height, bins;   /* W_t, H_t, D (2 <= D <= GGT_MAX_BINS) */
    const float* z_bins;           /* HOST, D strictly increasing z-depths (metres) */
    float trunc_bins;
    float trunc_metric;
    float w_sigma0, w_clip;
    int32_t w_window;              /* 0 or 7 */
    float weight_cap, decay;
    int32_t dtype;                 /* GGT_F32 | GGT_F16 */
} ggt_volume_desc;

typedef struct ggt_ctx ggt_ctx;
typedef struct ggt_volume ggt_volume;

/* ---- context ------------------------------------------------------------------------------------ */
/* Creates a context on the current CUDA device.  GGT_ERR_CUDA if there is none. */
int ggt_create(ggt_ctx** out);
int ggt_destroy(ggt_ctx* ctx);
/* Text of the last error on this context (or of the last ggt_create failure if ctx == NULL). */
const char* ggt_last_error(const ggt_ctx* ctx);
/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
int64_t ggt_launch_count(const ggt_ctx* ctx);

/* Optional per-stage device timing for bench.py's roofline: when enabled, every call records a pair of
 * CUDA events on the caller's stream around its kernels.  ggt_profile_collect waits for them, writes the
 * summed milliseconds and the number of timed groups per stage into host arrays of GGT_PROFILE_STAGES entries
 * (0 refine, 1 weight maps, 2 integrate main kernel, 3 extract, 4 raymarch kernel) and clears the records. */
#define GGT_PROFILE_STAGES 5
int ggt_profile_enable(ggt_ctx* ctx, int32_t enable);
int ggt_profile_collect(ggt_ctx* ctx, double* host_ms, int64_t* host_count);

/* Test hook (determinism contract, P14): the kernels form 1/w, A/W, sqrt and x/49 with their own
 * branch-free sequences; this runs them on n pairs (dev_a[i], dev_b[i]), b > 0, and ADDS to dev_mismatch[0..3] the
 * number of elements whose reciprocal 1/b, quotient a/b (packed and scalar forms), square root sqrt(b) and quotient
 * b/49 differ in any bit from the IEEE-754 round-to-nearest results (__frcp_rn, __fdiv_rn, __fsqrt_rn).  n even;
 * dev_mismatch: 4 words zeroed by the caller. */
int ggt_selftest_arith(ggt_ctx* ctx, int64_t n, const float* dev_a, const float* dev_b, uint32_t* dev_mismatch,
                       void* stream);

/* ---- workspace for the {depth, omega} maps of Eq. 11-12 ------------------------------------------ */
/* Bytes of device scratch ggt_integrate needs for n_views maps of width x height: 8 B per record of the
 * zero-padded (height+1) x (width+1) {depth, omega} map, each map rounded up to 256 B. */
size_t ggt_workspace_bytes(int32_t n_views, int32_t width, int32_t height);
/* Hands caller-owned device scratch (256-B aligned) to the context.  Without it ggt_integrate grows an internal
 * cudaMalloc'ed buffer, which synchronises the device once per growth; WITH it, a call whose views need more than
 * `bytes` fails with GGT_ERR_SHAPE (the library never replaces a caller's buffer).  NULL hands the job back to the
 * library. */
int ggt_set_workspace(ggt_ctx* ctx, void* dev_workspace, size_t bytes);

/* ---- volume ------------------------------------------------------------------------------------- */
/* Bytes the caller must allocate for a volume: a 256-B-aligned table header (z_j, tau_j) followed by
 * the voxels in the internal layout  T[ceil(D/G)][H_t][W_t][G]  then  W[ceil(D/G)][H_t][W_t][G]  with G = 4 (fp32)
 * or 8 (fp16) bins per 128-bit access (bins are padded to a multiple of G), followed by one
 * 32-bit search range per target ray (written by ggt_integrate*, read by ggt_extract_depth: the first and last group
 * of bins that hold an observed non-positive T).  The storage is opaque: only the ggt_* calls may write it. */
size_t ggt_volume_bytes(const ggt_volume_desc* desc);
/* Binds caller-owned device storage (>= ggt_volume_bytes, 256-B aligned) and uploads the bin tables (a small copy,
 * complete on return whatever stream later calls use).  The storage content is otherwise untouched: call
 * ggt_volume_reset. */
int ggt_volume_bind(ggt_ctx* ctx, const ggt_volume_desc* desc, void* dev_storage, size_t bytes,
                    ggt_volume** out);
int ggt_volume_unbind(ggt_ctx* ctx, ggt_volume* vol);
/* T = 0, W = 0 everywhere. */
int ggt_volume_reset(ggt_ctx* ctx, ggt_volume* vol, void* stream);
/* Canonical export for tests: bin-fastest idx = (v*W_t + u)*D + j, separate fp32 T and W arrays. */
int ggt_volume_export(ggt_ctx* ctx, const ggt_volume* vol, float* dev_T, float* dev_W, void* stream);
/* Copies of the tables the kernels use (host out arrays of D floats; either may be NULL). */
int ggt_volume_tables(const ggt_volume* vol, float* host_z, float* host_tau);

/* ---- step a1-a2: temporal depth refinement of one input view (Eq. 1-2) ----------- */
/* dev_rgb_cur / dev_rgb_prev: uint8, height x width pixels of rgb_pixel_stride (3 or 4) bytes, channels
 * 0..2 = RGB.  dev_rgb_prev == NULL -> first frame: M = 1, state = depth_cur.
 * dev_depth_state: in = refined depth of frame t-1, out = refined depth of frame t (in place).
 * dev_mask_out (optional): fp32 height x width soft mask M.  dev_pooled_out (optional): uint16
 * ceil(H/4) x ceil(W/4) max-pooled block L1 colour difference (integer, exact). */
int ggt_refine_depth(ggt_ctx* ctx, int32_t width, int32_t height, const uint8_t* dev_rgb_cur,
                     const uint8_t* dev_rgb_prev, int32_t rgb_pixel_stride, const float* dev_depth_cur,
                     float* dev_depth_state, float* dev_mask_out, uint16_t* dev_pooled_out,
                     const ggt_refine_params* params, void* stream);

/* ggt_refine_depth for callers that may not allocate device memory (code under stream capture, serving loops, harnesses
 * that forbid cudaMalloc): same arguments, same arithmetic, same result bits, but the quarter-resolution scratch of
 * Eq. 1 lives in a fixed array of GGT_REFINE_STATIC_MAX_CELLS x 2 B = 512 KB inside the library's device
 * image (held by every GPU that loads the library until the process exits) instead of the context's growing buffer.
 * The call makes no cudaMalloc / cudaFree and no other allocating call, and does no stage timing.
 *   - ceil(width/4) * ceil(height/4) > GGT_REFINE_STATIC_MAX_CELLS -> GGT_ERR_SHAPE, nothing launched.
 *   - the array is shared by ALL calls (all contexts, all streams) on a device and keeps the last call's contents; every
 *     cell a call reads is written by that call first, so nothing has to be cleared between calls -- but two calls that
 *     overlap on the GPU (different streams, no ordering between them) race on it: order them on one stream or by events.
 *   - the device address is looked up once per device on the first call made with that device current. */
int ggt_refine_depth_static(ggt_ctx* ctx, int32_t width, int32_t height, const uint8_t* dev_rgb_cur,
                            const uint8_t* dev_rgb_prev, int32_t rgb_pixel_stride, const float* dev_depth_cur,
                            float* dev_depth_state, float* dev_mask_out, uint16_t* dev_pooled_out,
                            const ggt_refine_params* params, void* stream);

/* The same for n_views views of ONE size in two launches (a frame's views at once): every argument of
 * ggt_refine_depth becomes a HOST array of n_views entries (device pointers).  dev_rgb_cur / dev_rgb_prev /
 * dev_mask_out / dev_pooled_out may be NULL as arrays or per entry, with ggt_refine_depth's meaning (a view
 * without dev_rgb_prev gets the first-frame rule).  1 <= n_views <= GGT_MAX_VIEWS. */
int ggt_refine_depth_batch(ggt_ctx* ctx, int32_t n_views, int32_t width, int32_t height,
                           const uint8_t* const* dev_rgb_cur, const uint8_t* const* dev_rgb_prev,
                           int32_t rgb_pixel_stride, const float* const* dev_depth_cur, float* const* dev_depth_state,
                           float* const* dev_mask_out, uint16_t* const* dev_pooled_out,
                           const ggt_refine_params* params, void* stream);

/* ---- steps a3-a6: fuse V depth maps into the target-view TSDF ----------------- */
/* target, views: HOST.  dev_depths: HOST array of n_views DEVICE pointers to fp32 height x width
 * z-depth maps of the corresponding view (<= 0 invalid).  1 <= n_views <= GGT_MAX_VIEWS.
 * target->width/height must equal the volume's.  flags: GGT_OVERWRITE or GGT_ACCUMULATE. */
int ggt_integrate(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                  const ggt_camera* views, const float* const* dev_depths, uint32_t flags, void* stream);

/* Batched novel views (BASELINE.json:configs[4]): n_targets targets of one frame, each with its own volume and
 * its own n_views input views chosen from the n_rig_views views of the frame.  The {depth, omega} maps (Eq. 11-12)
 * of the rig views are computed ONCE and shared by the targets; otherwise exactly n_targets ggt_integrate calls.
 *   vols, targets     HOST arrays of n_targets volume handles / cameras (targets[t] matches vols[t]; the volumes
 *                     share w_sigma0 / w_clip / w_window)
 *   rig_views, dev_depths  HOST arrays of n_rig_views cameras / DEVICE depth pointers, 1 <= n_rig_views <= GGT_MAX_VIEWS
 *   view_index        HOST, n_targets x n_views indices into rig_views (row t = the views of target t, in fusion order) */
int ggt_integrate_batch(ggt_ctx* ctx, int32_t n_targets, ggt_volume* const* vols, const ggt_camera* targets,
                        int32_t n_rig_views, const ggt_camera* rig_views, const float* const* dev_depths,
                        int32_t n_views, const int32_t* view_index, uint32_t flags, void* stream);

/* The batch with the zero-crossing search fused in (ggt_integrate_extract per target): dev_depth / dev_conf / dev_bin
 * are HOST arrays of n_targets DEVICE pointers (arrays or entries may be NULL). */
int ggt_integrate_extract_batch(ggt_ctx* ctx, int32_t n_targets, ggt_volume* const* vols, const ggt_camera* targets,
                                int32_t n_rig_views, const ggt_camera* rig_views, const float* const* dev_depths,
                                int32_t n_views, const int32_t* view_index, uint32_t flags, float* const* dev_depth,
                                float* const* dev_conf, int32_t* const* dev_bin, void* stream);

/* ---- step a7: zero-crossing depth (reading P13) ------------------------------------- */
/* Outputs are fp32 / int32 H_t x W_t; any may be NULL.  Miss: depth 0, conf 0, bin -1. */
int ggt_extract_depth(ggt_ctx* ctx, const ggt_volume* vol, float* dev_depth, float* dev_conf,
                      int32_t* dev_bin, void* stream);

/* ---- fused a3-a7: ggt_integrate that also emits what ggt_extract_depth would, in the same pass ---- */
/* Same volume result as ggt_integrate followed by ggt_extract_depth, without re-reading the volume. */
int ggt_integrate_extract(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                          const ggt_camera* views, const float* const* dev_depths, uint32_t flags,
                          float* dev_depth, float* dev_conf, int32_t* dev_bin, void* stream);

/* ---- the paper's own schedule: volume-free adaptive raymarch ----------------- */
/* PAPER.md:75 "integrates depth along each ray on the fly and, thus, avoids creating an explicit 3D voxel
 * grid"; "We advance along the ray with a step size of 0.8s until a surface intersection is
 * detected.  This is indicated by a change of sign in the value of s.  We subsequently perform three steps
 * of a bisection search to refine the intersection depth."  s(z) is Eq. 9-10 (signs / normalisation:
 * readings P1, P2) with the metric truncation `tau` (paper: 0.02 m) and the weights of Eq. 11-12, evaluated
 * on the fly at target z-depth z; no ggt_volume is involved.  Readings M1-M6:
 *   start at z_near; miss once z > z_far or after max_evals evaluations; advance max(step_scale * s,
 *   min_step) after a positive sample, max(step_scale * tau, min_step) after an unobserved one, min_step
 *   after a non-positive one that has no observed positive predecessor; a crossing is a sample s <= 0 whose
 *   previous sample was observed and positive; n_bisect bisection steps (an unobserved midpoint ends them);
 *   depth = midpoint of the final bracket; conf = sum of weights at its far end; steps = evaluations of s.
 * Paper values: tau 0.02, step_scale 0.8, n_bisect 3, w_sigma0 0.001, w_clip 0.02, w_window 7; min_step and
 * max_evals are this library's (defaults used by the binding: 1e-3 m, 4096). */
typedef struct ggt_raymarch_params {
    float z_near, z_far;           /* metres, z_far > z_near */
    float tau;                     /* > 0 */
    float step_scale;              /* > 0 */
    float min_step;                /* > 0 */
    int32_t max_evals;             /* >= 1 */
    int32_t n_bisect;              /* >= 0 */
    float w_sigma0, w_clip;
    int32_t w_window;              /* 0 or 7 */
} ggt_raymarch_params;

/* target, views: HOST.  dev_depths: HOST array of n_views DEVICE pointers (fp32 height x width z-depth,
 * <= 0 invalid).  Outputs: DEVICE, target->height x target->width, fp32 depth (0 = miss), fp32 conf
 * (0 = miss), int32 steps; any may be NULL.  Uses the context's {depth, omega} workspace like
 * ggt_integrate.  Errors: GGT_ERR_INVALID_ARG (NULLs, parameter ranges), GGT_ERR_SHAPE (sizes, n_views),
 * GGT_ERR_UNSUPPORTED (w_window), GGT_ERR_CUDA. */
int ggt_raymarch_depth(ggt_ctx* ctx, const ggt_camera* target, int32_t n_views, const ggt_camera* views,
                       const float* const* dev_depths, const ggt_raymarch_params* params, float* dev_depth,
                       float* dev_conf, int32_t* dev_steps, void* stream);

/* ---- paper-style temporal fusion: the previous output depth as one more view ---- */
/* PAPER.md:92-96 (Eq. 3): D^t = Raymarch(TSDF({D_k^t}, D^{t-1})); PAPER.md:352-360 (Eq. 13-14): D^{t-1} is fused
 * with the weight  omega_tmp^t = min(beta * omega_acc^t * max(1 - M^t, 0), eta),  omega_acc^t = omega_tmp^{t-1} +
 * sum_k omega_k^{t-1}  (eta = 15; beta "controls the relative contribution of previous frames").
 * ggt_temporal_weight computes omega_tmp^t per pixel of D^{t-1}:
 *   prev_target     HOST, the camera D^{t-1} was rendered from (its own pose: a moving target is handled)
 *   dev_prev_depth  DEVICE fp32 H_p x W_p, the previous output depth (<= 0 = none)
 *   dev_prev_conf   DEVICE fp32 H_p x W_p, omega_acc: the confidence the previous ggt_raymarch_depth* /
 *                   ggt_extract_depth call returned (sum of all fusion weights at the surface point, Eq. 14)
 *   views, dev_masks  the n_views input cameras (HOST) and their fp32 difference masks M_k^t of THIS frame
 *                   (DEVICE, height_k x width_k: ggt_refine_depth's dev_mask_out); 0 <= n_views <= GGT_MAX_VIEWS
 *   M^t (reading F1): the surface point of each pixel of D^{t-1} is projected into every input view (nearest
 *                   pixel) and M^t is the maximum of M_k^t over the views it lands in (0 if none); occlusion is
 *                   not tested.  The paper forward-splats the masks instead.
 *   dev_weight_out  DEVICE fp32 H_p x W_p.
 * The *_weighted calls are ggt_integrate / ggt_raymarch_depth with per-view given weights: dev_weights is a HOST
 * array of n_views DEVICE pointers; entry k NULL -> Eq. 11-12 from the depth map as usual, else the fp32
 * height_k x width_k weights of view k (>= 0) are used as its omega.  dev_weights itself may be NULL.
 * One frame of Eq. 3: ggt_temporal_weight(prev camera, D^{t-1}, conf^{t-1}, ...) -> w; then
 * ggt_raymarch_depth_weighted with views = {inputs..., prev camera}, depths = {..., D^{t-1}}, weights =
 * {NULL..., w}; its dev_conf output is the next frame's omega_acc. */
int ggt_temporal_weight(ggt_ctx* ctx, const ggt_camera* prev_target, const float* dev_prev_depth,
                        const float* dev_prev_conf, int32_t n_views, const ggt_camera* views,
                        const float* const* dev_masks, float beta, float eta, float* dev_weight_out, void* stream);
int ggt_integrate_weighted(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                           const ggt_camera* views, const float* const* dev_depths, const float* const* dev_weights,
                           uint32_t flags, void* stream);
int ggt_raymarch_depth_weighted(ggt_ctx* ctx, const ggt_camera* target, int32_t n_views, const ggt_camera* views,
                                const float* const* dev_depths, const float* const* dev_weights,
                                const ggt_raymarch_params* params, float* dev_depth, float* dev_conf,
                                int32_t* dev_steps, void* stream);

/* ---- forward warping with pixel-sized 3D Gaussians -------------------------------------- */
/* PAPER.md:63-65 (section 3.1): "for each pixel of an input I_k, we use the depth map D_k and pose to determine the 3D
 * position of an isotropic, fully-opaque Gaussian.  The RGB color of each Gaussian is set to the underlying pixel value,
 * and its scale is computed such that its projection in the source image I_k covers a single pixel.  This step produces
 * a set of forward-rendered images along with accumulated opacity of the Gaussians, and depths in the novel view";
 * PAPER.md:362-368 (A.3): the parameters are computed analytically; rendered with the 3D Gaussian
 * splatting rasteriser the paper cites.  Readings S1-S8: 3D standard deviation sigma_px * D / fx of the
 * source camera; EWA projection into the target (2D covariance sigma^2 J J^T + dilation I); alpha = min(0.99, exp(-1/2
 * d^T Sigma'^-1 d)), a Gaussian contributes to a pixel iff alpha >= 1/255; per target pixel the contributors are
 * composited front to back in ascending target depth (ties: ascending source pixel index) until the transmittance
 * would fall below 1e-4; Gaussians with depth <= 0 or target depth < z_cull are dropped.  Paper / rasteriser values:
 * sigma_px 0.5, dilation 0.3, z_cull 0.2.
 *   target, view     HOST cameras (view = the input view whose pixels are splatted; sizes <= 32767)
 *   dev_depth        DEVICE fp32 height x width z-depth of the view (<= 0 invalid), e.g. ggt_refine_depth's state
 *   dev_rgb          DEVICE uint8 height x width x rgb_pixel_stride (3 or 4), may be NULL
 *   dev_mask         DEVICE fp32 height x width (Eq. 1's M_k: ggt_refine_depth's dev_mask_out), may be NULL
 *   dev_out_rgb      DEVICE fp32 [3][H_t][W_t], colour in source units (0..255), premultiplied by opacity, no background
 *   dev_out_alpha    DEVICE fp32 H_t x W_t accumulated opacity 1 - T
 *   dev_out_depth    DEVICE fp32 H_t x W_t opacity-normalised depth (0 where nothing landed)
 *   dev_out_mask     DEVICE fp32 H_t x W_t the mask splatted like a colour channel
 *   dev_out_count    DEVICE int32 H_t x W_t number of Gaussians with alpha >= 1/255 at the pixel (diagnostic)
 * Every output may be NULL.  One call = one view (the paper renders the K views separately).
 * Scratch is owned by the context and grows between calls (cudaMalloc, synchronising once per growth): 32 B per source
 * pixel, 8 B per target pixel and 8 B per list entry; the list capacity is ggt_splat_reserve's, by default 40 entries per
 * source pixel (a dense single surface needs about 20).  If a call needs more entries than the capacity, its outputs
 * are zero and ggt_splat_status reports it: reserve what it asks for and call again.  Domain: views of comparable
 * resolution (the sum of the Gaussians' footprints, in target pixels, must stay below 2^32).
 * Errors: GGT_ERR_INVALID_ARG (NULL cameras / depth, parameter ranges), GGT_ERR_SHAPE (sizes), GGT_ERR_CUDA. */
typedef struct ggt_splat_params {
    float sigma_px;                /* > 0 */
    float dilation;                /* >= 0 */
    float z_cull;                  /* > 0 */
    int32_t reserved;              /* 0 */
} ggt_splat_params;
int ggt_splat_forward(ggt_ctx* ctx, const ggt_camera* target, const ggt_camera* view, const float* dev_depth,
                      const uint8_t* dev_rgb, int32_t rgb_pixel_stride, const float* dev_mask,
                      const ggt_splat_params* params, float* dev_out_rgb, float* dev_out_alpha, float* dev_out_depth,
                      float* dev_out_mask, int32_t* dev_out_count, void* stream);
/* List capacity of later ggt_splat_forward calls, in entries (0 = the default rule). */
int ggt_splat_reserve(ggt_ctx* ctx, int64_t entries);
/* Synchronises `stream`; host_entries_last = list entries the last call produced, host_entries_needed = the largest
 * number of entries any call since the last status query needed but did not have (0 = no call overflowed). */
int ggt_splat_status(ggt_ctx* ctx, int64_t* host_entries_last, int64_t* host_entries_needed, void* stream);
/* Eq. 13 with the paper's own novel-view mask: M^t = the channel-wise maximum of the n_masks
 * splatted masks (ggt_splat_forward's dev_out_mask of each input view, rendered into the camera of D^{t-1});
 * dev_weight_out = min(beta * omega_acc * max(1 - M^t, 0), eta) per pixel, 0 where depth or omega_acc is <= 0.
 *   dev_masks   HOST array of n_masks (1..GGT_MAX_VIEWS) DEVICE pointers, each fp32 n_pixels */
int ggt_temporal_weight_mask(ggt_ctx* ctx, int64_t n_pixels, const float* dev_prev_depth, const float* dev_prev_conf,
                             int32_t n_masks, const float* const* dev_masks, float beta, float eta,
                             float* dev_weight_out, void* stream);

/* ---- network-input geometry features of the guidance depth --------------------- */
/* PAPER.md:374-388 (A.4, items 5-8 of the blending network's input): per input view k and target pixel,
 *   (5) the dot product between the input-view ray direction and the normal of the TSDF depth D^t,
 *   (6) the dot product between the input-view ray direction and the target view direction,
 *   (7) the distance between the input and target cameras, repeated spatially,
 *   (8) the dot product between the input and target viewing directions, repeated spatially.
 * Readings G1-G4: surface point p = D ((u + 0.5 - cx)/fx, (v + 0.5 - cy)/fy, 1) in the target camera;
 * normal = normalised cross product of the central differences of p in u and v (one-sided where only one
 * neighbour has depth, undefined where neither has), oriented towards the camera; ray directions are unit
 * vectors from the camera centres -R^T t to the surface point; viewing directions are the optical axes.
 *   target, views   HOST; 1 <= n_views <= GGT_MAX_VIEWS (only R, t of the views are used)
 *   dev_depth       DEVICE fp32 H_t x W_t guidance depth (ggt_extract_depth / ggt_raymarch_depth output, <= 0 none)
 *   dev_features    DEVICE fp32 [4 K][H_t][W_t], planar: channels [0, K) item 5, [K, 2K) item 6, [2K, 3K) item 7,
 *                   [3K, 4K) item 8; items 5 and 6 are 0 where the depth or the normal is undefined. */
int ggt_guidance_features(ggt_ctx* ctx, const ggt_camera* target, const float* dev_depth, int32_t n_views,
                          const ggt_camera* views, float* dev_features, void* stream);

/* ---- end-to-end frame from HOST buffers (bench.py "e2e") ----------------------------------------- */
/* One whole frame through the three steps with host<->device copies inside the call, enqueued without
 * synchronising: kernels on `stream`; the input uploads and the result copies on two streams owned by the context,
 * ordered against `stream` with events.  Within a frame each view's refine kernels and weight map start as soon as
 * that view's upload has landed, and the fused integrate / extract kernel runs as four row slices whose results
 * travel while the next slice computes; consecutive calls overlap frame n + 1's uploads with frame n's kernels.  The host input buffers must stay valid until `stream` has passed this call's kernels; the results
 * are complete when `stream` is synchronised.  All n_views views must have the same width x height.
 *   host_rgb_cur[k]   uint8 HxWx3 colour of view k at this frame (host; array or entry may be NULL -> that
 *                     view is not refined, its depth is used as is); params NULL also disables refinement.
 *   host_depth_cur[k] fp32 HxW z-depth of view k (host).
 *   slots[k]          which history slot (0 <= slot < n_slots, e.g. the rig camera index) view k uses: the
 *                     slot keeps the previous colour image and the refined-depth state in `dev_staging`.
 *   host_slot_state   n_slots words, in/out, zero-initialised by the caller before the first frame
 *                     (bit 0: slot has history, bit 1: ping-pong parity).  A slot without history gets the
 *                     first-frame rule (M = 1).
 *   dev_staging       caller-owned device memory, >= ggt_frame_staging_bytes, 256-B aligned.
 *   host_depth / host_conf  fp32 H_t x W_t results (host; either may be NULL).
 *   flags             GGT_OVERWRITE or GGT_ACCUMULATE, optionally | GGT_FRAME_RESULTS_ASYNC: the device -> host result
 *                     copies then run on a stream of the context, out of two alternating sets of device buffers, so that the
 *                     next call's kernels do not wait behind them on `stream`; the results of all such calls made so far
 *                     are on the host once a stream that ggt_frame_host_results_wait(ctx, that stream) was called on has
 *                     been synchronised.  The host result buffers of two consecutive calls must differ.
 * Slots: the slots of one call must be distinct (GGT_ERR_INVALID_ARG otherwise).  host_slot_state is updated only when
 * the whole call has been enqueued successfully.  A slot's history is whatever frame it last took part in: callers that
 * want Eq. 2 against frame t-1 for every rig camera (as the paper refines all N views every frame) pass
 * every rig view each frame; a camera that re-enters after a gap is blended against its older state. */
size_t ggt_frame_staging_bytes(const ggt_volume_desc* desc, int32_t n_slots, int32_t n_views, int32_t width,
                               int32_t height);
int ggt_frame_host(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                   const ggt_camera* views, const uint8_t* const* host_rgb_cur, const float* const* host_depth_cur,
                   const int32_t* slots, int32_t n_slots, uint32_t* host_slot_state,
                   const ggt_refine_params* params, uint32_t flags, void* dev_staging, size_t staging_bytes,
                   float* host_depth, float* host_conf, void* stream);
/* Makes `stream` wait (on the device) for the result copies of every GGT_FRAME_RESULTS_ASYNC call made so far. */
int ggt_frame_host_results_wait(ggt_ctx* ctx, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* GGT_H_ */
