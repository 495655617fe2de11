// ggt_internal.h — private declarations of the CUDA path (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/ggt.h"

// ---- device-side parameter blocks (passed by value as __grid_constant__ kernel parameters) --------
struct GgtViewParams {      // (x, y, w) = z * H_k (uc, vc, 1)^T + e_k,  H_k = K_k R_k R_t^T K_t^{-1},  e_k = K_k (t_k - R_k R_t^T t_t)
    float nh[6];           // rows 0-1 of H_k, NEGATED (the kernel carries -x, -y and -1/w: see ggt_integrate.cu)
    float h2[3];           // row 2 of H_k
    float ne[2];           // -e_k[0], -e_k[1]
    float e2;              // e_k[2]
    const float2* map;     // interleaved {depth (0 if invalid), omega (0 if invalid)}, height x width
    int32_t width, height;
    uint32_t stride;       // records per map row = width + 1 (zero padding column)
    int32_t pad_;
};

struct GgtIntegrateParams {
    int32_t Wt, Ht, D;     // target width / height, bins
    int32_t n_views;
    int32_t n_groups;      // ceil(D / G)
    int32_t accumulate;    // 0 overwrite, 1 running average
    int32_t same_size;     // 1 if all views have the same width x height
    int32_t shared_w;      // 1 if additionally H_k and e_k[2] are bit-identical in all views (n_views >= 2)
    int32_t row0, row1;    // target rows [row0, row1) this launch covers (ggt_frame_host slices a frame; else 0, Ht)
    float decay, cap;
    unsigned long long plane;   // Wt * Ht: 128-bit words per group of the volume
    const float* tables;   // device: z[0..Dpad) then tau[0..Dpad), Dpad = n_groups * G
    void* voxels;          // device: T[n_groups][Ht][Wt][G] then W[n_groups][Ht][Wt][G]
    uint32_t* hint;        // device: per ray, first | (last + 1) << 16 of the groups holding an observed bin with T <= 0
    float* depth;          // fused extract outputs (may be null)
    float* conf;
    int32_t* bin;
    GgtViewParams v[GGT_MAX_VIEWS];
};

struct GgtRaymarchParams {  // the paper's own schedule: one thread per target ray, no volume
    int32_t Wt, Ht, n_views, max_evals, n_bisect;
    int32_t shared_w;      // row 2 of H_k and e_k[2] bit-identical in all views (n_views >= 2)
    float z_near, z_far, tau, step_scale, min_step;
    float* depth;          // outputs (each may be null)
    float* conf;
    int32_t* steps;
    GgtViewParams v[GGT_MAX_VIEWS];
};

struct GgtMaskView {        // ggt_temporal_weight: previous-target pixel/depth -> view k homogeneous pixel, and view k's mask
    float h[9];            // H_k = K_k R_k R_p^T K_p^-1
    float e[3];            // e_k = K_k (t_k - R_k R_p^T t_p)
    const float* mask;     // fp32 height x width (Eq. 1's M_k^t)
    int32_t width, height;
};

struct GgtTemporalParams {
    int32_t Wt, Ht, n_views, pad_;
    float beta, eta;
    const float* prev_depth;
    const float* prev_conf;
    float* out;
    GgtMaskView v[GGT_MAX_VIEWS];
};

struct GgtRefineView {
    const uint8_t* rgb_cur;
    const uint8_t* rgb_prev;
    const float* depth_cur;
    float* depth_state;
    float* mask_out;       // optional
    uint16_t* pooled_out;  // optional
    uint16_t* cq;          // quarter-res block differences (context scratch)
};

struct GgtRefineViews {     // views of one ggt_refine_depth(_batch) call that have a previous colour image
    int32_t n, pad_;
    GgtRefineView v[GGT_MAX_VIEWS];
};

struct GgtFeatureView {
    float C[3];            // camera centre -R_k^T t_k
    float dist;            // |C_k - C_t|
    float axes;            // optical axes: R_k row 2 . R_t row 2
};

struct GgtFeatureParams {   // ggt_guidance_features (A.4 items 5-8)
    int32_t W, H, n_views;
    int32_t fast_ok;       // fx, fy mid-range: the branch-free division is exact for (uc - cx) / fx
    float fx, fy, cx, cy;
    float R[9], t[3], Ct[3];
    const float* depth;
    float* out;            // [4 K][H][W]
    GgtFeatureView v[GGT_MAX_VIEWS];
};

struct GgtWeightView {
    const float* depth;    // fp32 height x width, <= 0 (or NaN) = invalid
    const float* weight;   // null: omega from Eq. 11-12; else the view's given per-pixel weights (e.g. Eq. 13)
    float2* out;           // (height + 1) x (width + 1) records {depth, omega}
    int32_t width, height;
};

struct GgtWeightParams {    // all views of one ggt_integrate call: one launch, blockIdx.z = view
    int32_t n_views, window;
    float sigma0, c2;      // c2 = clip * clip (one fp32 multiply, as the oracle states it)
    int32_t fast_ok;       // sigma0 within [1e-20, 1e20]: the branch-free division / sqrt fast paths are exact
    int32_t pad_;
    GgtWeightView v[GGT_MAX_VIEWS];
};

struct GgtSplatParams {     // ggt_splat_forward: one input view's pixel-sized Gaussians into the target
    int32_t W, H, Wt, Ht;  // source view / target size
    int32_t rgb_stride;    // bytes per source pixel of rgb (3 or 4)
    uint32_t capacity;     // list entries the scratch holds
    float h[9], e[3];      // source pixel / depth -> target homogeneous pixel: (x, y, w) = D * h (uc, vc, 1)^T + e
    float fx_t, fy_t, cx_t, cy_t, fx_s;
    float sigma_px, dilation, z_cull;
    const float* depth;    // source depth, fp32 H x W
    const uint8_t* rgb;    // source colour (may be null)
    const float* mask;     // source mask (may be null)
    float* gauss;          // scratch: 8 floats per source pixel
    uint32_t* counts;      // scratch: per target pixel
    uint32_t* pos;         // scratch: per target pixel (list start, then end)
    uint32_t* block_sums;  // scratch: scan
    uint32_t* total;       // scratch: 1 word, number of list entries of this call
    uint32_t* overflow;    // context: max entries ever needed when that exceeded the capacity (0 = never)
    uint2* entries;        // scratch: {depth bits, source index}
    float* out_rgb;        // [3][Ht][Wt] (may be null)
    float* out_alpha;
    float* out_depth;
    float* out_mask;
    int32_t* out_count;
};

struct GgtMaskList {        // ggt_temporal_weight_mask: the K splatted masks whose channel-wise maximum is M^t
    int32_t n, pad_;
    const float* m[GGT_MAX_VIEWS];
};

struct GgtExtractParams {
    int32_t Wt, Ht, D, n_groups;
    const float* tables;
    const void* voxels;
    const uint32_t* hint;  // per ray search range written by k_integrate (0 after a reset: nothing to find)
    float* depth;
    float* conf;
    int32_t* bin;
};

// ---- host objects -----------------------------------------------------------------------------------
struct ggt_ctx {
    int device = 0;
    int sm_count = 148;
    std::string err;
    int64_t launches = 0;
    void* ws = nullptr;            // {depth, omega} maps scratch
    size_t ws_bytes = 0;
    bool ws_owned = false;
    uint16_t* cq = nullptr;        // quarter-res block differences of ggt_refine_depth (context-owned)
    size_t cq_bytes = 0;
    // ggt_splat_forward scratch (context-owned, grown between calls): Gaussian parameters, per-pixel counts / positions,
    // scan sums, the per-pixel lists; `splat_flags` = {total entries of the last call, overflow high-water mark}
    void* splat_ws = nullptr;
    size_t splat_ws_bytes = 0;
    size_t splat_entries = 0;      // list capacity in entries (0 = automatic: 40 per source pixel)
    uint32_t* splat_flags = nullptr;
    // ggt_frame_host: host->device copies run on an internal stream so that the next frame's inputs upload while
    // this frame's integrate / extract kernels run.  ev_inputs_free is recorded on the caller's stream behind the last
    // kernel that reads the uploaded depth / colour buffers (the last view's refine kernel, or its weight map).
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_inputs_free = nullptr;
    bool inputs_free_pending = false;
    cudaEvent_t ev_view[GGT_MAX_VIEWS] = {};   // ggt_frame_host: view k's uploads have landed
    bool weights_prelaunched = false;          // ggt_frame_host launched the weight maps view by view already
    // GGT_FRAME_RESULTS_ASYNC: the device -> host result copies run on d2h_stream out of two alternating sets of device
    // result buffers, so the next frame's kernels do not queue behind them on the caller's stream
    cudaStream_t d2h_stream = nullptr;
    cudaEvent_t ev_kernels_done = nullptr, ev_d2h_done[2] = {nullptr, nullptr};
    bool d2h_pending[2] = {false, false};
    int result_set = 0;
    // optional per-stage device timing (ggt_profile_enable): pairs of events around each kernel group
    bool prof = false;
    struct ProfRec { int stage; cudaEvent_t a, b; };
    std::vector<ProfRec> prof_pool;
    size_t prof_used = 0;
};

enum { GGT_STAGE_REFINE = 0, GGT_STAGE_WEIGHT = 1, GGT_STAGE_INTEGRATE = 2, GGT_STAGE_EXTRACT = 3, GGT_STAGE_RAYMARCH = 4, GGT_N_STAGES = 5 };

struct ggt_volume {
    ggt_volume_desc desc;
    std::vector<float> z, tau;     // host copies of the tables (D entries)
    int32_t group = 2;             // G: bins per 128-bit access
    int32_t n_groups = 0;
    size_t header_bytes = 0;
    size_t voxel_bytes = 0;
    float* dev_tables = nullptr;   // inside the caller's storage
    void* dev_voxels = nullptr;    // inside the caller's storage
    uint32_t* dev_hints = nullptr; // inside the caller's storage, after the voxels: one search range per ray
    size_t hint_bytes = 0;
};

static inline int ggt_group_of(int dtype) { return dtype == GGT_F16 ? 8 : 4; }

// ---- kernel launchers (each returns cudaError_t of the launch) ----------------------------------------
cudaError_t ggt_launch_refine(int W, int H, const GgtRefineViews& tab, int stride, float lambda_t, float beta, float theta,
                              cudaStream_t st, int* n_launches);
cudaError_t ggt_refine_static_scratch(uint16_t** ptr);   // ggt_refine.cu: address of the fixed-size scratch on this device
cudaError_t ggt_launch_first_frame(int W, int H, const float* depth_cur, float* depth_state, float* mask_out, cudaStream_t st);
cudaError_t ggt_launch_weight_maps(const GgtWeightParams& p, cudaStream_t st);
cudaError_t ggt_launch_integrate(const GgtIntegrateParams& p, int dtype, bool fused, int sm_count, cudaStream_t st);
cudaError_t ggt_launch_temporal_weight(const GgtTemporalParams& p, cudaStream_t st);
cudaError_t ggt_launch_features(const GgtFeatureParams& p, cudaStream_t st);
cudaError_t ggt_launch_raymarch(const GgtRaymarchParams& p, cudaStream_t st);
cudaError_t ggt_launch_splat(const GgtSplatParams& p, cudaStream_t st, int* n_launches);
cudaError_t ggt_launch_temporal_weight_mask(size_t n, const float* prev_depth, const float* prev_conf, const GgtMaskList& masks,
                                            float beta, float eta, float* out, cudaStream_t st);
cudaError_t ggt_launch_extract(const GgtExtractParams& p, int dtype, cudaStream_t st);
cudaError_t ggt_launch_export(const GgtExtractParams& p, int dtype, float* T, float* W, cudaStream_t st);
cudaError_t ggt_launch_selftest_arith(long long n, const float* a, const float* b, unsigned* mismatch, cudaStream_t st);
