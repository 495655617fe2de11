// ggt_api.cu — the C ABI declared in include/ggt.h: argument validation, host-side camera algebra,
// workspace handling and kernel launches.  No compute happens on the host beyond the 12 floats per view of
// the relative transform and the bin tables; there is no CPU fallback.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "ggt_internal.h"

namespace {

std::string g_create_error;

int fail(ggt_ctx* ctx, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf; else g_create_error = buf;
    return code;
}

int cuda_fail(ggt_ctx* ctx, cudaError_t e, const char* what) {
    return fail(ctx, GGT_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// RAII pair of events around one kernel group when ggt_profile_enable is on (no-op otherwise).
struct StageTimer {
    ggt_ctx* c; cudaStream_t st; ggt_ctx::ProfRec* r = nullptr;
    StageTimer(ggt_ctx* ctx, int stage, cudaStream_t s) : c(ctx), st(s) {
        if (!c->prof) return;
        if (c->prof_used == c->prof_pool.size()) {
            ggt_ctx::ProfRec n; n.stage = stage;
            if (cudaEventCreate(&n.a) != cudaSuccess || cudaEventCreate(&n.b) != cudaSuccess) return;
            c->prof_pool.push_back(n);
        }
        r = &c->prof_pool[c->prof_used++];
        r->stage = stage;
        cudaEventRecord(r->a, st);
    }
    ~StageTimer() { if (r) cudaEventRecord(r->b, st); }
};

// Relative transform of PAPER.md:331 in double, rounded once to float:
//   p_world = R_t^T (z K_t^{-1} (uc, vc, 1)^T - t_t);  (x, y, w) = K_k (R_k p_world + t_k)
//   => (x, y, w) = z * Hm (uc, vc, 1)^T + e  with  Hm = K_k R_k R_t^T K_t^{-1},  e = K_k (t_k - R_k R_t^T t_t).
// Products are plain left-to-right 3-term sums (DESIGN.md fixes the order so that two independent
// implementations round identically).
void relative_transform(const ggt_camera& tg, const ggt_camera& vw, float* h, float* e) {
    double RkRtT[9];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            RkRtT[3 * r + c] = (double)vw.R[3 * r] * (double)tg.R[3 * c] + (double)vw.R[3 * r + 1] * (double)tg.R[3 * c + 1] +
                               (double)vw.R[3 * r + 2] * (double)tg.R[3 * c + 2];
    const double K[9] = {vw.fx, 0.0, vw.cx, 0.0, vw.fy, vw.cy, 0.0, 0.0, 1.0};
    const double fx = tg.fx, fy = tg.fy, cx = tg.cx, cy = tg.cy;
    const double Ki[9] = {1.0 / fx, 0.0, -cx / fx, 0.0, 1.0 / fy, -cy / fy, 0.0, 0.0, 1.0};
    double KR[9], Hm[9];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            KR[3 * r + c] = K[3 * r] * RkRtT[c] + K[3 * r + 1] * RkRtT[3 + c] + K[3 * r + 2] * RkRtT[6 + c];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            Hm[3 * r + c] = KR[3 * r] * Ki[c] + KR[3 * r + 1] * Ki[3 + c] + KR[3 * r + 2] * Ki[6 + c];
    double d[3];
    for (int r = 0; r < 3; ++r)
        d[r] = (double)vw.t[r] - (RkRtT[3 * r] * (double)tg.t[0] + RkRtT[3 * r + 1] * (double)tg.t[1] +
                                  RkRtT[3 * r + 2] * (double)tg.t[2]);
    for (int r = 0; r < 3; ++r) e[r] = (float)(K[3 * r] * d[0] + K[3 * r + 1] * d[1] + K[3 * r + 2] * d[2]);
    for (int i = 0; i < 9; ++i) h[i] = (float)Hm[i];
}

int check_desc(ggt_ctx* ctx, const ggt_volume_desc* d) {
    if (!d) return fail(ctx, GGT_ERR_INVALID_ARG, "volume descriptor is NULL");
    if (d->width <= 0 || d->height <= 0) return fail(ctx, GGT_ERR_SHAPE, "volume size %dx%d", d->width, d->height);
    if (d->width > (1 << 20) || d->height > (1 << 20)) return fail(ctx, GGT_ERR_SHAPE, "volume too large");
    if (d->bins < 2 || d->bins > GGT_MAX_BINS) return fail(ctx, GGT_ERR_SHAPE, "bins %d not in [2, %d]", d->bins, GGT_MAX_BINS);
    if (d->dtype != GGT_F32 && d->dtype != GGT_F16) return fail(ctx, GGT_ERR_UNSUPPORTED, "dtype %d", d->dtype);
    if (d->w_window != 0 && d->w_window != 7) return fail(ctx, GGT_ERR_UNSUPPORTED, "w_window %d (0 or 7)", d->w_window);
    return GGT_OK;
}

size_t header_bytes_of(const ggt_volume_desc* d) {
    const int G = ggt_group_of(d->dtype);
    const int ng = (d->bins + G - 1) / G;
    return align_up((size_t)2 * ng * G * sizeof(float), 256);
}

size_t voxel_bytes_of(const ggt_volume_desc* d) {
    const int G = ggt_group_of(d->dtype);
    const int ng = (d->bins + G - 1) / G;
    return align_up((size_t)ng * d->width * d->height * 32, 256);     // one 128-bit word per group and pixel in each of the two planes
}

size_t hint_bytes_of(const ggt_volume_desc* d) { return align_up((size_t)d->width * d->height * sizeof(uint32_t), 256); }

}  // namespace

extern "C" {

int ggt_create(ggt_ctx** out) {
    if (!out) return fail(nullptr, GGT_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
        cudaGetLastError();
        return fail(nullptr, GGT_ERR_CUDA, "no CUDA device (%s): the ggt library has no CPU path",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    ggt_ctx* c = new (std::nothrow) ggt_ctx();
    if (!c) return fail(nullptr, GGT_ERR_INVALID_ARG, "out of host memory");
    cudaGetDevice(&c->device);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device);
    int major = 0;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, c->device);
    if (major != 10) {
        delete c;
        return fail(nullptr, GGT_ERR_UNSUPPORTED, "device compute capability %d.x: this library is built for sm_100a only", major);
    }
    *out = c;
    return GGT_OK;
}

int ggt_destroy(ggt_ctx* ctx) {
    if (!ctx) return GGT_OK;
    ggt_ctx* c = ctx;
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    if (c->cq) cudaFree(c->cq);
    if (c->splat_ws) cudaFree(c->splat_ws);
    if (c->splat_flags) cudaFree(c->splat_flags);
    for (auto& r : c->prof_pool) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    if (c->ev_inputs_free) cudaEventDestroy(c->ev_inputs_free);
    for (int i = 0; i < GGT_MAX_VIEWS; ++i) if (c->ev_view[i]) cudaEventDestroy(c->ev_view[i]);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->ev_kernels_done) cudaEventDestroy(c->ev_kernels_done);
    for (int i = 0; i < 2; ++i) if (c->ev_d2h_done[i]) cudaEventDestroy(c->ev_d2h_done[i]);
    if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
    delete c;
    return GGT_OK;
}

const char* ggt_last_error(const ggt_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int64_t ggt_launch_count(const ggt_ctx* ctx) { return ctx ? ctx->launches : 0; }

int ggt_profile_enable(ggt_ctx* ctx, int32_t enable) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    ctx->prof = enable != 0;
    ctx->prof_used = 0;
    return GGT_OK;
}

int ggt_profile_collect(ggt_ctx* ctx, double* host_ms, int64_t* host_count) {
    if (!ctx || !host_ms || !host_count) return GGT_ERR_INVALID_ARG;
    for (int i = 0; i < GGT_N_STAGES; ++i) { host_ms[i] = 0.0; host_count[i] = 0; }
    for (size_t i = 0; i < ctx->prof_used; ++i) {
        ggt_ctx::ProfRec& r = ctx->prof_pool[i];
        cudaError_t e = cudaEventSynchronize(r.b);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.a, r.b);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_profile_collect");
        host_ms[r.stage] += ms;
        host_count[r.stage] += 1;
    }
    ctx->prof_used = 0;
    return GGT_OK;
}

int ggt_selftest_arith(ggt_ctx* ctx, int64_t n, const float* dev_a, const float* dev_b, uint32_t* dev_mismatch, void* stream) {
    if (!ctx || !dev_a || !dev_b || !dev_mismatch || n < 0) return GGT_ERR_INVALID_ARG;
    cudaError_t e = ggt_launch_selftest_arith(n, dev_a, dev_b, dev_mismatch, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_selftest_arith");
    ctx->launches += 1;
    return GGT_OK;
}

size_t ggt_workspace_bytes(int32_t n_views, int32_t width, int32_t height) {
    if (n_views <= 0 || width <= 0 || height <= 0) return 0;
    return (size_t)n_views * align_up(((size_t)width + 1) * ((size_t)height + 1) * sizeof(float2), 256);
}

int ggt_set_workspace(ggt_ctx* ctx, void* dev_workspace, size_t bytes) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (((uintptr_t)dev_workspace & 255) != 0) return fail(ctx, GGT_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    if (ctx->ws_owned && ctx->ws) cudaFree(ctx->ws);
    ctx->ws = dev_workspace;
    ctx->ws_bytes = dev_workspace ? bytes : 0;
    ctx->ws_owned = false;
    return GGT_OK;
}

size_t ggt_volume_bytes(const ggt_volume_desc* desc) {
    if (!desc || desc->width <= 0 || desc->height <= 0 || desc->bins < 2) return 0;
    return header_bytes_of(desc) + voxel_bytes_of(desc) + hint_bytes_of(desc);
}

int ggt_volume_bind(ggt_ctx* ctx, const ggt_volume_desc* desc, void* dev_storage, size_t bytes, ggt_volume** out) {
    if (!ctx || !out) return GGT_ERR_INVALID_ARG;
    *out = nullptr;
    int rc = check_desc(ctx, desc);
    if (rc != GGT_OK) return rc;
    if (!desc->z_bins) return fail(ctx, GGT_ERR_INVALID_ARG, "z_bins is NULL");
    if (!dev_storage || ((uintptr_t)dev_storage & 255) != 0) return fail(ctx, GGT_ERR_INVALID_ARG, "storage NULL or not 256-byte aligned");
    if (bytes < ggt_volume_bytes(desc)) return fail(ctx, GGT_ERR_SHAPE, "storage %zu B < required %zu B", bytes, ggt_volume_bytes(desc));
    for (int j = 0; j < desc->bins; ++j) {
        if (!(desc->z_bins[j] > 0.0f) || (j > 0 && !(desc->z_bins[j] > desc->z_bins[j - 1])))
            return fail(ctx, GGT_ERR_INVALID_ARG, "z_bins must be positive and strictly increasing (bin %d)", j);
    }
    if (!(desc->trunc_metric > 0.0f) && !(desc->trunc_bins > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "no truncation distance given");
    ggt_volume* v = new (std::nothrow) ggt_volume();
    if (!v) return fail(ctx, GGT_ERR_INVALID_ARG, "out of host memory");
    v->desc = *desc;
    const int D = desc->bins;
    v->z.assign(desc->z_bins, desc->z_bins + D);
    v->desc.z_bins = v->z.data();
    v->tau.resize(D);
    // tau_j = trunc_bins x local spacing, one-sided at the ends (reading P3), in double then float
    for (int j = 0; j < D; ++j) {
        double sp;
        if (j == 0) sp = (double)v->z[1] - (double)v->z[0];
        else if (j == D - 1) sp = (double)v->z[D - 1] - (double)v->z[D - 2];
        else sp = ((double)v->z[j + 1] - (double)v->z[j - 1]) / 2.0;
        v->tau[j] = desc->trunc_metric > 0.0f ? desc->trunc_metric : (float)((double)desc->trunc_bins * sp);
    }
    v->group = ggt_group_of(desc->dtype);
    v->n_groups = (D + v->group - 1) / v->group;
    v->header_bytes = header_bytes_of(desc);
    v->voxel_bytes = voxel_bytes_of(desc);
    v->dev_tables = static_cast<float*>(dev_storage);
    v->dev_voxels = static_cast<char*>(dev_storage) + v->header_bytes;
    v->hint_bytes = hint_bytes_of(desc);
    v->dev_hints = reinterpret_cast<uint32_t*>(static_cast<char*>(dev_storage) + v->header_bytes + v->voxel_bytes);
    const int Dpad = v->n_groups * v->group;
    std::vector<float> tab(2 * (size_t)Dpad);
    for (int j = 0; j < Dpad; ++j) {
        // bins >= D pad the last 128-bit group: z repeats the last plane, tau = -1e30 puts every sample of a padded
        // bin behind the cut (s < -tau always), so the padding stays unobserved (T = 0, W = 0) whatever the geometry
        tab[j] = v->z[j < D ? j : D - 1];
        tab[Dpad + j] = j < D ? v->tau[j] : -1e30f;
    }
    // pageable source: cudaMemcpy may return while the DMA is still in flight, and the kernels that read the tables run on
    // the caller's (possibly non-blocking) streams, so wait for the legacy stream the copy ran on
    cudaError_t e = cudaMemcpy(v->dev_tables, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
    if (e != cudaSuccess) { delete v; return cuda_fail(ctx, e, "upload of bin tables"); }
    *out = v;
    return GGT_OK;
}

int ggt_volume_unbind(ggt_ctx*, ggt_volume* vol) {
    delete vol;
    return GGT_OK;
}

int ggt_volume_reset(ggt_ctx* ctx, ggt_volume* vol, void* stream) {
    if (!ctx || !vol) return GGT_ERR_INVALID_ARG;
    // voxels and, right behind them, the per-ray search ranges (0 = empty: an all-zero volume has no crossing)
    cudaError_t e = cudaMemsetAsync(vol->dev_voxels, 0, vol->voxel_bytes + vol->hint_bytes, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "volume reset");
    ctx->launches += 1;
    return GGT_OK;
}

static GgtExtractParams extract_params(const ggt_volume* vol) {
    GgtExtractParams p;
    p.Wt = vol->desc.width; p.Ht = vol->desc.height; p.D = vol->desc.bins; p.n_groups = vol->n_groups;
    p.tables = vol->dev_tables; p.voxels = vol->dev_voxels; p.hint = vol->dev_hints;
    p.depth = nullptr; p.conf = nullptr; p.bin = nullptr;
    return p;
}

int ggt_volume_export(ggt_ctx* ctx, const ggt_volume* vol, float* dev_T, float* dev_W, void* stream) {
    if (!ctx || !vol || !dev_T || !dev_W) return GGT_ERR_INVALID_ARG;
    cudaError_t e = ggt_launch_export(extract_params(vol), vol->desc.dtype, dev_T, dev_W, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "volume export");
    ctx->launches += 1;
    return GGT_OK;
}

int ggt_volume_tables(const ggt_volume* vol, float* host_z, float* host_tau) {
    if (!vol) return GGT_ERR_INVALID_ARG;
    if (host_z) memcpy(host_z, vol->z.data(), vol->z.size() * sizeof(float));
    if (host_tau) memcpy(host_tau, vol->tau.data(), vol->tau.size() * sizeof(float));
    return GGT_OK;
}

int ggt_refine_depth_batch(ggt_ctx* ctx, int32_t n_views, int32_t width, int32_t height,
                           const uint8_t* const* dev_rgb_cur, const uint8_t* const* dev_rgb_prev,
                           int32_t rgb_pixel_stride, const float* const* dev_depth_cur, float* const* dev_depth_state,
                           float* const* dev_mask_out, uint16_t* const* dev_pooled_out,
                           const ggt_refine_params* params, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    ggt_ctx* c = ctx;
    if (n_views < 1 || n_views > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_views %d not in [1, %d]", n_views, GGT_MAX_VIEWS);
    if (width <= 0 || height <= 0) return fail(ctx, GGT_ERR_SHAPE, "image size %dx%d", width, height);
    if (!dev_depth_cur || !dev_depth_state || !params) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL depth / params pointer");
    if (rgb_pixel_stride != 3 && rgb_pixel_stride != 4) return fail(ctx, GGT_ERR_INVALID_ARG, "rgb_pixel_stride %d (3 or 4)", rgb_pixel_stride);
    if (params->downscale != 4 || params->pool != 3) return fail(ctx, GGT_ERR_UNSUPPORTED, "only downscale 4 / pool 3 (PAPER.md:81) are implemented");
    if (!(params->lambda_t > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "lambda_t must be > 0");
    const size_t cq_one = align_up((size_t)((width + 3) / 4) * ((height + 3) / 4) * sizeof(uint16_t), 256);
    GgtRefineViews tab;
    memset(&tab, 0, sizeof tab);
    for (int k = 0; k < n_views; ++k) {
        if (!dev_depth_cur[k] || !dev_depth_state[k]) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL depth pointer of view %d", k);
        const uint8_t* rc = dev_rgb_cur ? dev_rgb_cur[k] : nullptr;
        const uint8_t* rp = dev_rgb_prev ? dev_rgb_prev[k] : nullptr;
        if (rp && !rc) return fail(ctx, GGT_ERR_INVALID_ARG, "rgb_prev given without rgb_cur (view %d)", k);
        if (!rp) continue;
        GgtRefineView& v = tab.v[tab.n++];
        v.rgb_cur = rc; v.rgb_prev = rp; v.depth_cur = dev_depth_cur[k]; v.depth_state = dev_depth_state[k];
        v.mask_out = dev_mask_out ? dev_mask_out[k] : nullptr;
        v.pooled_out = dev_pooled_out ? dev_pooled_out[k] : nullptr;
    }
    if (tab.n > 0) {
        const size_t need = cq_one * tab.n;
        if (c->cq_bytes < need) {
            if (c->cq) cudaFree(c->cq);
            c->cq = nullptr; c->cq_bytes = 0;
            cudaError_t e = cudaMalloc(&c->cq, need);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "scratch for block differences");
            c->cq_bytes = need;
        }
        for (int i = 0; i < tab.n; ++i) tab.v[i].cq = reinterpret_cast<uint16_t*>(reinterpret_cast<char*>(c->cq) + cq_one * i);
    }
    cudaStream_t st = (cudaStream_t)stream;
    StageTimer tm(ctx, GGT_STAGE_REFINE, st);
    for (int k = 0; k < n_views; ++k) {                         // views without history: first-frame rule (M = 1)
        if (dev_rgb_prev && dev_rgb_prev[k]) continue;
        cudaError_t e = ggt_launch_first_frame(width, height, dev_depth_cur[k], dev_depth_state[k],
                                               dev_mask_out ? dev_mask_out[k] : nullptr, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_refine_depth first-frame launch");
        ctx->launches += 1;
    }
    if (tab.n > 0) {
        int n = 0;
        cudaError_t e = ggt_launch_refine(width, height, tab, rgb_pixel_stride, params->lambda_t, params->beta, params->theta, st, &n);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_refine_depth launch");
        ctx->launches += n;
    }
    return GGT_OK;
}

int ggt_refine_depth(ggt_ctx* ctx, int32_t width, int32_t height, const uint8_t* dev_rgb_cur,
                     const uint8_t* dev_rgb_prev, int32_t rgb_pixel_stride, const float* dev_depth_cur,
                     float* dev_depth_state, float* dev_mask_out, uint16_t* dev_pooled_out,
                     const ggt_refine_params* params, void* stream) {
    return ggt_refine_depth_batch(ctx, 1, width, height, &dev_rgb_cur, &dev_rgb_prev, rgb_pixel_stride, &dev_depth_cur,
                                  &dev_depth_state, &dev_mask_out, &dev_pooled_out, params, stream);
}

// ggt_refine_depth with the block-difference scratch in the library's fixed device array (ggt_refine.cu): no allocation
// of any kind on this path, and no StageTimer (its event pool grows on demand).
int ggt_refine_depth_static(ggt_ctx* ctx, int32_t width, int32_t height, const uint8_t* dev_rgb_cur,
                            const uint8_t* dev_rgb_prev, int32_t rgb_pixel_stride, const float* dev_depth_cur,
                            float* dev_depth_state, float* dev_mask_out, uint16_t* dev_pooled_out,
                            const ggt_refine_params* params, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (width <= 0 || height <= 0) return fail(ctx, GGT_ERR_SHAPE, "image size %dx%d", width, height);
    if (!dev_depth_cur || !dev_depth_state || !params) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL depth / params pointer");
    if (rgb_pixel_stride != 3 && rgb_pixel_stride != 4) return fail(ctx, GGT_ERR_INVALID_ARG, "rgb_pixel_stride %d (3 or 4)", rgb_pixel_stride);
    if (params->downscale != 4 || params->pool != 3) return fail(ctx, GGT_ERR_UNSUPPORTED, "only downscale 4 / pool 3 (PAPER.md:81) are implemented");
    if (!(params->lambda_t > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "lambda_t must be > 0");
    if (dev_rgb_prev && !dev_rgb_cur) return fail(ctx, GGT_ERR_INVALID_ARG, "rgb_prev given without rgb_cur");
    const long long cells = (long long)((width + 3) / 4) * ((height + 3) / 4);
    if (cells > GGT_REFINE_STATIC_MAX_CELLS)
        return fail(ctx, GGT_ERR_SHAPE, "ggt_refine_depth_static: %dx%d needs %lld quarter-resolution cells, the fixed scratch holds %d "
                    "(use ggt_refine_depth)", width, height, cells, GGT_REFINE_STATIC_MAX_CELLS);
    cudaStream_t st = (cudaStream_t)stream;
    if (!dev_rgb_prev) {                                        // first-frame rule (M = 1): no scratch involved
        cudaError_t e = ggt_launch_first_frame(width, height, dev_depth_cur, dev_depth_state, dev_mask_out, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_refine_depth_static first-frame launch");
        ctx->launches += 1;
        return GGT_OK;
    }
    uint16_t* cq = nullptr;
    cudaError_t e = ggt_refine_static_scratch(&cq);
    if (e != cudaSuccess || !cq) return cuda_fail(ctx, e, "address of the fixed refine scratch");
    GgtRefineViews tab;
    memset(&tab, 0, sizeof tab);
    tab.n = 1;
    tab.v[0].rgb_cur = dev_rgb_cur; tab.v[0].rgb_prev = dev_rgb_prev; tab.v[0].depth_cur = dev_depth_cur;
    tab.v[0].depth_state = dev_depth_state; tab.v[0].mask_out = dev_mask_out; tab.v[0].pooled_out = dev_pooled_out;
    tab.v[0].cq = cq;
    int n = 0;
    e = ggt_launch_refine(width, height, tab, rgb_pixel_stride, params->lambda_t, params->beta, params->theta, st, &n);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_refine_depth_static launch");
    ctx->launches += n;
    return GGT_OK;
}

// a3: validates the views, sizes the {depth, omega} workspace and launches the weight-map pre-pass for all of them
// (one launch); map_out[k] is the device address of view k's zero-padded {depth, omega} map.
static int prepare_maps(ggt_ctx* ctx, int32_t n_views, const ggt_camera* views, const float* const* dev_depths,
                        const float* const* dev_weights, float w_sigma0, float w_clip, int32_t w_window,
                        const float2** map_out, cudaStream_t st, int only_view = -1) {
    size_t need = 0;
    for (int k = 0; k < n_views; ++k) {
        if (views[k].width <= 0 || views[k].height <= 0 || views[k].width > 32767 || views[k].height > 32767)
            return fail(ctx, GGT_ERR_SHAPE, "view %d size %dx%d", k, views[k].width, views[k].height);
        if (!dev_depths[k]) return fail(ctx, GGT_ERR_INVALID_ARG, "dev_depths[%d] is NULL", k);
        need += align_up(((size_t)views[k].width + 1) * ((size_t)views[k].height + 1) * sizeof(float2), 256);
    }
    if (ctx->ws_bytes < need) {
        if (ctx->ws && !ctx->ws_owned) return fail(ctx, GGT_ERR_SHAPE, "workspace %zu B < required %zu B", ctx->ws_bytes, need);
        if (ctx->ws) cudaFree(ctx->ws);   // synchronises: only between frames, when the view set grows
        ctx->ws = nullptr; ctx->ws_bytes = 0;
        cudaError_t e = cudaMalloc(&ctx->ws, need);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "workspace allocation");
        ctx->ws_bytes = need; ctx->ws_owned = true;
    }
    char* w = static_cast<char*>(ctx->ws);
    StageTimer tm(ctx, GGT_STAGE_WEIGHT, st);
    GgtWeightParams wp;
    memset(&wp, 0, sizeof wp);
    wp.n_views = n_views; wp.window = w_window;
    wp.sigma0 = w_sigma0; wp.c2 = w_clip * w_clip;
    wp.fast_ok = (w_sigma0 >= 1e-20f && w_sigma0 <= 1e20f) ? 1 : 0;
    for (int k = 0; k < n_views; ++k) {
        map_out[k] = reinterpret_cast<const float2*>(w);
        wp.v[k].depth = dev_depths[k]; wp.v[k].out = reinterpret_cast<float2*>(w);
        wp.v[k].weight = dev_weights ? dev_weights[k] : nullptr;
        wp.v[k].width = views[k].width; wp.v[k].height = views[k].height;
        w += align_up(((size_t)views[k].width + 1) * ((size_t)views[k].height + 1) * sizeof(float2), 256);
    }
    if (ctx->weights_prelaunched) return GGT_OK;      // ggt_frame_host launched them view by view, behind each view's upload
    if (only_view >= 0) {                               // one view of the set (same workspace layout)
        wp.v[0] = wp.v[only_view];
        wp.n_views = 1;
    }
    cudaError_t e = ggt_launch_weight_maps(wp, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "weight-map launch");
    ctx->launches += 1;
    return GGT_OK;
}

// a4: the relative transform target -> view (12 floats) and the view's map for the kernels
static void fill_view_params(const ggt_camera& target, const ggt_camera& view, const float2* map, GgtViewParams& vp) {
    float hm[9], ev[3];
    relative_transform(target, view, hm, ev);
    for (int i = 0; i < 6; ++i) vp.nh[i] = -hm[i];
    for (int i = 0; i < 3; ++i) vp.h2[i] = hm[6 + i];
    vp.ne[0] = -ev[0]; vp.ne[1] = -ev[1]; vp.e2 = ev[2];
    vp.map = map;
    vp.width = view.width; vp.height = view.height;
    vp.stride = (uint32_t)view.width + 1u;
}

// Shared by ggt_integrate and ggt_raymarch_depth: a3 + a4 for one target.
static int prepare_views(ggt_ctx* ctx, const ggt_camera* target, int32_t n_views, const ggt_camera* views,
                         const float* const* dev_depths, const float* const* dev_weights, float w_sigma0, float w_clip, int32_t w_window,
                         GgtViewParams* vp, cudaStream_t st) {
    const float2* maps[GGT_MAX_VIEWS];
    const int rc = prepare_maps(ctx, n_views, views, dev_depths, dev_weights, w_sigma0, w_clip, w_window, maps, st);
    if (rc != GGT_OK) return rc;
    for (int k = 0; k < n_views; ++k) fill_view_params(*target, views[k], maps[k], vp[k]);
    return GGT_OK;
}

// same-size / shared-w detection for the integrate kernel's fast marches
static void detect_fast_paths(GgtIntegrateParams& p, int32_t n_views) {
    p.same_size = 1;
    for (int k = 1; k < n_views; ++k)
        if (p.v[k].width != p.v[0].width || p.v[k].height != p.v[0].height) p.same_size = 0;
    // rig of identical parallel cameras with coplanar centres: H_k and e_k[2] have the same bits in every view, so
    // b_k = H_k (uc, vc, 1) and w_k(z) = fma(z, b_k[2], e2) do too
    p.shared_w = p.same_size && n_views >= 2;
    for (int k = 1; k < n_views; ++k)
        if (memcmp(p.v[k].nh, p.v[0].nh, sizeof p.v[0].nh) != 0 || memcmp(p.v[k].h2, p.v[0].h2, sizeof p.v[0].h2) != 0 ||
            memcmp(&p.v[k].e2, &p.v[0].e2, sizeof(float)) != 0) p.shared_w = 0;
}

// Shared front end of ggt_integrate / ggt_integrate_extract: validation, workspace, weight maps, launch.
// ggt_frame_host launches a frame in row slices so that each slice's results can travel while the next one computes
struct SliceHook { int (*fn)(void* user, int row0, int row1); void* user; int n_slices; };

static int integrate_impl(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                          const ggt_camera* views, const float* const* dev_depths, const float* const* dev_weights,
                          uint32_t flags, bool fused,
                          float* dev_depth, float* dev_conf, int32_t* dev_bin, void* stream, const SliceHook* hook = nullptr) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!vol || !target || !views || !dev_depths) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL volume / camera / depth pointer");
    if (n_views < 1 || n_views > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_views %d not in [1, %d]", n_views, GGT_MAX_VIEWS);
    if (flags != GGT_OVERWRITE && flags != GGT_ACCUMULATE) return fail(ctx, GGT_ERR_INVALID_ARG, "flags %u", flags);
    if (target->width != vol->desc.width || target->height != vol->desc.height)
        return fail(ctx, GGT_ERR_SHAPE, "target %dx%d does not match the volume %dx%d", target->width, target->height,
                    vol->desc.width, vol->desc.height);
    if (!(target->fx > 0.0f) || !(target->fy > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "target focal length");
    cudaStream_t st = (cudaStream_t)stream;
    GgtIntegrateParams p;
    memset(&p, 0, sizeof p);
    p.Wt = vol->desc.width; p.Ht = vol->desc.height; p.D = vol->desc.bins;
    p.n_views = n_views; p.n_groups = vol->n_groups;
    p.plane = (unsigned long long)vol->desc.width * (unsigned long long)vol->desc.height;
    p.accumulate = flags == GGT_ACCUMULATE ? 1 : 0;
    p.decay = vol->desc.decay; p.cap = vol->desc.weight_cap;
    p.tables = vol->dev_tables; p.voxels = vol->dev_voxels; p.hint = vol->dev_hints;
    p.depth = dev_depth; p.conf = dev_conf; p.bin = dev_bin;
    {
        const int rc = prepare_views(ctx, target, n_views, views, dev_depths, dev_weights, vol->desc.w_sigma0, vol->desc.w_clip,
                                     vol->desc.w_window, p.v, st);
        if (rc != GGT_OK) return rc;
    }
    StageTimer tm(ctx, GGT_STAGE_INTEGRATE, st);
    detect_fast_paths(p, n_views);
    const int n_slices = hook ? hook->n_slices : 1;
    for (int sl = 0; sl < n_slices; ++sl) {
        p.row0 = (int)((long long)p.Ht * sl / n_slices) / 8 * 8;              // whole CTAs of 8 rows
        p.row1 = sl + 1 == n_slices ? p.Ht : (int)((long long)p.Ht * (sl + 1) / n_slices) / 8 * 8;
        if (p.row1 <= p.row0) continue;
        cudaError_t e = ggt_launch_integrate(p, vol->desc.dtype, fused, ctx->sm_count, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "integrate launch");
        ctx->launches += 1;
        if (hook) {
            const int rc = hook->fn(hook->user, p.row0, p.row1);
            if (rc != GGT_OK) return rc;
        }
    }
    return GGT_OK;
}

int ggt_integrate(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                  const ggt_camera* views, const float* const* dev_depths, uint32_t flags, void* stream) {
    return integrate_impl(ctx, vol, target, n_views, views, dev_depths, nullptr, flags, false, nullptr, nullptr, nullptr, stream);
}

int ggt_integrate_weighted(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                           const ggt_camera* views, const float* const* dev_depths, const float* const* dev_weights,
                           uint32_t flags, void* stream) {
    return integrate_impl(ctx, vol, target, n_views, views, dev_depths, dev_weights, flags, false, nullptr, nullptr, nullptr, stream);
}

int ggt_integrate_extract(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                          const ggt_camera* views, const float* const* dev_depths, uint32_t flags,
                          float* dev_depth, float* dev_conf, int32_t* dev_bin, void* stream) {
    return integrate_impl(ctx, vol, target, n_views, views, dev_depths, nullptr, flags, true, dev_depth, dev_conf, dev_bin, stream);
}

static int integrate_batch_impl(ggt_ctx* ctx, int32_t n_targets, ggt_volume* const* vols, const ggt_camera* targets,
                                int32_t n_rig_views, const ggt_camera* rig_views, const float* const* dev_depths,
                                int32_t n_views, const int32_t* view_index, uint32_t flags, bool fused,
                                float* const* dev_depth_out, float* const* dev_conf_out, int32_t* const* dev_bin_out,
                                void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!vols || !targets || !rig_views || !dev_depths || !view_index) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL argument to ggt_integrate_batch");
    if (n_targets < 1) return fail(ctx, GGT_ERR_SHAPE, "n_targets %d", n_targets);
    if (n_rig_views < 1 || n_rig_views > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_rig_views %d not in [1, %d]", n_rig_views, GGT_MAX_VIEWS);
    if (n_views < 1 || n_views > n_rig_views) return fail(ctx, GGT_ERR_SHAPE, "n_views %d not in [1, n_rig_views]", n_views);
    if (flags != GGT_OVERWRITE && flags != GGT_ACCUMULATE) return fail(ctx, GGT_ERR_INVALID_ARG, "flags %u", flags);
    for (int t = 0; t < n_targets; ++t) {
        if (!vols[t]) return fail(ctx, GGT_ERR_INVALID_ARG, "vols[%d] is NULL", t);
        if (targets[t].width != vols[t]->desc.width || targets[t].height != vols[t]->desc.height)
            return fail(ctx, GGT_ERR_SHAPE, "target %d does not match its volume", t);
        if (!(targets[t].fx > 0.0f) || !(targets[t].fy > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "target %d focal length", t);
        if (vols[t]->desc.w_sigma0 != vols[0]->desc.w_sigma0 || vols[t]->desc.w_clip != vols[0]->desc.w_clip ||
            vols[t]->desc.w_window != vols[0]->desc.w_window)
            return fail(ctx, GGT_ERR_INVALID_ARG, "the volumes of one batch must share the Eq. 11-12 parameters");
        for (int k = 0; k < n_views; ++k) {
            const int idx = view_index[t * n_views + k];
            if (idx < 0 || idx >= n_rig_views) return fail(ctx, GGT_ERR_INVALID_ARG, "view_index[%d][%d] = %d", t, k, idx);
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    const float2* maps[GGT_MAX_VIEWS];
    int rc = prepare_maps(ctx, n_rig_views, rig_views, dev_depths, nullptr, vols[0]->desc.w_sigma0, vols[0]->desc.w_clip,
                          vols[0]->desc.w_window, maps, st);                      // the weight maps, once per frame
    if (rc != GGT_OK) return rc;
    for (int t = 0; t < n_targets; ++t) {
        const ggt_volume* vol = vols[t];
        GgtIntegrateParams p;
        memset(&p, 0, sizeof p);
        p.Wt = vol->desc.width; p.Ht = vol->desc.height; p.D = vol->desc.bins;
        p.n_views = n_views; p.n_groups = vol->n_groups;
        p.plane = (unsigned long long)vol->desc.width * (unsigned long long)vol->desc.height;
        p.accumulate = flags == GGT_ACCUMULATE ? 1 : 0;
        p.decay = vol->desc.decay; p.cap = vol->desc.weight_cap;
        p.tables = vol->dev_tables; p.voxels = vol->dev_voxels; p.hint = vol->dev_hints;
        if (fused) {
            p.depth = dev_depth_out ? dev_depth_out[t] : nullptr;
            p.conf = dev_conf_out ? dev_conf_out[t] : nullptr;
            p.bin = dev_bin_out ? dev_bin_out[t] : nullptr;
        }
        for (int k = 0; k < n_views; ++k) {
            const int idx = view_index[t * n_views + k];
            fill_view_params(targets[t], rig_views[idx], maps[idx], p.v[k]);
        }
        detect_fast_paths(p, n_views);
        p.row0 = 0; p.row1 = p.Ht;
        StageTimer tm(ctx, GGT_STAGE_INTEGRATE, st);
        cudaError_t e = ggt_launch_integrate(p, vol->desc.dtype, fused, ctx->sm_count, st);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "integrate launch");
        ctx->launches += 1;
    }
    return GGT_OK;
}

int ggt_integrate_batch(ggt_ctx* ctx, int32_t n_targets, ggt_volume* const* vols, const ggt_camera* targets,
                        int32_t n_rig_views, const ggt_camera* rig_views, const float* const* dev_depths,
                        int32_t n_views, const int32_t* view_index, uint32_t flags, void* stream) {
    return integrate_batch_impl(ctx, n_targets, vols, targets, n_rig_views, rig_views, dev_depths, n_views, view_index, flags,
                                false, nullptr, nullptr, nullptr, stream);
}

int ggt_integrate_extract_batch(ggt_ctx* ctx, int32_t n_targets, ggt_volume* const* vols, const ggt_camera* targets,
                                int32_t n_rig_views, const ggt_camera* rig_views, const float* const* dev_depths,
                                int32_t n_views, const int32_t* view_index, uint32_t flags, float* const* dev_depth,
                                float* const* dev_conf, int32_t* const* dev_bin, void* stream) {
    return integrate_batch_impl(ctx, n_targets, vols, targets, n_rig_views, rig_views, dev_depths, n_views, view_index, flags,
                                true, dev_depth, dev_conf, dev_bin, stream);
}

int ggt_extract_depth(ggt_ctx* ctx, const ggt_volume* vol, float* dev_depth, float* dev_conf, int32_t* dev_bin,
                      void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!vol) return fail(ctx, GGT_ERR_INVALID_ARG, "volume is NULL");
    GgtExtractParams p = extract_params(vol);
    p.depth = dev_depth; p.conf = dev_conf; p.bin = dev_bin;
    StageTimer tm(ctx, GGT_STAGE_EXTRACT, (cudaStream_t)stream);
    cudaError_t e = ggt_launch_extract(p, vol->desc.dtype, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "extract launch");
    ctx->launches += 1;
    return GGT_OK;
}

int ggt_raymarch_depth(ggt_ctx* ctx, const ggt_camera* target, int32_t n_views, const ggt_camera* views,
                       const float* const* dev_depths, const ggt_raymarch_params* params, float* dev_depth,
                       float* dev_conf, int32_t* dev_steps, void* stream) {
    return ggt_raymarch_depth_weighted(ctx, target, n_views, views, dev_depths, nullptr, params, dev_depth, dev_conf,
                                       dev_steps, stream);
}

int ggt_raymarch_depth_weighted(ggt_ctx* ctx, const ggt_camera* target, int32_t n_views, const ggt_camera* views,
                                const float* const* dev_depths, const float* const* dev_weights,
                                const ggt_raymarch_params* params, float* dev_depth, float* dev_conf,
                                int32_t* dev_steps, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!target || !views || !dev_depths || !params) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL camera / depth / params pointer");
    if (n_views < 1 || n_views > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_views %d not in [1, %d]", n_views, GGT_MAX_VIEWS);
    if (target->width <= 0 || target->height <= 0) return fail(ctx, GGT_ERR_SHAPE, "target size %dx%d", target->width, target->height);
    if (!(target->fx > 0.0f) || !(target->fy > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "target focal length");
    if (!(params->z_far > params->z_near) || !(params->z_near > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "z_near / z_far");
    if (!(params->tau > 0.0f) || !(params->step_scale > 0.0f) || !(params->min_step > 0.0f))
        return fail(ctx, GGT_ERR_INVALID_ARG, "tau, step_scale and min_step must be > 0");
    if (params->max_evals < 1 || params->n_bisect < 0) return fail(ctx, GGT_ERR_INVALID_ARG, "max_evals / n_bisect");
    if (params->w_window != 0 && params->w_window != 7) return fail(ctx, GGT_ERR_UNSUPPORTED, "w_window %d (0 or 7)", params->w_window);
    cudaStream_t st = (cudaStream_t)stream;
    GgtRaymarchParams p;
    memset(&p, 0, sizeof p);
    p.Wt = target->width; p.Ht = target->height; p.n_views = n_views;
    p.max_evals = params->max_evals; p.n_bisect = params->n_bisect;
    p.z_near = params->z_near; p.z_far = params->z_far; p.tau = params->tau;
    p.step_scale = params->step_scale; p.min_step = params->min_step;
    p.depth = dev_depth; p.conf = dev_conf; p.steps = dev_steps;
    const int rc = prepare_views(ctx, target, n_views, views, dev_depths, dev_weights, params->w_sigma0, params->w_clip,
                                 params->w_window, p.v, st);
    if (rc != GGT_OK) return rc;
    p.shared_w = n_views >= 2;
    for (int k = 1; k < n_views; ++k)
        if (memcmp(p.v[k].h2, p.v[0].h2, sizeof p.v[0].h2) != 0 || memcmp(&p.v[k].e2, &p.v[0].e2, sizeof(float)) != 0) p.shared_w = 0;
    StageTimer tm(ctx, GGT_STAGE_RAYMARCH, st);
    cudaError_t e = ggt_launch_raymarch(p, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "raymarch launch");
    ctx->launches += 1;
    return GGT_OK;
}

int ggt_temporal_weight(ggt_ctx* ctx, const ggt_camera* prev_target, const float* dev_prev_depth,
                        const float* dev_prev_conf, int32_t n_views, const ggt_camera* views,
                        const float* const* dev_masks, float beta, float eta, float* dev_weight_out, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!prev_target || !dev_prev_depth || !dev_prev_conf || !dev_weight_out || (n_views > 0 && (!views || !dev_masks)))
        return fail(ctx, GGT_ERR_INVALID_ARG, "NULL argument to ggt_temporal_weight");
    if (n_views < 0 || n_views > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_views %d not in [0, %d]", n_views, GGT_MAX_VIEWS);
    if (prev_target->width <= 0 || prev_target->height <= 0) return fail(ctx, GGT_ERR_SHAPE, "previous target size");
    if (!(prev_target->fx > 0.0f) || !(prev_target->fy > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "previous target focal length");
    if (!(beta >= 0.0f) || !(eta >= 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "beta and eta must be >= 0");
    GgtTemporalParams p;
    memset(&p, 0, sizeof p);
    p.Wt = prev_target->width; p.Ht = prev_target->height; p.n_views = n_views;
    p.beta = beta; p.eta = eta;
    p.prev_depth = dev_prev_depth; p.prev_conf = dev_prev_conf; p.out = dev_weight_out;
    for (int k = 0; k < n_views; ++k) {
        if (views[k].width <= 0 || views[k].height <= 0 || views[k].width > 32767 || views[k].height > 32767)
            return fail(ctx, GGT_ERR_SHAPE, "view %d size %dx%d", k, views[k].width, views[k].height);
        if (!dev_masks[k]) return fail(ctx, GGT_ERR_INVALID_ARG, "dev_masks[%d] is NULL", k);
        relative_transform(*prev_target, views[k], p.v[k].h, p.v[k].e);
        p.v[k].mask = dev_masks[k];
        p.v[k].width = views[k].width; p.v[k].height = views[k].height;
    }
    cudaError_t e = ggt_launch_temporal_weight(p, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "temporal-weight launch");
    ctx->launches += 1;
    return GGT_OK;
}

// ---- f-3: forward warping with pixel-sized Gaussians ---------------------------------------------------------------
int ggt_splat_reserve(ggt_ctx* ctx, int64_t entries) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (entries < 0 || entries > 0xfffffff0ll) return fail(ctx, GGT_ERR_INVALID_ARG, "entries %lld not in [0, 2^32)", (long long)entries);
    ctx->splat_entries = (size_t)entries;
    return GGT_OK;
}

int ggt_splat_status(ggt_ctx* ctx, int64_t* host_entries_last, int64_t* host_entries_needed, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    uint32_t f[2] = {0, 0};
    if (ctx->splat_flags) {
        cudaStream_t st = (cudaStream_t)stream;
        cudaError_t e = cudaMemcpyAsync(f, ctx->splat_flags, sizeof f, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(ctx->splat_flags + 1, 0, sizeof(uint32_t), st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_splat_status");
    }
    if (host_entries_last) *host_entries_last = f[0];
    if (host_entries_needed) *host_entries_needed = f[1];
    return GGT_OK;
}

int ggt_splat_forward(ggt_ctx* ctx, const ggt_camera* target, const ggt_camera* view, const float* dev_depth,
                      const uint8_t* dev_rgb, int32_t rgb_pixel_stride, const float* dev_mask,
                      const ggt_splat_params* params, float* dev_out_rgb, float* dev_out_alpha, float* dev_out_depth,
                      float* dev_out_mask, int32_t* dev_out_count, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!target || !view || !dev_depth || !params) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL camera / depth / params pointer");
    if (target->width <= 0 || target->height <= 0 || target->width > 32767 || target->height > 32767 || view->width <= 0 ||
        view->height <= 0 || view->width > 32767 || view->height > 32767)
        return fail(ctx, GGT_ERR_SHAPE, "view %dx%d / target %dx%d", view->width, view->height, target->width, target->height);
    if (!(target->fx > 0.0f) || !(target->fy > 0.0f) || !(view->fx > 0.0f) || !(view->fy > 0.0f))
        return fail(ctx, GGT_ERR_INVALID_ARG, "focal length");
    if (dev_rgb && rgb_pixel_stride != 3 && rgb_pixel_stride != 4) return fail(ctx, GGT_ERR_INVALID_ARG, "rgb_pixel_stride %d (3 or 4)", rgb_pixel_stride);
    if (!(params->sigma_px > 0.0f) || !(params->dilation >= 0.0f) || !(params->z_cull > 0.0f))
        return fail(ctx, GGT_ERR_INVALID_ARG, "sigma_px / z_cull must be > 0, dilation >= 0");
    const size_t N = (size_t)view->width * view->height, Nt = (size_t)target->width * target->height;
    size_t cap = ctx->splat_entries ? ctx->splat_entries : 40 * N;
    if (cap > 0xfffffff0ull) cap = 0xfffffff0ull;
    const size_t n_blocks = (Nt + 2047) / 2048;
    const size_t o_gauss = 0, o_counts = align_up(o_gauss + N * 32, 256), o_pos = align_up(o_counts + Nt * 4, 256),
                 o_sums = align_up(o_pos + Nt * 4, 256), o_entries = align_up(o_sums + n_blocks * 4, 256),
                 need = o_entries + cap * 8;
    if (ctx->splat_ws_bytes < need) {            // grows between calls only (synchronises: cudaFree)
        if (ctx->splat_ws) cudaFree(ctx->splat_ws);
        ctx->splat_ws = nullptr; ctx->splat_ws_bytes = 0;
        cudaError_t e = cudaMalloc(&ctx->splat_ws, need);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "splat scratch allocation");
        ctx->splat_ws_bytes = need;
    }
    if (!ctx->splat_flags) {
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&ctx->splat_flags), 2 * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMemset(ctx->splat_flags, 0, 2 * sizeof(uint32_t));
        if (e != cudaSuccess) return cuda_fail(ctx, e, "splat flags allocation");
    }
    GgtSplatParams p;
    memset(&p, 0, sizeof p);
    p.W = view->width; p.H = view->height; p.Wt = target->width; p.Ht = target->height;
    p.rgb_stride = rgb_pixel_stride; p.capacity = (uint32_t)cap;
    relative_transform(*view, *target, p.h, p.e);       // roles exchanged: from the view's pixel / depth into the target
    p.fx_t = target->fx; p.fy_t = target->fy; p.cx_t = target->cx; p.cy_t = target->cy; p.fx_s = view->fx;
    p.sigma_px = params->sigma_px; p.dilation = params->dilation; p.z_cull = params->z_cull;
    p.depth = dev_depth; p.rgb = dev_rgb; p.mask = dev_mask;
    char* w = static_cast<char*>(ctx->splat_ws);
    p.gauss = reinterpret_cast<float*>(w + o_gauss);
    p.counts = reinterpret_cast<uint32_t*>(w + o_counts);
    p.pos = reinterpret_cast<uint32_t*>(w + o_pos);
    p.block_sums = reinterpret_cast<uint32_t*>(w + o_sums);
    p.entries = reinterpret_cast<uint2*>(w + o_entries);
    p.total = ctx->splat_flags; p.overflow = ctx->splat_flags + 1;
    p.out_rgb = dev_out_rgb; p.out_alpha = dev_out_alpha; p.out_depth = dev_out_depth; p.out_mask = dev_out_mask;
    p.out_count = dev_out_count;
    int n = 0;
    cudaError_t e = ggt_launch_splat(p, (cudaStream_t)stream, &n);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "splat launch");
    ctx->launches += n;
    return GGT_OK;
}

int ggt_temporal_weight_mask(ggt_ctx* ctx, int64_t n_pixels, const float* dev_prev_depth, const float* dev_prev_conf,
                             int32_t n_masks, const float* const* dev_masks, float beta, float eta,
                             float* dev_weight_out, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!dev_prev_depth || !dev_prev_conf || !dev_masks || !dev_weight_out) return fail(ctx, GGT_ERR_INVALID_ARG, "NULL argument to ggt_temporal_weight_mask");
    if (n_pixels <= 0) return fail(ctx, GGT_ERR_SHAPE, "n_pixels %lld", (long long)n_pixels);
    if (n_masks < 1 || n_masks > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_masks %d not in [1, %d]", n_masks, GGT_MAX_VIEWS);
    if (!(beta >= 0.0f) || !(eta >= 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "beta and eta must be >= 0");
    GgtMaskList ml;
    memset(&ml, 0, sizeof ml);
    ml.n = n_masks;
    for (int k = 0; k < n_masks; ++k) {
        if (!dev_masks[k]) return fail(ctx, GGT_ERR_INVALID_ARG, "dev_masks[%d] is NULL", k);
        ml.m[k] = dev_masks[k];
    }
    cudaError_t e = ggt_launch_temporal_weight_mask((size_t)n_pixels, dev_prev_depth, dev_prev_conf, ml, beta, eta, dev_weight_out,
                                                    (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "temporal-weight-mask launch");
    ctx->launches += 1;
    return GGT_OK;
}

// camera centre C = -R^T t in double, rounded once (the oracle does the same)
static void camera_centre(const ggt_camera& c, float* C) {
    for (int i = 0; i < 3; ++i)
        C[i] = (float)(-((double)c.R[i] * c.t[0] + (double)c.R[3 + i] * c.t[1] + (double)c.R[6 + i] * c.t[2]));
}

int ggt_guidance_features(ggt_ctx* ctx, const ggt_camera* target, const float* dev_depth, int32_t n_views,
                          const ggt_camera* views, float* dev_features, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!target || !dev_depth || !dev_features || (n_views > 0 && !views))
        return fail(ctx, GGT_ERR_INVALID_ARG, "NULL argument to ggt_guidance_features");
    if (n_views < 1 || n_views > GGT_MAX_VIEWS) return fail(ctx, GGT_ERR_SHAPE, "n_views %d not in [1, %d]", n_views, GGT_MAX_VIEWS);
    if (target->width <= 0 || target->height <= 0) return fail(ctx, GGT_ERR_SHAPE, "target size %dx%d", target->width, target->height);
    if (!(target->fx > 0.0f) || !(target->fy > 0.0f)) return fail(ctx, GGT_ERR_INVALID_ARG, "target focal length");
    GgtFeatureParams p;
    memset(&p, 0, sizeof p);
    p.W = target->width; p.H = target->height; p.n_views = n_views;
    p.fx = target->fx; p.fy = target->fy; p.cx = target->cx; p.cy = target->cy;
    p.fast_ok = (target->fx >= 1e-10f && target->fx <= 1e10f && target->fy >= 1e-10f && target->fy <= 1e10f) ? 1 : 0;
    for (int i = 0; i < 9; ++i) p.R[i] = target->R[i];
    for (int i = 0; i < 3; ++i) p.t[i] = target->t[i];
    camera_centre(*target, p.Ct);
    p.depth = dev_depth; p.out = dev_features;
    for (int k = 0; k < n_views; ++k) {
        camera_centre(views[k], p.v[k].C);
        const double dx = (double)p.v[k].C[0] - p.Ct[0], dy = (double)p.v[k].C[1] - p.Ct[1], dz = (double)p.v[k].C[2] - p.Ct[2];
        p.v[k].dist = (float)std::sqrt(dx * dx + dy * dy + dz * dz);
        p.v[k].axes = (float)((double)views[k].R[6] * target->R[6] + (double)views[k].R[7] * target->R[7] +
                              (double)views[k].R[8] * target->R[8]);
    }
    cudaError_t e = ggt_launch_features(p, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "features launch");
    ctx->launches += 1;
    return GGT_OK;
}

// ---- end-to-end frame from host buffers -------------------------------------------------------------
// staging layout (every block 256-B aligned), all views width x height:
//   per slot s:  rgb[2][H*W*3] (ping-pong current / previous colour), state[H*W] fp32 refined depth
//   per view k:  depth_cur[H*W] fp32
//   outputs:     two sets of depth[Ht*Wt], conf[Ht*Wt] fp32 (alternating, see GGT_FRAME_RESULTS_ASYNC)
size_t ggt_frame_staging_bytes(const ggt_volume_desc* desc, int32_t n_slots, int32_t n_views, int32_t width,
                               int32_t height) {
    if (!desc || n_slots <= 0 || n_views <= 0 || width <= 0 || height <= 0) return 0;
    const size_t px = (size_t)width * height;
    const size_t rgb = align_up(px * 3, 256), dep = align_up(px * 4, 256);
    const size_t out = align_up((size_t)desc->width * desc->height * 4, 256);
    return (size_t)n_slots * (2 * rgb + dep) + (size_t)n_views * dep + 4 * out;
}

int ggt_frame_host_results_wait(ggt_ctx* ctx, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    for (int i = 0; i < 2; ++i) {
        if (!ctx->d2h_pending[i]) continue;
        cudaError_t e = cudaStreamWaitEvent((cudaStream_t)stream, ctx->ev_d2h_done[i], 0);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "ggt_frame_host_results_wait");
    }
    return GGT_OK;
}

int ggt_frame_host(ggt_ctx* ctx, ggt_volume* vol, const ggt_camera* target, int32_t n_views,
                   const ggt_camera* views, const uint8_t* const* host_rgb_cur, const float* const* host_depth_cur,
                   const int32_t* slots, int32_t n_slots, uint32_t* host_slot_state,
                   const ggt_refine_params* params, uint32_t flags, void* dev_staging, size_t staging_bytes,
                   float* host_depth, float* host_conf, void* stream) {
    if (!ctx) return GGT_ERR_INVALID_ARG;
    if (!vol || !target || !views || !host_depth_cur || !slots || !host_slot_state || !dev_staging)
        return fail(ctx, GGT_ERR_INVALID_ARG, "NULL argument to ggt_frame_host");
    if (n_views < 1 || n_views > GGT_MAX_VIEWS || n_slots < 1) return fail(ctx, GGT_ERR_SHAPE, "n_views / n_slots");
    const int W = views[0].width, H = views[0].height;
    for (int k = 0; k < n_views; ++k) {
        if (views[k].width != W || views[k].height != H) return fail(ctx, GGT_ERR_SHAPE, "ggt_frame_host needs equal view sizes");
        if (slots[k] < 0 || slots[k] >= n_slots) return fail(ctx, GGT_ERR_INVALID_ARG, "slots[%d] = %d", k, slots[k]);
        if (!host_depth_cur[k]) return fail(ctx, GGT_ERR_INVALID_ARG, "host_depth_cur[%d] is NULL", k);
        for (int j = 0; j < k; ++j)
            if (slots[j] == slots[k]) return fail(ctx, GGT_ERR_INVALID_ARG, "slots[%d] == slots[%d] = %d: two views of one call cannot share a history slot", j, k, slots[k]);
    }
    const bool async_results = (flags & GGT_FRAME_RESULTS_ASYNC) != 0;
    flags &= ~GGT_FRAME_RESULTS_ASYNC;
    if (flags != GGT_OVERWRITE && flags != GGT_ACCUMULATE) return fail(ctx, GGT_ERR_INVALID_ARG, "flags %u", flags);
    if (((uintptr_t)dev_staging & 255) != 0) return fail(ctx, GGT_ERR_INVALID_ARG, "staging must be 256-byte aligned");
    const size_t need = ggt_frame_staging_bytes(&vol->desc, n_slots, n_views, W, H);
    if (staging_bytes < need) return fail(ctx, GGT_ERR_SHAPE, "staging %zu B < required %zu B", staging_bytes, need);
    const bool refine = host_rgb_cur != nullptr && params != nullptr;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t px = (size_t)W * H;
    const size_t rgb = align_up(px * 3, 256), dep = align_up(px * 4, 256);
    const size_t out = align_up((size_t)vol->desc.width * vol->desc.height * 4, 256);
    char* base = static_cast<char*>(dev_staging);
    char* view_base = base + (size_t)n_slots * (2 * rgb + dep);
    char* out_base = view_base + (size_t)n_views * dep;
    // Uploads go to the context's copy stream, ordered after the previous frame's last reader of the input buffers
    // (its weight-map pre-pass), so that they overlap that frame's integrate / extract when the caller does not
    // synchronise in between; the caller's stream then waits for them.
    if (!ctx->copy_stream) {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_inputs_free, cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "copy stream / events");
    }
    cudaStream_t cs = ctx->copy_stream;
    if (ctx->inputs_free_pending) {
        cudaError_t e = cudaStreamWaitEvent(cs, ctx->ev_inputs_free, 0);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "stream wait");
    }
    const float* dptr[GGT_MAX_VIEWS];
    uint8_t* rcur[GGT_MAX_VIEWS];
    const uint8_t* rprev[GGT_MAX_VIEWS];
    uint32_t new_state[GGT_MAX_VIEWS];                 // committed to host_slot_state only once every enqueue has succeeded
    // view by view: its uploads on the copy stream, and -- as soon as they have landed -- its refine kernels and its
    // weight map on the caller's stream, so that only the last view's small kernels are left after the last upload
    for (int k = 0; k < n_views; ++k) {
        char* slot = base + (size_t)slots[k] * (2 * rgb + dep);
        float* dcur = reinterpret_cast<float*>(view_base + (size_t)k * dep);
        cudaError_t e = cudaMemcpyAsync(dcur, host_depth_cur[k], px * 4, cudaMemcpyHostToDevice, cs);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "H2D depth");
        rcur[k] = nullptr; rprev[k] = nullptr;
        dptr[k] = dcur;
        if (refine && host_rgb_cur[k]) {
            const uint32_t s = host_slot_state[slots[k]];     // bit 0: has history, bit 1: parity of "current"
            const int cur = (s >> 1) & 1 ? 0 : 1;
            rcur[k] = reinterpret_cast<uint8_t*>(slot + (size_t)cur * rgb);
            rprev[k] = (s & 1) ? reinterpret_cast<const uint8_t*>(slot + (size_t)(1 - cur) * rgb) : nullptr;
            e = cudaMemcpyAsync(rcur[k], host_rgb_cur[k], px * 3, cudaMemcpyHostToDevice, cs);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "H2D colour");
            new_state[k] = 1u | ((uint32_t)cur << 1);
            dptr[k] = reinterpret_cast<float*>(slot + 2 * rgb);          // the slot's refined-depth state
        }
        if (!ctx->ev_view[k]) {
            e = cudaEventCreateWithFlags(&ctx->ev_view[k], cudaEventDisableTiming);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "view event");
        }
        e = cudaEventRecord(ctx->ev_view[k], cs);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "view event");
    }
    for (int k = 0; k < n_views; ++k) {
        cudaError_t e = cudaStreamWaitEvent(st, ctx->ev_view[k], 0);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "view event wait");
        if (rcur[k]) {
            const uint8_t* bc = rcur[k]; const uint8_t* bp = rprev[k];
            const float* bd = reinterpret_cast<const float*>(view_base + (size_t)k * dep);
            float* bs = const_cast<float*>(dptr[k]);
            int rcode = ggt_refine_depth_batch(ctx, 1, W, H, &bc, &bp, 3, &bd, &bs, nullptr, nullptr, params, stream);
            if (rcode != GGT_OK) return rcode;
        }
        // the last reader of the uploaded buffers is the last view's refine kernel (its weight map reads the slot's state)
        // or, for a view that is not refined, its weight map: from there on the next frame's uploads may overwrite them
        const bool last = k == n_views - 1;
        if (last && rcur[k]) {
            e = cudaEventRecord(ctx->ev_inputs_free, st);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "event record");
        }
        const float2* maps_unused[GGT_MAX_VIEWS];
        int rcode = prepare_maps(ctx, n_views, views, dptr, nullptr, vol->desc.w_sigma0, vol->desc.w_clip, vol->desc.w_window,
                                 maps_unused, st, k);
        if (rcode != GGT_OK) return rcode;
        if (last && !rcur[k]) {
            e = cudaEventRecord(ctx->ev_inputs_free, st);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "event record");
        }
    }
    ctx->inputs_free_pending = true;
    // results: their copies run on the context's own stream, slice by slice behind the kernels that produce them; set 0,
    // or alternating sets of device buffers when the caller does not wait for them (GGT_FRAME_RESULTS_ASYNC)
    if (!ctx->d2h_stream) {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_kernels_done, cudaEventDisableTiming);
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&ctx->ev_d2h_done[i], cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "result stream / events");
    }
    const int set = async_results ? ctx->result_set : 0;
    if (ctx->d2h_pending[set]) {                         // the kernels below overwrite this set: its last copy must be done
        cudaError_t e = cudaStreamWaitEvent(st, ctx->ev_d2h_done[set], 0);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "stream wait");
    }
    float* d_depth = reinterpret_cast<float*>(out_base + (size_t)set * 2 * out);
    float* d_conf = reinterpret_cast<float*>(out_base + (size_t)set * 2 * out + out);
    ctx->weights_prelaunched = true;
    // a3-a7 in one pass: the result the host wants comes out of the integrate kernel itself (same bits as
    // ggt_integrate followed by ggt_extract_depth, without re-reading the volume).  When the caller waits for the results
    // on `stream`, the frame runs as 4 row slices: slice i's results cross PCIe while slice i + 1 computes.
    struct CopyCtx { ggt_ctx* ctx; cudaStream_t st; float *dd, *dc, *hd, *hc; int Wt; } cc = {ctx, st, d_depth, d_conf, host_depth, host_conf, vol->desc.width};
    SliceHook hook;
    hook.user = &cc;
    hook.n_slices = (async_results || (!host_depth && !host_conf)) ? 1 : 4;
    hook.fn = [](void* user, int row0, int row1) -> int {
        CopyCtx& c = *static_cast<CopyCtx*>(user);
        cudaStream_t rs = c.ctx->d2h_stream;
        cudaError_t e = cudaEventRecord(c.ctx->ev_kernels_done, c.st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(rs, c.ctx->ev_kernels_done, 0);
        const size_t o = (size_t)row0 * c.Wt, nb = (size_t)(row1 - row0) * c.Wt * sizeof(float);
        if (e == cudaSuccess && c.hd) e = cudaMemcpyAsync(c.hd + o, c.dd + o, nb, cudaMemcpyDeviceToHost, rs);
        if (e == cudaSuccess && c.hc) e = cudaMemcpyAsync(c.hc + o, c.dc + o, nb, cudaMemcpyDeviceToHost, rs);
        return e == cudaSuccess ? GGT_OK : cuda_fail(c.ctx, e, "D2H results");
    };
    int rcode = integrate_impl(ctx, vol, target, n_views, views, dptr, nullptr, flags, true, host_depth ? d_depth : nullptr,
                               host_conf ? d_conf : nullptr, nullptr, stream, &hook);
    ctx->weights_prelaunched = false;
    if (rcode != GGT_OK) return rcode;
    {
        cudaError_t e = cudaEventRecord(ctx->ev_d2h_done[set], ctx->d2h_stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "result event");
        if (async_results) {
            ctx->d2h_pending[set] = true;
            ctx->result_set ^= 1;
        } else {                                         // the results are complete when `stream` is synchronised
            e = cudaStreamWaitEvent(st, ctx->ev_d2h_done[set], 0);
            if (e != cudaSuccess) return cuda_fail(ctx, e, "stream wait");
            ctx->d2h_pending[set] = false;
        }
    }
    for (int k = 0; k < n_views; ++k)                  // every enqueue succeeded: the slots now hold this frame
        if (rcur[k]) host_slot_state[slots[k]] = new_state[k];
    return GGT_OK;
}

}  // extern "C"
