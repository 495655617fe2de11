// ggt_refine.cu — steps a1-a2: colour-difference soft mask and temporal depth filter of one input view.
//
// PAPER.md:79-81 (Eq. 1: M = min(|I^t - I^{t-1}| / lambda_t + beta, 1), computed at quarter resolution,
// 3x3 max-pool, bilinear upscale) and PAPER.md:83-84 (Eq. 2: D' = M D + (1 - M) D'_{t-1}).
// Readings P5-P8, P17 of DESIGN.md fix what the paper leaves open (L1 over RGB, 4x4 box sums, clipped
// pooling window, half-pixel bilinear, valid-term handling).
//
// Two kernels per call, for one view (ggt_refine_depth) or all views of a frame at once (ggt_refine_depth_batch,
// blockIdx.z = view):
//   k_block_diff   one thread per quarter-res cell: 4x4 box sums of both images, L1 over RGB  (integer)
//   k_mask_blend   one CTA per 64x16 pixel tile: 3x3 max-pool + Eq. 1 on the 18x6 cells the tile's bilinear
//                  footprint touches (shared memory), then per pixel bilinear x4 + Eq. 2, 128-bit accesses.
// HBM traffic per pixel: 6 B colour + 12 B depth (+4 B mask if requested) -> streaming, HBM-bound.
#include "ggt_internal.h"

#include <mutex>

namespace {

constexpr int S = 4;           // quarter resolution per axis (reading P7)
constexpr int TILE_W = 64, TILE_H = 16;
constexpr int CW = TILE_W / S + 2, CH = TILE_H / S + 2;      // Mq cells a tile touches: 18 x 6
constexpr int QW = CW + 2, QH = CH + 2;                      // cq cells the pooling of those needs: 20 x 8

__device__ __forceinline__ int iabs_diff(int a, int b) { return a > b ? a - b : b - a; }

// Sum of the R, G, B bytes of 4 consecutive packed RGB pixels held in three little-endian words.
__device__ __forceinline__ void rgb4_sums(uint32_t w0, uint32_t w1, uint32_t w2, int& r, int& g, int& b) {
    // bytes: w0 = r0 g0 b0 r1 | w1 = g1 b1 r2 g2 | w2 = b2 r3 g3 b3
    r += (w0 & 0xff) + (w0 >> 24) + ((w1 >> 16) & 0xff) + ((w2 >> 8) & 0xff);
    g += ((w0 >> 8) & 0xff) + (w1 & 0xff) + (w1 >> 24) + ((w2 >> 16) & 0xff);
    b += ((w0 >> 16) & 0xff) + ((w1 >> 8) & 0xff) + (w2 & 0xff) + (w2 >> 24);
}

template <bool FAST>
__global__ void __launch_bounds__(256)
k_block_diff(int W, int H, int Wq, int Hq, const __grid_constant__ GgtRefineViews tab, int stride) {
    const uint8_t* __restrict__ cur = tab.v[blockIdx.z].rgb_cur;
    const uint8_t* __restrict__ prev = tab.v[blockIdx.z].rgb_prev;
    uint16_t* __restrict__ cq = tab.v[blockIdx.z].cq;
    const int xq = blockIdx.x * 32 + threadIdx.x;
    const int yq = blockIdx.y * 8 + threadIdx.y;
    if (xq >= Wq || yq >= Hq) return;
    int rc = 0, gc = 0, bc = 0, rp = 0, gp = 0, bp = 0;
    if (FAST && (xq * S + S <= W)) {
        // stride 3, W % 4 == 0, 4-byte aligned rows: three 32-bit loads per row per image
#pragma unroll
        for (int dy = 0; dy < S; ++dy) {
            int y = yq * S + dy;
            y = y > H - 1 ? H - 1 : y;
            const size_t o = ((size_t)y * W + (size_t)xq * S) * 3;
            const uint32_t* c = reinterpret_cast<const uint32_t*>(cur + o);
            const uint32_t* p = reinterpret_cast<const uint32_t*>(prev + o);
            const uint32_t c0 = __ldg(c), c1 = __ldg(c + 1), c2 = __ldg(c + 2);
            const uint32_t p0 = __ldg(p), p1 = __ldg(p + 1), p2 = __ldg(p + 2);
            rgb4_sums(c0, c1, c2, rc, gc, bc);
            rgb4_sums(p0, p1, p2, rp, gp, bp);
        }
    } else {
        for (int dy = 0; dy < S; ++dy) {
            int y = yq * S + dy;
            y = y > H - 1 ? H - 1 : y;
            for (int dx = 0; dx < S; ++dx) {
                int x = xq * S + dx;
                x = x > W - 1 ? W - 1 : x;
                const size_t o = ((size_t)y * W + x) * stride;
                rc += cur[o]; gc += cur[o + 1]; bc += cur[o + 2];
                rp += prev[o]; gp += prev[o + 1]; bp += prev[o + 2];
            }
        }
    }
    cq[(size_t)yq * Wq + xq] = (uint16_t)(iabs_diff(rc, rp) + iabs_diff(gc, gp) + iabs_diff(bc, bp));
}

__global__ void __launch_bounds__(256)
k_mask_blend(int W, int H, int Wq, int Hq, const __grid_constant__ GgtRefineViews tab, float lambda_t, float beta,
             float theta, int vec_ok) {
    const uint16_t* __restrict__ cq = tab.v[blockIdx.z].cq;
    const float* __restrict__ depth_cur = tab.v[blockIdx.z].depth_cur;
    float* __restrict__ depth_state = tab.v[blockIdx.z].depth_state;
    float* __restrict__ mask_out = tab.v[blockIdx.z].mask_out;
    uint16_t* __restrict__ pooled_out = tab.v[blockIdx.z].pooled_out;
    __shared__ int s_cq[QH][QW];
    __shared__ float s_m[CH][CW];
    const int tid = threadIdx.x;
    const int x0q = blockIdx.x * (TILE_W / S), y0q = blockIdx.y * (TILE_H / S);
    // cq window starting at (x0q - 2, y0q - 2); out-of-image cells hold 0 (= excluded from the max, cq >= 0)
    for (int i = tid; i < QW * QH; i += 256) {
        const int cx = x0q - 2 + i % QW, cy = y0q - 2 + i / QW;
        int v = 0;
        if (cx >= 0 && cx < Wq && cy >= 0 && cy < Hq) v = cq[(size_t)cy * Wq + cx];
        s_cq[i / QW][i % QW] = v;
    }
    __syncthreads();
    // Mq of cell (clamp(x0q-1+i), clamp(y0q-1+j)): 3x3 max (window clipped to the image), then Eq. 1
    if (tid < CW * CH) {
        const int i = tid % CW, j = tid / CW;
        int cx = x0q - 1 + i, cy = y0q - 1 + j;
        cx = cx < 0 ? 0 : (cx > Wq - 1 ? Wq - 1 : cx);
        cy = cy < 0 ? 0 : (cy > Hq - 1 ? Hq - 1 : cy);
        const int lx = cx - (x0q - 2), ly = cy - (y0q - 2);     // position in s_cq, >= 1 by construction
        int m = 0;
        if (lx >= 1 && lx < QW - 1 && ly >= 1 && ly < QH - 1) {
#pragma unroll
            for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) m = max(m, s_cq[ly + dy][lx + dx]);
        }
        const float delta = __fdiv_rn((float)m, (float)(S * S * 255));
        float a = __fsub_rn(delta, theta);
        a = a > 0.0f ? a : 0.0f;
        const float b = __fdiv_rn(a, lambda_t);
        float mq = __fadd_rn(b, beta);
        mq = mq > 1.0f ? 1.0f : mq;
        s_m[j][i] = mq;
        if (pooled_out && i >= 1 && i <= TILE_W / S && j >= 1 && j <= TILE_H / S) {
            const int ox = x0q - 1 + i, oy = y0q - 1 + j;
            if (ox < Wq && oy < Hq) pooled_out[(size_t)oy * Wq + ox] = (uint16_t)m;
        }
    }
    __syncthreads();
    // 4 consecutive pixels per thread: thread -> (row tid / 16, columns 4 * (tid % 16) .. +3)
    const int y = blockIdx.y * TILE_H + tid / 16;
    const int xb = blockIdx.x * TILE_W + (tid % 16) * 4;
    if (y >= H || xb >= W) return;
    float sy = __fsub_rn(__fmul_rn(__fadd_rn((float)y, 0.5f), 0.25f), 0.5f);
    sy = sy < 0.0f ? 0.0f : sy;
    sy = sy > (float)(Hq - 1) ? (float)(Hq - 1) : sy;
    const int yq0 = (int)sy;                                  // sy >= 0: truncation == floor
    const float fy = __fsub_rn(sy, (float)yq0);
    const int yq1 = yq0 + 1 < Hq ? yq0 + 1 : Hq - 1;
    const int ly0 = yq0 - (y0q - 1), ly1 = yq1 - (y0q - 1);
    const size_t base = (size_t)y * W + xb;
    const bool vec = vec_ok && (xb + 3 < W);         // vec_ok: W % 4 == 0 and every depth / mask pointer 16-B aligned
    float dc[4], dp[4], out[4], mk[4];
    if (vec) {
        const float4 c4 = __ldg(reinterpret_cast<const float4*>(depth_cur + base));
        const float4 p4 = *reinterpret_cast<const float4*>(depth_state + base);
        dc[0] = c4.x; dc[1] = c4.y; dc[2] = c4.z; dc[3] = c4.w;
        dp[0] = p4.x; dp[1] = p4.y; dp[2] = p4.z; dp[3] = p4.w;
    } else {
        for (int i = 0; i < 4; ++i) {
            const bool in = xb + i < W;
            dc[i] = in ? depth_cur[base + i] : 0.0f;
            dp[i] = in ? depth_state[base + i] : 0.0f;
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int x = xb + i;
        float sx = __fsub_rn(__fmul_rn(__fadd_rn((float)x, 0.5f), 0.25f), 0.5f);
        sx = sx < 0.0f ? 0.0f : sx;
        sx = sx > (float)(Wq - 1) ? (float)(Wq - 1) : sx;
        const int xq0 = (int)sx;
        const float fx = __fsub_rn(sx, (float)xq0);
        const int xq1 = xq0 + 1 < Wq ? xq0 + 1 : Wq - 1;
        const int lx0 = xq0 - (x0q - 1), lx1 = xq1 - (x0q - 1);
        const float a00 = s_m[ly0][lx0], a01 = s_m[ly0][lx1], a10 = s_m[ly1][lx0], a11 = s_m[ly1][lx1];
        const float top = fmaf(fx, __fsub_rn(a01, a00), a00);
        const float bot = fmaf(fx, __fsub_rn(a11, a10), a10);
        const float M = fmaf(fy, __fsub_rn(bot, top), top);
        const bool vc = dc[i] > 0.0f, vp = dp[i] > 0.0f;
        // wc + wp == 0  <=>  neither term carries weight (M in [beta, 1] may be exactly 1 -> wp = 0)
        const float wc = vc ? M : 0.0f;
        const float wp = vp ? __fsub_rn(1.0f, M) : 0.0f;
        float o;
        if (__fadd_rn(wc, wp) == 0.0f) o = 0.0f;
        else if (vc && vp) o = fmaf(M, __fsub_rn(dc[i], dp[i]), dp[i]);
        else o = vc ? dc[i] : dp[i];
        out[i] = o;
        mk[i] = M;
    }
    if (vec) {
        *reinterpret_cast<float4*>(depth_state + base) = make_float4(out[0], out[1], out[2], out[3]);
        if (mask_out) *reinterpret_cast<float4*>(mask_out + base) = make_float4(mk[0], mk[1], mk[2], mk[3]);
    } else {
        for (int i = 0; i < 4; ++i)
            if (xb + i < W) {
                depth_state[base + i] = out[i];
                if (mask_out) mask_out[base + i] = mk[i];
            }
    }
}

__global__ void __launch_bounds__(256)
k_first_frame(size_t n, const float* __restrict__ depth_cur, float* __restrict__ depth_state,
              float* __restrict__ mask_out) {
    const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    depth_state[i] = depth_cur[i];
    if (mask_out) mask_out[i] = 1.0f;
}

// ---- ggt_refine_depth_static: the block-difference scratch without an allocation -----------------------------------
// The one piece of scratch memory of the refine step (k_block_diff's quarter-resolution L1 differences, read back by
// k_mask_blend) as a file-scope device array of a fixed size, for callers that may not allocate (stream capture, serving
// loops).  512 KB: quarter-resolution cells of one view of up to 2048 x 2048 pixels (1920 x 1080 needs 259 200 B); every
// GPU that loads the library holds it until the process exits.  All calls share it.
__device__ __align__(256) uint16_t g_refine_static_cq[GGT_REFINE_STATIC_MAX_CELLS];

// In host code `g_refine_static_cq` is only a handle of the symbol, not a device address: the address is asked for once
// per device, with that device current, and kept.
constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
uint16_t* g_static_ptr[kMaxDevices] = {};

}  // namespace

// All views of `tab` have the same size and a previous colour image; one launch of each kernel, blockIdx.z = view.
cudaError_t ggt_launch_refine(int W, int H, const GgtRefineViews& tab, int stride, float lambda_t, float beta, float theta,
                              cudaStream_t st, int* n_launches) {
    const int Wq = (W + S - 1) / S, Hq = (H + S - 1) / S;
    const dim3 blk(32, 8), grd((Wq + 31) / 32, (Hq + 7) / 8, tab.n);
    bool fast = stride == 3 && (W % 4) == 0;
    for (int k = 0; k < tab.n; ++k) fast = fast && (((uintptr_t)tab.v[k].rgb_cur | (uintptr_t)tab.v[k].rgb_prev) & 3) == 0;
    if (fast) k_block_diff<true><<<grd, blk, 0, st>>>(W, H, Wq, Hq, tab, stride);
    else k_block_diff<false><<<grd, blk, 0, st>>>(W, H, Wq, Hq, tab, stride);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const dim3 grd2((W + TILE_W - 1) / TILE_W, (H + TILE_H - 1) / TILE_H, tab.n);
    // 128-bit accesses only when every row start is 16-B aligned: W % 4 == 0 and 16-B aligned caller pointers (a tensor
    // view at a 4-byte offset is legal input and takes the scalar path)
    uintptr_t bits = 0;
    for (int k = 0; k < tab.n; ++k)
        bits |= (uintptr_t)tab.v[k].depth_cur | (uintptr_t)tab.v[k].depth_state | (uintptr_t)tab.v[k].mask_out;
    const int vec_ok = ((W & 3) == 0 && (bits & 15) == 0) ? 1 : 0;
    k_mask_blend<<<grd2, 256, 0, st>>>(W, H, Wq, Hq, tab, lambda_t, beta, theta, vec_ok);
    *n_launches = 2;
    return cudaGetLastError();
}

cudaError_t ggt_launch_first_frame(int W, int H, const float* depth_cur, float* depth_state, float* mask_out, cudaStream_t st) {
    const size_t n = (size_t)W * H;
    k_first_frame<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, depth_cur, depth_state, mask_out);
    return cudaGetLastError();
}

// Device address of the static scratch on the CURRENT device (cached per device; no allocation).
cudaError_t ggt_refine_static_scratch(uint16_t** ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* a = nullptr;
        e = cudaGetSymbolAddress(&a, g_refine_static_cq);
        if (e != cudaSuccess) return e;
        g_static_ptr[dev] = static_cast<uint16_t*>(a);
    }
    *ptr = g_static_ptr[dev];
    return cudaSuccess;
}
