// ggt_splat.cu — SURVEY.md 8(f) row f-3: forward warping with pixel-sized 3D Gaussians (section 3.1,
// PAPER.md:362-368 A.3; rasterised as in the 3D Gaussian splatting paper the text cites).
//
// One isotropic, fully opaque Gaussian per pixel of an input view, at the 3D point its depth gives, with the standard
// deviation that projects to sigma_px source pixels; EWA projection into the target view (2D covariance
// sigma^2 J J^T + dilation I); per target pixel, the Gaussians with alpha >= 1/255 are composited front to back in
// ascending depth (ties: ascending source index) until the transmittance would fall below 1e-4.  Readings S1-S8 of
// DESIGN.md; every fp32 operation is in the oracle's stated order (this file is compiled with --fmad=false and IEEE
// division / square root, so plain operators are single correctly rounded operations).
//
// B200 design: the Gaussians of a view are a dense grid of ~2 million tiny splats (radius < 3 px), so instead of the
// tile / duplicate / global radix sort of a general rasteriser the kernels build exact PER-PIXEL lists:
//   k_splat_scatter<0> one thread per source pixel: project (S1-S3), keep the 8 parameters, and count, with one
//                      atomic per covered target pixel, the pixels where alpha >= 1/255
//   k_scan_*           exclusive prefix sum of the per-pixel counts (three small kernels)
//   k_splat_scatter<1> the same traversal again, writing {depth bits, source index} into each pixel's list
//   k_splat_composite  one thread per target pixel: a warp stages the lists of its 32 pixels in shared memory, each
//                      lane sorts its own by (depth, index) and blends it front to back
// The order of a list in memory is arbitrary (atomics); the (depth, index) key makes the result deterministic.
#include "ggt_internal.h"

namespace {

// exp(q), q <= 0 (reading S8): 2^n times a degree-7 polynomial of the fractional part, fp32, fixed operation order
__device__ __forceinline__ float exp_le0(float q) {
    if (q < -80.0f) return 0.0f;
    const float t = q * 1.44269504f;
    const float big = 12582912.0f;
    const float n = __fadd_rn(__fadd_rn(t, big), -big);
    const float f = t - n;
    float p = 1.52527338e-5f;
    p = fmaf(p, f, 1.54035304e-4f);
    p = fmaf(p, f, 1.33335581e-3f);
    p = fmaf(p, f, 9.61812911e-3f);
    p = fmaf(p, f, 5.55041087e-2f);
    p = fmaf(p, f, 2.40226507e-1f);
    p = fmaf(p, f, 6.93147181e-1f);
    p = fmaf(p, f, 1.0f);
    return p * __int_as_float(((int)n + 127) << 23);
}

struct Gauss { float mx, my, z, ca, cb, cc, rad, ok; };      // 32 bytes: two 128-bit words

// q = -1/2 d^T Sigma'^-1 d of a Gaussian at the pixel centre (pcx, pcy); alpha = min(0.99, exp(q)) (S4)
__device__ __forceinline__ float q_at(float mx, float my, float ca, float cb, float cc, float pcx, float pcy) {
    const float dx = mx - pcx, dy = my - pcy;
    const float t1 = dx * dx, t2 = dy * dy, t3 = dx * dy;
    const float s3 = ca * t1 + cc * t2;
    return (-0.5f * s3) - cb * t3;
}

// alpha >= 1/255 without the exponential: exp_le0 is monotone across alpha = 1/255 and kQStar is the smallest q with
// exp_le0(q) >= 1/255 (every float in [-5.56, -5.52] is checked against the oracle's exponential in
// tests/test_oracle_splat_pins.py; outside that interval its 1e-6 accuracy decides).
constexpr float kQStar = -5.541263580322266f;      // 0xC0B15208

// S1-S3, S7 for source pixel (u, v) with depth D
__device__ __forceinline__ bool project(const GgtSplatParams& p, int u, int v, float D, Gauss& g) {
    g.mx = g.my = g.z = g.ca = g.cb = g.cc = g.rad = 0.0f;
    g.ok = 0.0f;
    if (!(D > 0.0f)) return false;
    const float uc = (float)u + 0.5f, vc = (float)v + 0.5f;
    const float bx = fmaf(p.h[0], uc, fmaf(p.h[1], vc, p.h[2]));
    const float by = fmaf(p.h[3], uc, fmaf(p.h[4], vc, p.h[5]));
    const float bw = fmaf(p.h[6], uc, fmaf(p.h[7], vc, p.h[8]));
    const float x = fmaf(D, bx, p.e[0]), y = fmaf(D, by, p.e[1]), w = fmaf(D, bw, p.e[2]);
    if (!(w >= p.z_cull)) return false;
    const float rw = 1.0f / w;
    const float mx = x * rw, my = y * rw;
    const float tx = (mx - p.cx_t) / p.fx_t, ty = (my - p.cy_t) / p.fy_t;
    const float sig = p.sigma_px * D / p.fx_s;
    const float gx = p.fx_t * rw, gy = p.fy_t * rw;
    const float s2 = sig * sig;
    const float a = s2 * (gx * gx) * (1.0f + tx * tx) + p.dilation;
    const float b = s2 * (gx * gy) * (tx * ty);
    const float c = s2 * (gy * gy) * (1.0f + ty * ty) + p.dilation;
    const float det = a * c - b * b;
    if (!(det > 0.0f)) return false;
    const float idet = 1.0f / det;
    const float mid = 0.5f * (a + c);
    const float disc = fmaxf(mid * mid - det, 0.0f);
    const float lmax = mid + sqrtf(disc);
    g.mx = mx; g.my = my; g.z = w;
    g.ca = c * idet; g.cb = -b * idet; g.cc = a * idet;
    g.rad = 3.34f * sqrtf(lmax);
    g.ok = 1.0f;
    return true;
}

// candidate pixel rectangle of a Gaussian (centres within the conservative radius), clipped to the target image
__device__ __forceinline__ bool rect_of(const Gauss& g, int Wt, int Ht, int& x0, int& x1, int& y0, int& y1) {
    const float x0f = floorf(g.mx - g.rad - 0.5f), x1f = ceilf(g.mx + g.rad - 0.5f);
    const float y0f = floorf(g.my - g.rad - 0.5f), y1f = ceilf(g.my + g.rad - 0.5f);
    if (!(x1f >= 0.0f) || !(y1f >= 0.0f) || !(x0f <= (float)(Wt - 1)) || !(y0f <= (float)(Ht - 1))) return false;
    x0 = (int)fmaxf(x0f, 0.0f); x1 = (int)fminf(x1f, (float)(Wt - 1));
    y0 = (int)fmaxf(y0f, 0.0f); y1 = (int)fminf(y1f, (float)(Ht - 1));
    return true;
}

template <bool FILL>
__global__ void __launch_bounds__(256)
k_splat_scatter(const __grid_constant__ GgtSplatParams p) {
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (u >= p.W || v >= p.H) return;
    const size_t i = (size_t)v * p.W + u;
    Gauss g;
    if (!FILL) {
        project(p, u, v, __ldg(p.depth + i), g);
        float4* o = reinterpret_cast<float4*>(p.gauss) + 2 * i;
        o[0] = make_float4(g.mx, g.my, g.z, g.ca);
        o[1] = make_float4(g.cb, g.cc, g.rad, g.ok);
    } else {
        const float4* s = reinterpret_cast<const float4*>(p.gauss) + 2 * i;
        const float4 a = s[0], b = s[1];
        g.mx = a.x; g.my = a.y; g.z = a.z; g.ca = a.w; g.cb = b.x; g.cc = b.y; g.rad = b.z; g.ok = b.w;
    }
    if (g.ok == 0.0f) return;
    int x0, x1, y0, y1;
    if (!rect_of(g, p.Wt, p.Ht, x0, x1, y0, y1)) return;
    for (int py = y0; py <= y1; ++py)
        for (int px = x0; px <= x1; ++px) {
            const float q = q_at(g.mx, g.my, g.ca, g.cb, g.cc, (float)px + 0.5f, (float)py + 0.5f);
            if (!(q <= 0.0f && q >= kQStar)) continue;          // alpha >= 1/255 (S4), without the exponential
            const size_t t = (size_t)py * p.Wt + px;
            if (!FILL) {
                atomicAdd(p.counts + t, 1u);
            } else {
                const unsigned slot = atomicAdd(p.pos + t, 1u);
                if (slot < p.capacity) p.entries[slot] = make_uint2(__float_as_uint(g.z), (unsigned)i);
            }
        }
}

// ---- exclusive prefix sum of n 32-bit counts: per-block sums, one-block scan of the sums, per-block scan + offset ----
constexpr int SCAN_T = 256, SCAN_E = 8, SCAN_B = SCAN_T * SCAN_E;      // 2048 elements per block

__device__ __forceinline__ unsigned block_exclusive_scan(unsigned v, unsigned* s_warp, unsigned& total) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned y = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += y;
    }
    if (lane == 31) s_warp[wid] = x;
    __syncthreads();
    if (wid == 0) {
        unsigned w = lane < SCAN_T / 32 ? s_warp[lane] : 0u;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned y = __shfl_up_sync(0xffffffffu, w, d);
            if (lane >= d) w += y;
        }
        if (lane < SCAN_T / 32) s_warp[lane] = w;
    }
    __syncthreads();
    total = s_warp[SCAN_T / 32 - 1];
    const unsigned base = wid > 0 ? s_warp[wid - 1] : 0u;
    __syncthreads();
    return base + x - v;
}

__global__ void __launch_bounds__(SCAN_T)
k_scan_block_sums(size_t n, const unsigned* __restrict__ in, unsigned* __restrict__ sums) {
    __shared__ unsigned s_warp[SCAN_T / 32];
    const size_t b0 = (size_t)blockIdx.x * SCAN_B + (size_t)threadIdx.x * SCAN_E;
    unsigned v = 0;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) v += b0 + e < n ? in[b0 + e] : 0u;
    unsigned total;
    block_exclusive_scan(v, s_warp, total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(SCAN_T)
k_scan_sums(int n_blocks, unsigned* __restrict__ sums, unsigned* __restrict__ total_out, unsigned capacity,
            unsigned* __restrict__ overflow) {
    __shared__ unsigned s_warp[SCAN_T / 32];
    unsigned carry = 0;
    for (int b = 0; b < n_blocks; b += SCAN_T) {
        const int i = b + threadIdx.x;
        const unsigned v = i < n_blocks ? sums[i] : 0u;
        unsigned total;
        const unsigned ex = block_exclusive_scan(v, s_warp, total);
        if (i < n_blocks) sums[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) {
        *total_out = carry;
        if (carry > capacity) atomicMax(overflow, carry);       // the lists do not fit: the call writes zeros
    }
}

__global__ void __launch_bounds__(SCAN_T)
k_scan_apply(size_t n, const unsigned* __restrict__ in, const unsigned* __restrict__ sums, unsigned* __restrict__ out) {
    __shared__ unsigned s_warp[SCAN_T / 32];
    const size_t b0 = (size_t)blockIdx.x * SCAN_B + (size_t)threadIdx.x * SCAN_E;
    unsigned c[SCAN_E], v = 0;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) { c[e] = b0 + e < n ? in[b0 + e] : 0u; v += c[e]; }
    unsigned total;
    unsigned run = sums[blockIdx.x] + block_exclusive_scan(v, s_warp, total);
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        if (b0 + e < n) out[b0 + e] = run;
        run += c[e];
    }
}

// ---- per target pixel: front-to-back compositing of its list (S5-S6) ------------------------------------------------
// The lists of a warp's 32 consecutive pixels are one contiguous run of the entries array (the prefix sum is in pixel
// order), so the warp copies its run into shared memory with coalesced loads, every lane sorts its own list there
// (insertion sort by (depth, index): lists are ~20 entries) and blends it in one pass, gathering each Gaussian's
// parameters, colour and mask.  The CTA's 8 warps share a pool of kPool entries; a warp whose run does not fit (heavy
// occlusion) selects the smallest remaining key from global memory instead.  Measured alternatives on a 1352 x 1014 view
// (profiles/r2_splat.md): selection from global memory for every warp 1.33 ms (L1 pipeline 96 % busy: noisy surfaces
// rarely saturate early, so a list is re-read ~n times); 16-byte entries that carry alpha and colour, so that nothing is
// gathered here, 1.07 ms (the sort then moves twice the bytes and only two CTAs fit an SM); this version 0.92 ms.
constexpr int kPool = 8192;                                 // entries per CTA: 64 KB -> three CTAs per SM

struct Blend { float T, C0, C1, C2, Dacc, Macc; };

__device__ __forceinline__ unsigned long long key_of(uint2 e) { return ((unsigned long long)e.x << 32) | e.y; }   // {z bits, index}

// blends Gaussian gi into b (S6); false once the transmittance would fall below 1e-4
__device__ __forceinline__ bool blend_one(const GgtSplatParams& p, unsigned gi, float pcx, float pcy, Blend& b) {
    const float4* s = reinterpret_cast<const float4*>(p.gauss) + 2 * (size_t)gi;
    const float4 ga = __ldg(s), gb = __ldg(s + 1);
    const float a = fminf(exp_le0(q_at(ga.x, ga.y, ga.w, gb.x, gb.y, pcx, pcy)), 0.99f);     // >= 1/255: it is on the list
    const float tt = b.T * (1.0f - a);
    if (tt < 1e-4f) return false;
    const float wgt = a * b.T;
    if (p.rgb) {
        const uint8_t* c = p.rgb + (size_t)gi * p.rgb_stride;
        b.C0 = fmaf((float)c[0], wgt, b.C0); b.C1 = fmaf((float)c[1], wgt, b.C1); b.C2 = fmaf((float)c[2], wgt, b.C2);
    }
    b.Dacc = fmaf(ga.z, wgt, b.Dacc);
    if (p.mask) b.Macc = fmaf(__ldg(p.mask + gi), wgt, b.Macc);
    b.T = tt;
    return true;
}

__device__ __forceinline__ void composite_sorted(const GgtSplatParams& p, uint2* L, unsigned n, float pcx, float pcy, Blend& b) {
    for (unsigned i = 1; i < n; ++i) {
        const uint2 cur = L[i];
        const unsigned long long k = key_of(cur);
        unsigned j = i;
        while (j > 0 && key_of(L[j - 1]) > k) { L[j] = L[j - 1]; --j; }
        L[j] = cur;
    }
    for (unsigned e = 0; e < n; ++e)
        if (!blend_one(p, L[e].y, pcx, pcy, b)) break;
}

// list left in global memory: repeated selection of the smallest remaining key
__device__ __forceinline__ void composite_select(const GgtSplatParams& p, const uint2* L, unsigned n, float pcx, float pcy, Blend& b) {
    unsigned long long last = 0ull;                          // keys are > 0: depth bits of z > 0 in the high word
    for (unsigned step = 0; step < n; ++step) {
        unsigned long long best = ~0ull;
        for (unsigned e = 0; e < n; ++e) {
            const unsigned long long key = key_of(L[e]);
            if (key > last && key < best) best = key;
        }
        last = best;
        if (!blend_one(p, (unsigned)(best & 0xffffffffull), pcx, pcy, b)) break;
    }
}

__global__ void __launch_bounds__(256)
k_splat_composite(const __grid_constant__ GgtSplatParams p) {
    extern __shared__ __align__(16) uint2 s_pool[];          // [kPool]
    __shared__ unsigned s_len[8];
    const int px = blockIdx.x * 32 + threadIdx.x;
    const int py = blockIdx.y * 8 + threadIdx.y;
    const bool row = py < p.Ht, live = row && px < p.Wt;
    const size_t t = (size_t)(row ? py : p.Ht - 1) * p.Wt + (px < p.Wt ? px : p.Wt - 1);
    const size_t Nt = (size_t)p.Wt * p.Ht;
    const bool fits = *p.total <= p.capacity;                // else the lists did not fit: the whole call writes zeros
    const unsigned cnt = p.counts[t];
    const unsigned n = (live && fits) ? cnt : 0u;
    const unsigned end = p.pos[t];                           // after the fill pass: start + counts
    const unsigned start = end - cnt;
    // the warp's run: [start of its first pixel, end of its last live pixel)
    const unsigned run0 = __shfl_sync(0xffffffffu, start, 0);
    const unsigned run1 = __reduce_max_sync(0xffffffffu, live ? end : 0u);
    const unsigned run_n = (row && fits && run1 > run0) ? run1 - run0 : 0u;
    if (threadIdx.x == 0) s_len[threadIdx.y] = run_n;
    __syncthreads();
    unsigned off = 0;                                        // pool offset: warps are placed in order while they fit
    bool staged = true;
    for (int w = 0; w <= (int)threadIdx.y; ++w) {
        const unsigned len = s_len[w];
        const bool ok = off + len <= kPool;
        if (w == (int)threadIdx.y) staged = ok;
        else if (ok) off += len;
    }
    Blend b = {1.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
    const float pcx = (float)px + 0.5f, pcy = (float)py + 0.5f;
    if (staged) {
        uint2* sw = s_pool + off;
        for (unsigned i = threadIdx.x; i < run_n; i += 32) sw[i] = p.entries[run0 + i];
        __syncwarp();
        composite_sorted(p, sw + (start - run0), n, pcx, pcy, b);
    } else {
        composite_select(p, p.entries + start, n, pcx, pcy, b);
    }
    if (!live) return;
    const float acc = 1.0f - b.T;
    if (p.out_rgb) { p.out_rgb[t] = b.C0; p.out_rgb[Nt + t] = b.C1; p.out_rgb[2 * Nt + t] = b.C2; }
    if (p.out_alpha) p.out_alpha[t] = acc;
    if (p.out_depth) p.out_depth[t] = acc > 0.0f ? b.Dacc / acc : 0.0f;
    if (p.out_mask) p.out_mask[t] = b.Macc;
    if (p.out_count) p.out_count[t] = fits ? (int)cnt : 0;
}

// Eq. 13 with the paper's own novel-view mask: M^t = channel-wise maximum of the K splatted masks
__global__ void __launch_bounds__(256)
k_temporal_weight_mask(size_t n, const float* __restrict__ prev_depth, const float* __restrict__ prev_conf,
                       const __grid_constant__ GgtMaskList masks, float beta, float eta, float* __restrict__ out) {
    const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const float d = __ldg(prev_depth + i), acc = __ldg(prev_conf + i);
    float wt = 0.0f;
    if (d > 0.0f && acc > 0.0f) {
        float M = __ldg(masks.m[0] + i);
        for (int k = 1; k < masks.n; ++k) M = fmaxf(M, __ldg(masks.m[k] + i));
        const float stat = fmaxf(1.0f - M, 0.0f);
        const float t = (beta * acc) * stat;
        wt = t < eta ? t : eta;
    }
    out[i] = wt;
}

}  // namespace

cudaError_t ggt_launch_splat(const GgtSplatParams& p, cudaStream_t st, int* n_launches) {
    const size_t Nt = (size_t)p.Wt * p.Ht;
    const int n_blocks = (int)((Nt + SCAN_B - 1) / SCAN_B);
    cudaError_t e = cudaMemsetAsync(p.counts, 0, Nt * sizeof(unsigned), st);
    if (e != cudaSuccess) return e;
    const dim3 blk(32, 8), gs((p.W + 31) / 32, (p.H + 7) / 8), gt((p.Wt + 31) / 32, (p.Ht + 7) / 8);
    k_splat_scatter<false><<<gs, blk, 0, st>>>(p);
    k_scan_block_sums<<<n_blocks, SCAN_T, 0, st>>>(Nt, p.counts, p.block_sums);
    k_scan_sums<<<1, SCAN_T, 0, st>>>(n_blocks, p.block_sums, p.total, p.capacity, p.overflow);
    k_scan_apply<<<n_blocks, SCAN_T, 0, st>>>(Nt, p.counts, p.block_sums, p.pos);
    k_splat_scatter<true><<<gs, blk, 0, st>>>(p);
    // 64 KB of dynamic shared memory needs the opt-in (per device and context, so it is simply set before every launch)
    e = cudaFuncSetAttribute(k_splat_composite, cudaFuncAttributeMaxDynamicSharedMemorySize, kPool * (int)sizeof(uint2));
    if (e != cudaSuccess) return e;
    k_splat_composite<<<gt, blk, kPool * sizeof(uint2), st>>>(p);
    *n_launches = 7;
    return cudaGetLastError();
}

cudaError_t ggt_launch_temporal_weight_mask(size_t n, const float* prev_depth, const float* prev_conf, const GgtMaskList& masks,
                                            float beta, float eta, float* out, cudaStream_t st) {
    k_temporal_weight_mask<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, prev_depth, prev_conf, masks, beta, eta, out);
    return cudaGetLastError();
}
