// ggt_weight.cu — step a3: per-pixel depth-variance fusion weight (Eq. 11-12)
//   nu    = sum over the w x w window (w = 7) of min((D0 - D[p,q])^2, clip^2)
//   omega = min(sigma0 * (nu / (w*w))^(-1/2), 1)
// and packing of {depth, omega} into one 8-byte record per pixel so that the integrate kernel needs a single
// gather per voxel.view.  Reading P11: missing / invalid neighbours contribute clip^2; nu == 0 -> omega = 1.
// The 49 terms are added in row-major window order in fp32 (the order the oracle states), so the result is
// bit-reproducible.  The output is padded to (H+1) x (W+1) records, the extra column and row holding {0, 0}.
// One CTA = 32 x 8 pixels, depth tile + 3-pixel halo staged in shared memory.
#include "ggt_internal.h"

namespace {

constexpr int BW = 32, BH = 8, R = 3;
constexpr int SW = BW + 2 * R, SH = BH + 2 * R;   // 38 x 14

__global__ void __launch_bounds__(BW * BH)
k_weight_map(int W, int H, const float* __restrict__ depth, float2* __restrict__ out, float sigma0, float c2,
             int window) {
    __shared__ float s_d[SH][SW + 1];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int x0 = blockIdx.x * BW, y0 = blockIdx.y * BH;
    for (int i = ty * BW + tx; i < SW * SH; i += BW * BH) {
        const int lx = i % SW, ly = i / SW;
        const int x = x0 - R + lx, y = y0 - R + ly;
        float d = 0.0f;                                   // out of image == invalid == contributes clip^2
        if (x >= 0 && x < W && y >= 0 && y < H) d = __ldg(depth + (size_t)y * W + x);
        s_d[ly][lx] = d;
    }
    __syncthreads();
    const int x = x0 + tx, y = y0 + ty;
    if (x > W || y > H) return;
    const size_t Ws = (size_t)W + 1;                      // padded record stride (see ggt_integrate.cu view_pair)
    if (x == W || y == H) {                               // zero column / row the clamped gathers land on
        out[(size_t)y * Ws + x] = make_float2(0.0f, 0.0f);
        return;
    }
    const float D0 = s_d[ty + R][tx + R];
    float omega;
    if (!(D0 > 0.0f)) {
        omega = 0.0f;
    } else if (window == 0) {
        omega = 1.0f;
    } else {
        float nu = 0.0f;
#pragma unroll
        for (int dq = 0; dq < 2 * R + 1; ++dq)
#pragma unroll
            for (int dp = 0; dp < 2 * R + 1; ++dp) {
                const float Dn = s_d[ty + dq][tx + dp];
                const float d = __fsub_rn(D0, Dn);
                const float dd = __fmul_rn(d, d);
                float m = dd < c2 ? dd : c2;
                m = Dn > 0.0f ? m : c2;
                nu = __fadd_rn(nu, m);
            }
        if (nu == 0.0f) {
            omega = 1.0f;
        } else {
            const float v = __fdiv_rn(nu, 49.0f);
            const float sd = __fsqrt_rn(v);
            const float w = __fdiv_rn(sigma0, sd);
            omega = w < 1.0f ? w : 1.0f;
        }
    }
    out[(size_t)y * Ws + x] = make_float2(D0 > 0.0f ? D0 : 0.0f, omega);   // invalid -> {0, 0}: zero weight, finite depth
}

}  // namespace

cudaError_t ggt_launch_weight_map(int W, int H, const float* depth, float2* out, float sigma0, float clip,
                                  int window, cudaStream_t st) {
    const dim3 blk(BW, BH), grd((W + 1 + BW - 1) / BW, (H + 1 + BH - 1) / BH);   // + the padding column / row
    const float c2 = clip * clip;   // one fp32 multiply, as the oracle states it
    k_weight_map<<<grd, blk, 0, st>>>(W, H, depth, out, sigma0, c2, window);
    return cudaGetLastError();
}
