// ggt_weight.cu — step a3: per-pixel depth-variance fusion weight (Eq. 11-12)
//   nu    = sum over the w x w window (w = 7) of min((D0 - D[p,q])^2, clip^2)
//   omega = min(sigma0 * (nu / (w*w))^(-1/2), 1)
// and packing of {depth, omega} into one 8-byte record per pixel so that the integrate kernel needs a single
// gather per voxel.view.  Reading P11: missing / invalid neighbours contribute clip^2; nu == 0 -> omega = 1.
// The 49 terms are added in row-major window order in fp32 (the order the oracle states), so the result is
// bit-reproducible.  The output is padded to (H+1) x (W+1) records, the extra column and row holding {0, 0}.
//
// The kernel is bound by instruction issue (49 x {subtract, square, min, add} per pixel against 12 bytes), so:
//   * one CTA = 64 x 16 pixels, depth tile + 3-pixel halo in shared memory; each thread owns the 2 x 2 pixels
//     (x, y), (x + 32, y), (x, y + 1), (x + 32, y + 1): the two columns run as the two lanes of packed fp32x2
//     instructions (FADD2 / FMUL2: IEEE round-to-nearest per lane, so each lane is the scalar computation) and
//     are stored interleaved, so one LDS.64 fetches a neighbour of both; the two rows share 6 of their 7 tile
//     rows in registers (shared-memory bandwidth is the other limit).  Each pixel still adds its 49 terms in
//     row-major window order;
//   * invalid and out-of-image neighbours are stored in the tile as NaN: (D0 - NaN)^2 = NaN and min(NaN, c2) = c2
//     (min.f32 returns the non-NaN operand), which is exactly "contributes clip^2" with no validity test, and it
//     matches the oracle's `dd < c2 ? dd : c2` for every other input as well (inf, huge values);
//   * all views of a call are one launch (blockIdx.z = view); a view that brings its own per-pixel weights (the
//     previous output depth with Eq. 13's weight, ggt_*_weighted) is only packed.
#include "ggt_internal.h"
#include "ggt_packed.cuh"

namespace {

constexpr int BW = 64, BH = 16, R = 3;
constexpr int SW = 32 + 2 * R, SH = BH + 2 * R;   // 38 pairs x 22 rows

__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// Eq. 11: omega = min(sigma0 / sqrt(nu / 49), 1).  The three IEEE operations run as their branch-free fast paths
// (ggt_packed.cuh; verified bit for bit against __fdiv_rn / __fsqrt_rn by ggt_selftest_arith) wherever all operands and
// results are normal numbers far from the exponent limits -- every realistic depth map -- and as the compiler's
// intrinsics otherwise.
__device__ __forceinline__ float omega_of(float D0, float nu, float sigma0, int window, bool fast_ok) {
    if (!(D0 > 0.0f)) return 0.0f;
    if (window == 0 || nu == 0.0f) return 1.0f;
    float w;
    if (fast_ok && nu >= 1e-30f && nu <= 1e30f) {
        w = div1_neg(-sigma0, sqrt1(div49(nu)));
    } else {
        const float v = __fdiv_rn(nu, 49.0f);
        const float sd = __fsqrt_rn(v);
        w = __fdiv_rn(sigma0, sd);
    }
    return w < 1.0f ? w : 1.0f;
}

__device__ __forceinline__ float tile_value(const float* __restrict__ depth, int W, int H, int x, int y) {
    float d = __int_as_float(0x7fc00000);                 // NaN: out of image == invalid == contributes clip^2
    if (x >= 0 && x < W && y >= 0 && y < H) {
        const float g = __ldg(depth + (size_t)y * W + x);
        if (g > 0.0f) d = g;
    }
    return d;
}

__device__ __forceinline__ void accumulate(u64& nu, u64 D0, u64 Dn, float c2) {
    const u64 d = sub2(D0, Dn);
    float dd0, dd1;
    upk(mul2(d, d), dd0, dd1);
    nu = add2(nu, pk(fminf(dd0, c2), fminf(dd1, c2)));
}

__global__ void __launch_bounds__(256)
k_weight_map(const GgtWeightParams p) {
    __shared__ u64 s_d[SH][SW + 1];                       // {tile(ly, lx), tile(ly, lx + 32)}
    const GgtWeightView& vw = p.v[blockIdx.z];
    const int W = vw.width, H = vw.height;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int x0 = blockIdx.x * BW, y0 = blockIdx.y * BH;
    if (x0 > W || y0 > H) return;                         // views of different sizes share one grid
    const float* __restrict__ depth = vw.depth;
    if (vw.weight) {                                      // given weights: just pack {D, w} (and the zero padding)
        for (int i = ty * 32 + tx; i < BW * BH; i += 256) {
            const int x = x0 + i % BW, y = y0 + i / BW;
            if (x > W || y > H) continue;
            float2 rec = make_float2(0.0f, 0.0f);
            if (x < W && y < H) {
                const float g = __ldg(depth + (size_t)y * W + x);
                if (g > 0.0f) rec = make_float2(g, __ldg(vw.weight + (size_t)y * W + x));
            }
            vw.out[(size_t)y * ((size_t)W + 1) + x] = rec;
        }
        return;
    }
    for (int i = ty * 32 + tx; i < SW * SH; i += 256) {
        const int lx = i % SW, ly = i / SW;
        const int x = x0 - R + lx, y = y0 - R + ly;
        s_d[ly][lx] = pk(tile_value(depth, W, H, x, y), tile_value(depth, W, H, x + 32, y));
    }
    __syncthreads();
    const int ya = y0 + 2 * ty;                           // rows ya, ya + 1
    if (ya > H) return;
    const u64 Da = s_d[2 * ty + R][tx + R], Db = s_d[2 * ty + 1 + R][tx + R];   // NaN lanes where invalid
    u64 nua = pk(0.0f, 0.0f), nub = pk(0.0f, 0.0f);
    if (p.window != 0) {
#pragma unroll
        for (int r = 0; r < 2 * R + 2; ++r) {             // tile rows 2 ty + r: window row r of pixel a, r - 1 of pixel b
            u64 n[2 * R + 1];
#pragma unroll
            for (int dp = 0; dp < 2 * R + 1; ++dp) n[dp] = s_d[2 * ty + r][tx + dp];
            if (r <= 2 * R) {
#pragma unroll
                for (int dp = 0; dp < 2 * R + 1; ++dp) accumulate(nua, Da, n[dp], p.c2);
            }
            if (r >= 1) {
#pragma unroll
                for (int dp = 0; dp < 2 * R + 1; ++dp) accumulate(nub, Db, n[dp], p.c2);
            }
        }
    }
    float2* __restrict__ out = vw.out;
    const int xs[2] = {x0 + tx, x0 + tx + 32};
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        const int y = ya + rr;
        if (y > H) break;
        float D[2], nu[2];
        upk(rr ? Db : Da, D[0], D[1]);
        upk(rr ? nub : nua, nu[0], nu[1]);
        const size_t row = (size_t)y * ((size_t)W + 1);   // padded record stride (see ggt_integrate.cu gather_core)
#pragma unroll
        for (int l = 0; l < 2; ++l) {
            if (xs[l] > W) continue;
            // the zero row / column the clamped gathers land on, and invalid pixels: {0, 0}
            const bool z = y == H || xs[l] == W || !(D[l] > 0.0f);
            out[row + xs[l]] = z ? make_float2(0.0f, 0.0f) : make_float2(D[l], omega_of(D[l], nu[l], p.sigma0, p.window, p.fast_ok != 0));
        }
    }
}

}  // namespace

cudaError_t ggt_launch_weight_maps(const GgtWeightParams& p, cudaStream_t st) {
    int Wm = 0, Hm = 0;
    for (int k = 0; k < p.n_views; ++k) { Wm = p.v[k].width > Wm ? p.v[k].width : Wm; Hm = p.v[k].height > Hm ? p.v[k].height : Hm; }
    const dim3 blk(32, 8), grd((Wm + 1 + BW - 1) / BW, (Hm + 1 + BH - 1) / BH, p.n_views);   // + the padding column / row
    k_weight_map<<<grd, blk, 0, st>>>(p);
    return cudaGetLastError();
}
