// ggt_extract.cu — step a7: per-ray zero-crossing search ("change of sign in the value of s";
// reading P13: first bin pair with T_j > 0 >= T_{j+1} and both weights > 0; linear interpolation in z;
// confidence = interpolated weight), plus the canonical-layout export used by the tests.
//
// One thread per target ray.  The volume layout [group][v][u][G][{T,W}] makes every load a 128-bit word and
// every warp request 512 contiguous bytes.  Loads are issued UNROLL groups ahead; after each batch a warp
// vote (__all_sync) ends the march for the warp once all 32 rays have their crossing, so the kernel reads
// the volume only up to the front-most surface instead of all of it.
#include "ggt_internal.h"

namespace {

template <bool HALF>
__device__ __forceinline__ void unpack(const uint4& w, float* T, float* Wv) {
    if (HALF) {
        const uint32_t a[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&a[i]));
            T[i] = f.x; Wv[i] = f.y;
        }
    } else {
        T[0] = __uint_as_float(w.x); Wv[0] = __uint_as_float(w.y);
        T[1] = __uint_as_float(w.z); Wv[1] = __uint_as_float(w.w);
    }
}

template <bool HALF>
__global__ void __launch_bounds__(256)
k_extract(const __grid_constant__ GgtExtractParams p) {
    constexpr int G = HALF ? 4 : 2;
    constexpr int UNROLL = 4;
    extern __shared__ float s_z[];                       // z[Dpad]
    const int Dpad = p.n_groups * G;
    for (int i = threadIdx.y * 32 + threadIdx.x; i < Dpad; i += 256) s_z[i] = __ldg(p.tables + i);
    __syncthreads();
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (v >= p.Ht) return;                               // whole warp leaves together (one row per warp)
    const bool live = u < p.Wt;
    const size_t plane = (size_t)p.Wt * p.Ht;
    const uint4* vox = reinterpret_cast<const uint4*>(p.voxels) + ((size_t)v * p.Wt + (live ? u : 0));

    bool found = !live;
    float pT = 0.0f, pW = 0.0f, pz = 0.0f;
    float out_d = 0.0f, out_c = 0.0f;
    int out_b = -1;
    for (int g = 0; g < p.n_groups; g += UNROLL) {
        uint4 w[UNROLL];
#pragma unroll
        for (int q = 0; q < UNROLL; ++q)
            w[q] = (g + q < p.n_groups && !found) ? __ldcs(vox + (size_t)(g + q) * plane) : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int q = 0; q < UNROLL; ++q) {
            float T[G], Wv[G];
            unpack<HALF>(w[q], T, Wv);
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int j = (g + q) * G + i;
                const float z = s_z[min(j, Dpad - 1)];
                const bool hit = !found && (j > 0) && (j < p.D) && (pW > 0.0f) && (Wv[i] > 0.0f) && (pT > 0.0f) &&
                                 !(T[i] > 0.0f);
                if (hit) {
                    const float f = __fdiv_rn(pT, __fsub_rn(pT, T[i]));
                    out_d = fmaf(f, __fsub_rn(z, pz), pz);
                    out_c = fmaf(f, __fsub_rn(Wv[i], pW), pW);
                    out_b = j - 1;
                    found = true;
                }
                pT = T[i]; pW = Wv[i]; pz = z;
            }
        }
        if (__all_sync(0xffffffffu, found)) break;
    }
    if (!live) return;
    const size_t o = (size_t)v * p.Wt + u;
    if (p.depth) p.depth[o] = out_d;
    if (p.conf) p.conf[o] = out_c;
    if (p.bin) p.bin[o] = out_b;
}

template <bool HALF>
__global__ void __launch_bounds__(256)
k_export(GgtExtractParams p, float* __restrict__ T_out, float* __restrict__ W_out) {
    constexpr int G = HALF ? 4 : 2;
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (u >= p.Wt || v >= p.Ht) return;
    const size_t plane = (size_t)p.Wt * p.Ht;
    const size_t ray = (size_t)v * p.Wt + u;
    const uint4* vox = reinterpret_cast<const uint4*>(p.voxels) + ray;
    for (int g = 0; g < p.n_groups; ++g) {
        float T[G], Wv[G];
        unpack<HALF>(vox[(size_t)g * plane], T, Wv);
        for (int i = 0; i < G; ++i) {
            const int j = g * G + i;
            if (j < p.D) {
                T_out[ray * p.D + j] = T[i];
                W_out[ray * p.D + j] = Wv[i];
            }
        }
    }
}

}  // namespace

cudaError_t ggt_launch_extract(const GgtExtractParams& p, int dtype, cudaStream_t st) {
    const dim3 blk(32, 8), grd((p.Wt + 31) / 32, (p.Ht + 7) / 8);
    const int G = dtype == GGT_F16 ? 4 : 2;
    const size_t smem = (size_t)p.n_groups * G * sizeof(float);
    if (dtype == GGT_F16) k_extract<true><<<grd, blk, smem, st>>>(p);
    else k_extract<false><<<grd, blk, smem, st>>>(p);
    return cudaGetLastError();
}

cudaError_t ggt_launch_export(const GgtExtractParams& p, int dtype, float* T, float* W, cudaStream_t st) {
    const dim3 blk(32, 8), grd((p.Wt + 31) / 32, (p.Ht + 7) / 8);
    if (dtype == GGT_F16) k_export<true><<<grd, blk, 0, st>>>(p, T, W);
    else k_export<false><<<grd, blk, 0, st>>>(p, T, W);
    return cudaGetLastError();
}
