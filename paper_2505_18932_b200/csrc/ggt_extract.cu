// ggt_extract.cu — step a7: per-ray zero-crossing search ("change of sign in the value of s";
// reading P13: first bin pair with T_j > 0 >= T_{j+1} and both weights > 0; linear interpolation in z;
// confidence = interpolated weight), plus the canonical-layout export used by the tests.
//
// One thread per target ray.  The volume is two planes per group, [group][v][u] x {G values of T} and the same for
// W (G = 4 bins fp32, 8 bins fp16): the search reads the T plane only (128-bit words, 512 contiguous bytes per warp
// request), UNROLL groups ahead, over the per-ray range k_integrate left (the groups with an observed bin T <= 0),
// and fetches weights just for the candidates; after each batch a warp vote (__all_sync) ends the march for the warp
// once all 32 rays have their crossing: a warp reads the groups between its front-most hint and its last crossing
// (or the rear-most hint of the rays that have none).
#include "ggt_internal.h"


namespace {

// G values of one plane word (T or W) of a group
template <bool HALF>
__device__ __forceinline__ void unpack(const uint4& w, float* x) {
    if (HALF) {
        const uint32_t c[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&c[i]));
            x[2 * i] = f.x; x[2 * i + 1] = f.y;
        }
    } else {
        x[0] = __uint_as_float(w.x); x[1] = __uint_as_float(w.y); x[2] = __uint_as_float(w.z); x[3] = __uint_as_float(w.w);
    }
}

// W of bin j of this ray (a rare, on-demand load from the W plane)
template <bool HALF>
__device__ __forceinline__ float weight_at(const uint4* wplane, size_t plane, int j) {
    constexpr int G = HALF ? 8 : 4;
    float x[G];
    unpack<HALF>(__ldg(wplane + (size_t)(j / G) * plane), x);
    float r = x[0];
#pragma unroll
    for (int i = 1; i < G; ++i) r = (j % G) == i ? x[i] : r;
    return r;
}

template <bool HALF>
__global__ void __launch_bounds__(256)
k_extract(const __grid_constant__ GgtExtractParams p) {
    constexpr int G = HALF ? 8 : 4;
    constexpr int UNROLL = HALF ? 2 : 4;                 // 128-bit loads in flight per thread: 16 bins per batch
    extern __shared__ float s_z[];                       // z[Dpad]
    const int Dpad = p.n_groups * G;
    for (int i = threadIdx.y * 32 + threadIdx.x; i < Dpad; i += 256) s_z[i] = __ldg(p.tables + i);
    __syncthreads();
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (v >= p.Ht) return;                               // whole warp leaves together (one row per warp)
    const bool live = u < p.Wt;
    const size_t plane = (size_t)p.Wt * p.Ht;
    const uint4* tpl = reinterpret_cast<const uint4*>(p.voxels) + ((size_t)v * p.Wt + (live ? u : 0));   // T plane
    const uint4* wpl = tpl + (size_t)p.n_groups * plane;                                                  // W plane

    // The search runs on the T plane alone (half of the volume's bytes): a candidate is T_{j-1} > 0 >= T_j; only then
    // are the two weights fetched, and the candidate is a crossing if both bins were observed (reading P13).  An
    // unobserved bin holds T = 0, so it ends a positive run as a candidate and is then rejected by its W = 0.
    // k_integrate left, per ray, the range of groups that hold an observed bin with T <= 0 (first | end << 16; end <=
    // first: none).  The far bin of a crossing is such a bin, so the search runs from one group before the first to the
    // last one -- for the warp, from the front-most start to the rear-most end of its 32 rays, which keeps the loads
    // coalesced.  A ray with an empty range has no crossing.
    const uint32_t hw = live ? __ldg(p.hint + ((size_t)v * p.Wt + u)) : 0u;
    const int h_first = (int)(hw & 0xffffu), h_end = min((int)(hw >> 16), p.n_groups);
    bool found = !live || h_end <= h_first;
    const int g_start = max((int)__reduce_min_sync(0xffffffffu, found ? 0xffffu : (unsigned)h_first) - 1, 0) / UNROLL * UNROLL;
    const int g_end = (int)__reduce_max_sync(0xffffffffu, found ? 0u : (unsigned)h_end);
    // the far bin of a crossing lies inside this ray's own range: groups past it are loaded only for other rays of the
    // warp, or not at all (zero words), and must not end a positive run of this ray
    const int j_lim = min(p.D, h_end * G);
    float pT = 0.0f;
    float out_d = 0.0f, out_c = 0.0f;
    int out_b = -1;
    // the G bins of one T word, in order; pT = T of the bin before it
    auto scan = [&](const uint4& word, int j0) {
        float T[G];
        unpack<HALF>(word, T);
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const int j = j0 + i;
            if (!found && pT > 0.0f && !(T[i] > 0.0f) && j < j_lim) {
                const float Wa = weight_at<HALF>(wpl, plane, j - 1), Wb = weight_at<HALF>(wpl, plane, j);
                if (Wa > 0.0f && Wb > 0.0f) {
                    const float pz = s_z[j - 1], z = s_z[j];
                    const float f = __fdiv_rn(pT, __fsub_rn(pT, T[i]));
                    out_d = fmaf(f, __fsub_rn(z, pz), pz);
                    out_c = fmaf(f, __fsub_rn(Wb, Wa), Wa);
                    out_b = j - 1;
                    found = true;
                }
            }
            pT = T[i];
        }
    };
    uint32_t ppos = 0, plast = 0;                        // fp16: "> 0" mask and raw bits of the previous half2
    for (int g = g_start; g < g_end; g += UNROLL) {
        uint4 w[UNROLL];
#pragma unroll
        for (int q = 0; q < UNROLL; ++q)
            w[q] = (g + q < g_end && !found) ? __ldcs(tpl + (size_t)(g + q) * plane) : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int q = 0; q < UNROLL; ++q) {
            if (HALF) {
                // Candidates are found on the binary16 values themselves, two per instruction: pos = 0xffff per half
                // that is > 0 (NaN: no, as in fp32), shifted by one bin against itself; only a word with a candidate
                // is converted and walked bin by bin.
                const uint32_t c[4] = {w[q].x, w[q].y, w[q].z, w[q].w};
                uint32_t cand = 0;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t pos = __hgt2_mask(*reinterpret_cast<const __half2*>(&c[k]), __half2(__ushort_as_half(0), __ushort_as_half(0)));
                    cand |= __funnelshift_l(ppos, pos, 16) & ~pos;
                    ppos = pos;
                }
                if (cand) {
                    pT = __high2float(*reinterpret_cast<const __half2*>(&plast));
                    scan(w[q], (g + q) * G);
                }
                plast = c[3];
            } else {
                // fp32: the same filter with four compares per word; the bin-by-bin walk runs only on a candidate
                const float a = __uint_as_float(w[q].x), b = __uint_as_float(w[q].y), c = __uint_as_float(w[q].z), d = __uint_as_float(w[q].w);
                const bool pa = a > 0.0f, pb = b > 0.0f, pc = c > 0.0f, pd = d > 0.0f;
                if ((pT > 0.0f && !pa) || (pa && !pb) || (pb && !pc) || (pc && !pd)) scan(w[q], (g + q) * G);
                pT = d;
            }
        }
        found = found || g + UNROLL >= h_end;            // every group of this ray's range has been searched
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
    constexpr int G = HALF ? 8 : 4;
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (u >= p.Wt || v >= p.Ht) return;
    const size_t plane = (size_t)p.Wt * p.Ht;
    const size_t ray = (size_t)v * p.Wt + u;
    const uint4* tpl = reinterpret_cast<const uint4*>(p.voxels) + ray;
    const uint4* wpl = tpl + (size_t)p.n_groups * plane;
    for (int g = 0; g < p.n_groups; ++g) {
        float T[G], Wv[G];
        unpack<HALF>(tpl[(size_t)g * plane], T);
        unpack<HALF>(wpl[(size_t)g * plane], Wv);
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
    const int G = dtype == GGT_F16 ? 8 : 4;
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
