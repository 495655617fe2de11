// ggt_features.cu — SURVEY.md 8(f) row f-4: geometry features of the guidance depth for the blending network's input
// (A.4 items 5-8): per input view k and target pixel, the dot product of the input-view ray with the
// normal of the TSDF depth (5) and with the target view ray (6), and the spatially constant camera distance (7) and
// optical-axis dot product (8).  Readings G1-G4: surface point p = D ((uc - cx)/fx, (vc - cy)/fy, 1);
// normal = normalised cross product of central differences of p (one-sided next to holes and borders, undefined
// without a neighbour in either axis), oriented towards the camera; rays = unit vectors from the camera centres to the
// surface point.  Output [4 K][H][W] fp32, planar.
// One thread per pixel: 5 depth loads (L1), 4 K coalesced plane stores = 16 K bytes per pixel written: HBM-bound.
// IEEE operations in the oracle's order (plain intrinsics; sqrt and divisions are a handful per pixel).
#include "ggt_internal.h"

namespace {

struct V3 { float x, y, z; };

__device__ __forceinline__ float dot3(V3 a, V3 b) { return fmaf(a.z, b.z, fmaf(a.y, b.y, __fmul_rn(a.x, b.x))); }
__device__ __forceinline__ V3 sub3(V3 a, V3 b) { return {__fsub_rn(a.x, b.x), __fsub_rn(a.y, b.y), __fsub_rn(a.z, b.z)}; }
// w = R^T q (R row-major)
__device__ __forceinline__ V3 rt_mul(const float* R, V3 q) {
    return {fmaf(R[6], q.z, fmaf(R[3], q.y, __fmul_rn(R[0], q.x))), fmaf(R[7], q.z, fmaf(R[4], q.y, __fmul_rn(R[1], q.x))),
            fmaf(R[8], q.z, fmaf(R[5], q.y, __fmul_rn(R[2], q.x)))};
}

__device__ __forceinline__ float depth_at(const GgtFeatureParams& p, int u, int v) {
    if (u < 0 || v < 0 || u >= p.W || v >= p.H) return 0.0f;
    return __ldg(p.depth + (size_t)v * p.W + u);
}
__device__ __forceinline__ V3 cam_point(const GgtFeatureParams& p, int u, int v, float d) {
    const float uc = __fadd_rn((float)u, 0.5f), vc = __fadd_rn((float)v, 0.5f);
    return {__fmul_rn(d, __fdiv_rn(__fsub_rn(uc, p.cx), p.fx)), __fmul_rn(d, __fdiv_rn(__fsub_rn(vc, p.cy), p.fy)), d};
}
// difference along one axis: central where both neighbours have depth, else one-sided, else undefined
__device__ __forceinline__ bool diff_axis(const GgtFeatureParams& p, int u, int v, int du, int dv, V3 centre, V3& out) {
    const float dp = depth_at(p, u + du, v + dv), dm = depth_at(p, u - du, v - dv);
    const bool hp = dp > 0.0f, hm = dm > 0.0f;
    if (!hp && !hm) return false;
    const V3 a = hp ? cam_point(p, u + du, v + dv, dp) : centre;
    const V3 b = hm ? cam_point(p, u - du, v - dv, dm) : centre;
    out = sub3(a, b);
    return true;
}

__global__ void __launch_bounds__(256)
k_features(const __grid_constant__ GgtFeatureParams p) {
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (u >= p.W || v >= p.H) return;
    const size_t i = (size_t)v * p.W + u;
    const float d = depth_at(p, u, v);
    bool ok = d > 0.0f;
    V3 n = {0.0f, 0.0f, 0.0f}, P = {0.0f, 0.0f, 0.0f}, rt = {0.0f, 0.0f, 0.0f};
    if (ok) {
        const V3 pc = cam_point(p, u, v, d);
        V3 dx, dy;
        ok = diff_axis(p, u, v, 1, 0, pc, dx);
        ok = diff_axis(p, u, v, 0, 1, pc, dy) && ok;
        if (ok) {
            V3 c = {__fsub_rn(__fmul_rn(dx.y, dy.z), __fmul_rn(dx.z, dy.y)), __fsub_rn(__fmul_rn(dx.z, dy.x), __fmul_rn(dx.x, dy.z)),
                    __fsub_rn(__fmul_rn(dx.x, dy.y), __fmul_rn(dx.y, dy.x))};
            if (dot3(c, pc) > 0.0f) c = {-c.x, -c.y, -c.z};                   // towards the camera
            const float l2 = dot3(c, c);
            ok = l2 > 0.0f;
            if (ok) {
                const float l = __fsqrt_rn(l2);
                const V3 nc = {__fdiv_rn(c.x, l), __fdiv_rn(c.y, l), __fdiv_rn(c.z, l)};
                n = rt_mul(p.R, nc);
                P = rt_mul(p.R, sub3(pc, V3{p.t[0], p.t[1], p.t[2]}));
            }
        }
    }
    if (ok) {
        const V3 dt = sub3(P, V3{p.Ct[0], p.Ct[1], p.Ct[2]});
        const float l = __fsqrt_rn(dot3(dt, dt));
        ok = l > 0.0f;
        if (ok) rt = {__fdiv_rn(dt.x, l), __fdiv_rn(dt.y, l), __fdiv_rn(dt.z, l)};
    }
    const size_t plane = (size_t)p.W * p.H;
    for (int k = 0; k < p.n_views; ++k) {
        float f5 = 0.0f, f6 = 0.0f;
        if (ok) {
            const V3 dk = sub3(P, V3{p.v[k].C[0], p.v[k].C[1], p.v[k].C[2]});
            const float l = __fsqrt_rn(dot3(dk, dk));
            if (l > 0.0f) {
                const V3 rk = {__fdiv_rn(dk.x, l), __fdiv_rn(dk.y, l), __fdiv_rn(dk.z, l)};
                f5 = dot3(rk, n);                                              // item 5
                f6 = dot3(rk, rt);                                             // item 6
            }
        }
        __stcs(p.out + (size_t)k * plane + i, f5);
        __stcs(p.out + (size_t)(p.n_views + k) * plane + i, f6);
        __stcs(p.out + (size_t)(2 * p.n_views + k) * plane + i, p.v[k].dist);  // item 7
        __stcs(p.out + (size_t)(3 * p.n_views + k) * plane + i, p.v[k].axes);  // item 8
    }
}

}  // namespace

cudaError_t ggt_launch_features(const GgtFeatureParams& p, cudaStream_t st) {
    const dim3 blk(32, 8), grd((p.W + 31) / 32, (p.H + 7) / 8);
    k_features<<<grd, blk, 0, st>>>(p);
    return cudaGetLastError();
}
