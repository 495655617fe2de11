// ggt_features.cu — SURVEY.md 8(f) row f-4: geometry features of the guidance depth for the blending network's input
// (A.4 items 5-8): per input view k and target pixel, the dot product of the input-view ray with the
// normal of the TSDF depth (5) and with the target view ray (6), and the spatially constant camera distance (7) and
// optical-axis dot product (8).  Readings G1-G4: surface point p = D ((uc - cx)/fx, (vc - cy)/fy, 1);
// normal = normalised cross product of central differences of p (one-sided next to holes and borders, undefined
// without a neighbour in either axis), oriented towards the camera; rays = unit vectors from the camera centres to the
// surface point.  Output [4 K][H][W] fp32, planar.
// One thread per pixel: 5 depth loads (L1), 4 K coalesced plane stores = 16 K bytes per pixel written: HBM-bound.
// IEEE operations in the oracle's order; the ~25 divisions and 2 + K square roots per pixel are what the kernel's time
// goes to, so they run as the branch-free fast paths wherever their operands are mid-range (see div_ieee below).
#include "ggt_internal.h"
#include "ggt_packed.cuh"

namespace {

struct V3 { float x, y, z; };

__device__ __forceinline__ float dot3(V3 a, V3 b) { return fmaf(a.z, b.z, fmaf(a.y, b.y, __fmul_rn(a.x, b.x))); }
__device__ __forceinline__ V3 sub3(V3 a, V3 b) { return {__fsub_rn(a.x, b.x), __fsub_rn(a.y, b.y), __fsub_rn(a.z, b.z)}; }
// w = R^T q (R row-major)
__device__ __forceinline__ V3 rt_mul(const float* R, V3 q) {
    return {fmaf(R[6], q.z, fmaf(R[3], q.y, __fmul_rn(R[0], q.x))), fmaf(R[7], q.z, fmaf(R[4], q.y, __fmul_rn(R[1], q.x))),
            fmaf(R[8], q.z, fmaf(R[5], q.y, __fmul_rn(R[2], q.x)))};
}

// IEEE a / b and sqrt(x): the branch-free fast paths of ggt_packed.cuh (verified bit for bit by ggt_selftest_arith) where
// every operand and result is a normal number far from the exponent limits, the compiler's intrinsics otherwise.
__device__ __forceinline__ bool mid(float x) { return x >= 1e-30f && x <= 1e30f; }
__device__ __forceinline__ float div_ieee(float a, float b, bool fast) { return fast ? div1_neg(-a, b) : __fdiv_rn(a, b); }
// v / |v| given l = |v| and whether l is mid-range: |v_i| <= l, so each quotient is 0 or a normal number
__device__ __forceinline__ V3 unit3(V3 v, float l, bool fast) { return {div_ieee(v.x, l, fast), div_ieee(v.y, l, fast), div_ieee(v.z, l, fast)}; }
__device__ __forceinline__ float sqrt_ieee(float x, bool fast) { return fast ? sqrt1(x) : __fsqrt_rn(x); }

__device__ __forceinline__ float depth_at(const GgtFeatureParams& p, int u, int v) {
    if (u < 0 || v < 0 || u >= p.W || v >= p.H) return 0.0f;
    return __ldg(p.depth + (size_t)v * p.W + u);
}
__device__ __forceinline__ V3 cam_point(const GgtFeatureParams& p, int u, int v, float d) {
    const float uc = __fadd_rn((float)u, 0.5f), vc = __fadd_rn((float)v, 0.5f);
    return {__fmul_rn(d, div_ieee(__fsub_rn(uc, p.cx), p.fx, p.fast_ok != 0)), __fmul_rn(d, div_ieee(__fsub_rn(vc, p.cy), p.fy, p.fast_ok != 0)), d};
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
                const bool f = mid(l2);
                const V3 nc = unit3(c, sqrt_ieee(l2, f), f);
                n = rt_mul(p.R, nc);
                P = rt_mul(p.R, sub3(pc, V3{p.t[0], p.t[1], p.t[2]}));
            }
        }
    }
    if (ok) {
        const V3 dt = sub3(P, V3{p.Ct[0], p.Ct[1], p.Ct[2]});
        const float l2 = dot3(dt, dt);
        const bool f = mid(l2);
        const float l = sqrt_ieee(l2, f);
        ok = l > 0.0f;
        if (ok) rt = unit3(dt, l, f);
    }
    const size_t plane = (size_t)p.W * p.H;
    for (int k = 0; k < p.n_views; ++k) {
        float f5 = 0.0f, f6 = 0.0f;
        if (ok) {
            const V3 dk = sub3(P, V3{p.v[k].C[0], p.v[k].C[1], p.v[k].C[2]});
            const float l2 = dot3(dk, dk);
            const bool f = mid(l2);
            const float l = sqrt_ieee(l2, f);
            if (l > 0.0f) {
                const V3 rk = unit3(dk, l, f);
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
