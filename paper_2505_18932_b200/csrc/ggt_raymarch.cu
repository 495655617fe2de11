// ggt_raymarch.cu — the paper's own schedule: image-based TSDF evaluated on the fly along
// each target ray, no volume.  PAPER.md:75 ("integrates depth along each ray on the fly and, thus, avoids creating
// an explicit 3D voxel grid") and PAPER.md:348 ("We advance along the ray with a step size of 0.8s until a surface
// intersection is detected.  This is indicated by a change of sign in the value of s.  We subsequently perform
// three steps of a bisection search to refine the intersection depth."), tau = 0.02 m.
//
// One thread per target ray.  s(z) is the per-sample arithmetic of k_integrate (projection, nearest sample,
// Eq. 9, cut, Eq. 10, normalised: reading P2) at an arbitrary depth z instead of a bin; the readings for what the
// paper leaves open are M1-M6 of DESIGN.md (start at z_near, min_step, unobserved samples advance like free space,
// a crossing needs an observed positive predecessor, bisection ends on an unobserved midpoint, depth = bracket
// midpoint).  The march of a ray is one dependent chain (z_{n+1} needs s(z_n), which needs V gathers), so:
//   * the V views of one evaluation are the instruction-level parallelism: their projections run as packed fp32x2
//     instructions over PAIRS OF VIEWS (the same IEEE operations per lane as the scalar order the oracle states) and
//     their V gathers are in flight together; Eq. 10's sums are then accumulated in view order;
//   * occupancy covers the rest: <= 64 registers, 4 CTAs of 256 threads per SM;
//   * rays of a warp leave the loop at different evaluations; a warp retires when its last ray does (neighbouring
//     rays see neighbouring depths, so the spread is small except across depth edges).
#include "ggt_internal.h"
#include "ggt_packed.cuh"

namespace {

struct RayView {            // per-ray, per-view constants: -(H_k rows 0, 1 . (uc, vc, 1)) and H_k row 2 . (uc, vc, 1)
    float nbx, nby, bw;
};

// clamped nearest-pixel gather on the zero-padded {depth, omega} map (see ggt_integrate.cu gather_core)
template <bool WCHK>
__device__ __forceinline__ float2 gather1(const GgtViewParams& vp, float fx, float fy, float w) {
    unsigned ix = min((unsigned)(__float_as_int(fx) - kMagicBits), (unsigned)vp.width);
    const unsigned iy = min((unsigned)(__float_as_int(fy) - kMagicBits), (unsigned)vp.height);
    if (WCHK) ix = w >= 1e-6f ? ix : (unsigned)vp.width;         // w < 1e-6: skip == the zero padding column
    return __ldg(vp.map + (iy * vp.stride + ix));
}

// Eq. 9-10 for one gathered sample, in view order: A += omega min(s, tau), W += omega, omega = 0 behind the cut
__device__ __forceinline__ void blend1(float w, float2 m, float tau, float& NA, float& Wn) {
    const float ns = __fsub_rn(w, m.x);                          // -s_k
    const float om = ns > tau ? 0.0f : m.y;                      // omega_k = 0 if s_k < -tau
    const float nc = fmaxf(ns, -tau);                            // -min(s_k, tau)
    NA = fmaf(om, nc, NA);
    Wn = __fadd_rn(Wn, om);
}

// One evaluation of s at depth z: returns Wn, and NA = -sum(omega c).
// WCHK: keep the per-sample w >= 1e-6 test (dropped when it holds at z_near and z_far for every view of every ray
// of the warp: w_k(z) is monotone in z).  SHW: w_k(z) has the same bits in every view (parallel rig, see
// ggt_integrate.cu), so it and its reciprocal are computed once per evaluation.
template <int NV, bool WCHK, bool SHW>
__device__ __forceinline__ void eval_s(const GgtRaymarchParams& p, const RayView* rv, float z, float& NA, float& Wn) {
    constexpr int NP = NV / 2;
    float2 m[NV > 0 ? NV : 1];
    float wv[NV > 0 ? NV : 1];
    float w_sh = 0.0f, nr_sh = 0.0f;
    if (SHW) {
        w_sh = fmaf(z, rv[0].bw, p.v[0].e2);
        nr_sh = neg_rcp1(w_sh);
    }
#pragma unroll
    for (int q = 0; q < NP; ++q) {                               // views 2q, 2q + 1 as the two lanes
        const int k0 = 2 * q, k1 = 2 * q + 1;
        const u64 zz = bc(z);
        const u64 nxx = fma2(zz, pk(rv[k0].nbx, rv[k1].nbx), pk(p.v[k0].ne[0], p.v[k1].ne[0]));
        const u64 nyy = fma2(zz, pk(rv[k0].nby, rv[k1].nby), pk(p.v[k0].ne[1], p.v[k1].ne[1]));
        u64 nr;
        if (SHW) {
            wv[k0] = w_sh; wv[k1] = w_sh;
            nr = bc(nr_sh);
        } else {
            const u64 ww = fma2(zz, pk(rv[k0].bw, rv[k1].bw), pk(p.v[k0].e2, p.v[k1].e2));  // z_k of Eq. 9
            nr = neg_rcp2(ww);
            upk(ww, wv[k0], wv[k1]);
        }
        const u64 fx = add2_rd(mul2(nxx, nr), bc(kMagic));       // floor(px) in the low mantissa bits
        const u64 fy = add2_rd(mul2(nyy, nr), bc(kMagic));
        float fx0, fx1, fy0, fy1;
        upk(fx, fx0, fx1); upk(fy, fy0, fy1);
        m[k0] = gather1<WCHK>(p.v[k0], fx0, fy0, wv[k0]);
        m[k1] = gather1<WCHK>(p.v[k1], fx1, fy1, wv[k1]);
    }
    if (NV & 1) {                                                // odd view count: the last view alone
        const int k = NV - 1;
        const float nx = fmaf(z, rv[k].nbx, p.v[k].ne[0]);
        const float ny = fmaf(z, rv[k].nby, p.v[k].ne[1]);
        const float w = SHW ? w_sh : fmaf(z, rv[k].bw, p.v[k].e2);
        const float nr = SHW ? nr_sh : neg_rcp1(w);
        float fx, fy;
        asm("add.rm.f32 %0, %1, %2;" : "=f"(fx) : "f"(__fmul_rn(nx, nr)), "f"(kMagic));
        asm("add.rm.f32 %0, %1, %2;" : "=f"(fy) : "f"(__fmul_rn(ny, nr)), "f"(kMagic));
        wv[k] = w;
        m[k] = gather1<WCHK>(p.v[k], fx, fy, w);
    }
    NA = 0.0f; Wn = 0.0f;
#pragma unroll
    for (int k = 0; k < NV; ++k) blend1(wv[k], m[k], p.tau, NA, Wn);
}

// generic view count: one view at a time, per-ray constants recomputed (no register arrays)
__device__ __forceinline__ void eval_s_generic(const GgtRaymarchParams& p, float uc, float vc, float z, float& NA, float& Wn) {
    NA = 0.0f; Wn = 0.0f;
    for (int k = 0; k < p.n_views; ++k) {
        const GgtViewParams& vp = p.v[k];
        const float nbx = fmaf(vp.nh[0], uc, fmaf(vp.nh[1], vc, vp.nh[2]));
        const float nby = fmaf(vp.nh[3], uc, fmaf(vp.nh[4], vc, vp.nh[5]));
        const float bw = fmaf(vp.h2[0], uc, fmaf(vp.h2[1], vc, vp.h2[2]));
        const float nx = fmaf(z, nbx, vp.ne[0]);
        const float ny = fmaf(z, nby, vp.ne[1]);
        const float w = fmaf(z, bw, vp.e2);
        const float nr = neg_rcp1(w);
        float fx, fy;
        asm("add.rm.f32 %0, %1, %2;" : "=f"(fx) : "f"(__fmul_rn(nx, nr)), "f"(kMagic));
        asm("add.rm.f32 %0, %1, %2;" : "=f"(fy) : "f"(__fmul_rn(ny, nr)), "f"(kMagic));
        blend1(w, gather1<true>(vp, fx, fy, w), p.tau, NA, Wn);
    }
}

template <int NV, bool WCHK, bool SHW>
__device__ __forceinline__ void march_ray(const GgtRaymarchParams& p, int u, int v, float uc, float vc) {
    RayView rv[NV > 0 ? NV : 1];
    if (NV > 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            rv[k].nbx = fmaf(p.v[k].nh[0], uc, fmaf(p.v[k].nh[1], vc, p.v[k].nh[2]));
            rv[k].nby = fmaf(p.v[k].nh[3], uc, fmaf(p.v[k].nh[4], vc, p.v[k].nh[5]));
            rv[k].bw = fmaf(p.v[k].h2[0], uc, fmaf(p.v[k].h2[1], vc, p.v[k].h2[2]));
        }
    }
    auto eval = [&](float z, float& NA, float& Wn) {
        if (NV > 0) eval_s<NV, WCHK, SHW>(p, rv, z, NA, Wn);
        else eval_s_generic(p, uc, vc, z, NA, Wn);
    };
    const float free_step = fmaxf(__fmul_rn(p.step_scale, p.tau), p.min_step);          // M3
    float z = p.z_near, za = 0.0f, zb = 0.0f, Wb = 0.0f;
    bool prev_pos = false, hit = false;
    int n = 0;
    // The loop body is written with selects instead of branches (one exit test per evaluation): s is formed even
    // when nothing was observed (the quotient is then NaN or inf and is never selected).
    while (n < p.max_evals && !(z > p.z_far)) {                                         // M1
        float NA, Wn;
        eval(z, NA, Wn);
        ++n;
        const bool observed = Wn > 0.0f;
        const float s = div1_neg(NA, Wn);                                               // s = A / W (reading P2)
        const bool pos = observed && s > 0.0f;
        if (observed && !pos && prev_pos) { zb = z; Wb = Wn; hit = true; break; }       // M4: change of sign
        const float adv = fmaxf(__fmul_rn(p.step_scale, s), p.min_step);                // M2
        const float step = pos ? adv : (observed ? p.min_step : free_step);             // M4 / M3
        za = pos ? z : za;
        prev_pos = pos;
        z = __fadd_rn(z, step);
    }
    float d = 0.0f, c = 0.0f;
    if (hit) {
        for (int i = 0; i < p.n_bisect; ++i) {                                          // M5
            const float m = __fmul_rn(0.5f, __fadd_rn(za, zb));
            float NA, Wn;
            eval(m, NA, Wn);
            ++n;
            if (!(Wn > 0.0f)) break;
            const float s = div1_neg(NA, Wn);
            if (s > 0.0f) za = m; else { zb = m; Wb = Wn; }
        }
        d = __fmul_rn(0.5f, __fadd_rn(za, zb));
        c = Wb;                                                                         // M6
    }
    const size_t o = (size_t)v * p.Wt + u;
    if (p.depth) p.depth[o] = d;
    if (p.conf) p.conf[o] = c;
    if (p.steps) p.steps[o] = n;
}

template <int NV>
__global__ void __launch_bounds__(256, 4)
k_raymarch(const __grid_constant__ GgtRaymarchParams p) {
    const int u_raw = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (v >= p.Ht) return;                                       // whole warp (one row per warp)
    const bool live = u_raw < p.Wt;
    const int u = live ? u_raw : p.Wt - 1;                       // ragged tail lanes shadow the last pixel (same value, same address)
    const float uc = __fadd_rn((float)u, 0.5f), vc = __fadd_rn((float)v, 0.5f);
    bool wok = NV > 0;
    if (NV > 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const float b = fmaf(p.v[k].h2[0], uc, fmaf(p.v[k].h2[1], vc, p.v[k].h2[2]));
            wok = wok && (fmaf(p.z_near, b, p.v[k].e2) >= 1e-6f) && (fmaf(p.z_far, b, p.v[k].e2) >= 1e-6f);
        }
    }
    if (NV > 0 && __all_sync(0xffffffffu, wok)) {
        if (p.shared_w) march_ray<NV, false, true>(p, u, v, uc, vc);
        else march_ray<NV, false, false>(p, u, v, uc, vc);
    } else {
        march_ray<NV, true, false>(p, u, v, uc, vc);
    }
}

}  // namespace

cudaError_t ggt_launch_raymarch(const GgtRaymarchParams& p, cudaStream_t st) {
    const dim3 blk(32, 8), grd((p.Wt + 31) / 32, (p.Ht + 7) / 8);
    switch (p.n_views) {
        case 1: k_raymarch<1><<<grd, blk, 0, st>>>(p); break;
        case 2: k_raymarch<2><<<grd, blk, 0, st>>>(p); break;
        case 3: k_raymarch<3><<<grd, blk, 0, st>>>(p); break;
        case 4: k_raymarch<4><<<grd, blk, 0, st>>>(p); break;
        case 5: k_raymarch<5><<<grd, blk, 0, st>>>(p); break;     // V + the previous output depth (Eq. 3)
        case 6: k_raymarch<6><<<grd, blk, 0, st>>>(p); break;
        case 7: k_raymarch<7><<<grd, blk, 0, st>>>(p); break;
        case 8: k_raymarch<8><<<grd, blk, 0, st>>>(p); break;
        case 9: k_raymarch<9><<<grd, blk, 0, st>>>(p); break;
        default: k_raymarch<0><<<grd, blk, 0, st>>>(p); break;
    }
    return cudaGetLastError();
}
