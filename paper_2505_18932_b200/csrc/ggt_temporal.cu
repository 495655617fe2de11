// ggt_temporal.cu — SURVEY.md 8(f) row f-2: the fusion weight of the previous output depth (Eq. 3,
// PAPER.md:352-360 Eq. 13-14).  D^{t-1} enters the TSDF of frame t as one more depth view with its own pose and the
// per-pixel weight
//   omega_tmp^t = min(beta * omega_acc^t * max(1 - M^t, 0), eta),   omega_acc^t = omega_tmp^{t-1} + sum_k omega_k^{t-1}
// where omega_acc is the confidence the previous frame's raymarch / extract returned (the sum of all fusion weights at
// its surface point) and M^t is the difference mask in the novel view.  Reading F1: the paper forward-splats
// the K masks M_k^t and takes the maximum; here the surface point of each pixel of D^{t-1} is projected into every input
// view (A.1's projection, nearest pixel) and M^t is the maximum of M_k^t over the views it lands in (0 if none).
// One thread per pixel of D^{t-1}: 8 bytes read, 4 written, V mask gathers served by L2: HBM-bound and tiny next to
// the fusion itself.  IEEE operations in the oracle's order (plain intrinsics: this kernel is not issue-bound).
#include "ggt_internal.h"

namespace {

__global__ void __launch_bounds__(256)
k_temporal_weight(const __grid_constant__ GgtTemporalParams p) {
    const int u = blockIdx.x * 32 + threadIdx.x;
    const int v = blockIdx.y * 8 + threadIdx.y;
    if (u >= p.Wt || v >= p.Ht) return;
    const size_t i = (size_t)v * p.Wt + u;
    const float d = __ldg(p.prev_depth + i), acc = __ldg(p.prev_conf + i);
    float wt = 0.0f;
    if (d > 0.0f && acc > 0.0f) {
        const float uc = __fadd_rn((float)u, 0.5f), vc = __fadd_rn((float)v, 0.5f);
        float Mmax = 0.0f;
        for (int k = 0; k < p.n_views; ++k) {
            const GgtMaskView& vw = p.v[k];
            const float bx = fmaf(vw.h[0], uc, fmaf(vw.h[1], vc, vw.h[2]));
            const float by = fmaf(vw.h[3], uc, fmaf(vw.h[4], vc, vw.h[5]));
            const float bw = fmaf(vw.h[6], uc, fmaf(vw.h[7], vc, vw.h[8]));
            const float x = fmaf(d, bx, vw.e[0]);
            const float y = fmaf(d, by, vw.e[1]);
            const float w = fmaf(d, bw, vw.e[2]);
            if (w < 1e-6f) continue;
            const float rcp = __frcp_rn(w);
            const float fxp = floorf(__fmul_rn(x, rcp)), fyp = floorf(__fmul_rn(y, rcp));
            if (!(fxp >= 0.0f) || !(fyp >= 0.0f) || !(fxp < (float)vw.width) || !(fyp < (float)vw.height)) continue;
            const float Mk = __ldg(vw.mask + ((size_t)(int)fyp * vw.width + (int)fxp));
            if (Mk > Mmax) Mmax = Mk;
        }
        const float stat = fmaxf(__fsub_rn(1.0f, Mmax), 0.0f);      // max(1 - M^t, 0)
        const float t = __fmul_rn(__fmul_rn(p.beta, acc), stat);
        wt = t < p.eta ? t : p.eta;                                  // Eq. 13
    }
    p.out[i] = wt;
}

}  // namespace

cudaError_t ggt_launch_temporal_weight(const GgtTemporalParams& p, cudaStream_t st) {
    const dim3 blk(32, 8), grd((p.Wt + 31) / 32, (p.Ht + 7) / 8);
    k_temporal_weight<<<grd, blk, 0, st>>>(p);
    return cudaGetLastError();
}
