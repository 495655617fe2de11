// ggt_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU restatement of the geometry-guidance hot path of
// arxiv/paper_2505_18932 ("Geometry-guided Online 3D Video Synthesis with Multi-View Temporal
// Consistency"), written from /root/reference/PAPER.md and the readings listed in DESIGN.md.
// It shares no code with the CUDA path (paper_2505_18932_b200/csrc, include/ggt.h): own types, own
// constants, own helpers.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call it.
//
// Build:  g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC -o libggt_oracle.so ggt_oracle.cpp
// Arithmetic is fp32 in exactly the order written below (the paper fixes no precision; its CUDA
// implementation is fp32 by every indication, and the discrete decisions -- pixel index, validity,
// behind-surface cut, zero crossing -- are only comparable if both sides round the same way;
// DESIGN.md reading P14).  `fmaf` is the correctly-rounded fused multiply-add; nothing else is fused.
//
// Passages followed (PAPER.md line : what):
//   79-81  Eq. 1   soft colour-difference mask, beta = 0.6, lambda_t = 0.7, quarter resolution,
//                  3x3 max-pool, bilinear upscale                         -> orc_refine
//   83-84  Eq. 2   temporal depth filter                                   -> orc_refine
//   331    A.1     projection (x,y,z) = K(Rp + t), (u,v) = (x/z, y/z)       -> orc_relative / orc_integrate
//   333    Eq. 9   per-view signed distance (sign: reading P1)              -> orc_integrate
//   339-341 Eq. 10 truncated weighted fusion                                -> orc_integrate
//   343-348 Eq. 11-12 depth-variance weight, w = 7                          -> orc_weight_map
//   348    omega_k = 0 if s_k < -tau; surface = change of sign of s         -> orc_integrate / orc_extract
//   75, 348 the paper's own schedule: on-the-fly TSDF, advance 0.8 s, sign change,
//          three bisection steps (no volume)                                 -> orc_raymarch
//   92-96, 352-360 Eq. 3, 13-14: previous output depth as one more view with a
//          mask-gated, capped accumulated weight                             -> orc_temporal_weight
//   374-388 A.4 items 5-8: ray / normal / view-direction dot products and camera
//          distance maps of the guidance depth (network input features)     -> orc_features
//   356-360 Eq. 13-14 accumulated temporal weight with cap (analogue: P9)   -> orc_integrate (accumulate)
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): T1 analytic planes/spheres, T2 coincident camera,
// T3 view-order invariance, T4 brute-force fp64 per-voxel, T5 Eq. 1 closed forms, T6 Eq. 2 EMA,
// T7 Eq. 11-12 closed forms (0.050518), T8 cut/clamp sweep, T9 running-average closed form, T10 extract,
// T11-T14 raymarch (planes / sphere closed form, dense fp64 first-crossing brute force, coincident camera,
// closed-form evaluation counts), T15-T18 temporal weight (Eq. 13 closed forms, fp64 brute-force mask gather,
// Eq. 14 recursion in closed form, variance reduction), T19-T22 network-input features (plane / sphere normals,
// fp64 ray dot products and constant maps, undefined pixels).
// The forward warp with pixel-sized Gaussians (row f-3) and Eq. 13 from a splatted mask live in ggt_oracle_splat.cpp (the
// second source file of this library; pins T23-T28 in tests/test_oracle_splat_pins.py).
// Parity unpinned (choices, not derivable): the VALUES of tau in C2-C5 (P3), the
// dead-zone threshold semantics (P6), decay/cap without mask gate (P9-P10), the border rule of
// Eq. 12 (P11), the confidence output (P13); in orc_raymarch the min_step / max_evals / unobserved-sample
// rules and the confidence (M2-M4, M6); in orc_temporal_weight the gather that stands in for the paper's
// forward splat of the masks, without an occlusion test (F1); in orc_features the finite-difference stencil
// of the normal (G2).
#include <cmath>
#include <cstdint>
#include <cstring>

namespace {

struct OrcCamera {          // world -> camera: x_cam = R p + t
    float fx, fy, cx, cy;
    float R[9];             // row-major
    float t[3];
    int32_t width, height;
};

// ---- binary16 storage emulation (round-to-nearest-even), written from the IEEE 754 layout ----
inline uint16_t f32_to_f16_bits(float f) {
    uint32_t x;
    std::memcpy(&x, &f, 4);
    const uint32_t sign = (x >> 16) & 0x8000u;
    const uint32_t ax = x & 0x7fffffffu;
    if (ax >= 0x7f800000u) {                       // inf / nan
        return (uint16_t)(sign | 0x7c00u | ((ax > 0x7f800000u) ? 0x200u : 0u));
    }
    if (ax >= 0x477ff000u) {                       // >= 65520 rounds to inf
        return (uint16_t)(sign | 0x7c00u);
    }
    if (ax < 0x33000001u) {                        // <= 2^-25 rounds to zero
        return (uint16_t)sign;
    }
    const int32_t e = (int32_t)(ax >> 23) - 127;   // unbiased exponent
    uint32_t mant = (ax & 0x7fffffu) | 0x800000u;  // 24-bit significand
    int shift;                                     // bits to drop
    uint32_t base;
    if (e >= -14) {                                // normal half
        shift = 13;
        base = (uint32_t)(e + 15) << 10;
        mant &= 0x7fffffu;                         // implicit bit not stored
    } else {                                       // subnormal half: value = mant * 2^(e-23), unit 2^-24
        shift = 13 + (-14 - e);
        base = 0;
    }
    uint32_t q = mant >> shift;
    const uint32_t rem = mant & ((1u << shift) - 1u);
    const uint32_t half = 1u << (shift - 1);
    if (rem > half || (rem == half && (q & 1u))) q++;
    return (uint16_t)(sign | (base + q));          // carry into the exponent is the right answer
}

inline float f16_bits_to_f32(uint16_t h) {
    const uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
    const uint32_t e = (h >> 10) & 0x1fu;
    const uint32_t m = h & 0x3ffu;
    float v;
    if (e == 0) {
        v = std::ldexp((float)m, -24);
    } else if (e == 31) {
        v = m ? NAN : INFINITY;
    } else {
        v = std::ldexp((float)(m | 0x400u), (int)e - 25);
    }
    uint32_t b;
    std::memcpy(&b, &v, 4);
    b |= sign;
    std::memcpy(&v, &b, 4);
    return v;
}

inline float round_f16(float f) { return f16_bits_to_f32(f32_to_f16_bits(f)); }

}  // namespace

extern "C" {

float orc_round_f16(float f) { return round_f16(f); }

// --------------------------------------------------------------------------------------------------
// O-R  Temporal depth refinement of ONE input view (Eq. 1-2).
//   rgb_cur / rgb_prev: uint8, H x W pixels of `stride` bytes (3 or 4), channels 0..2 = RGB.
//   rgb_prev == NULL  -> first frame: M = 1, state = depth_cur.
//   depth_state: in = refined depth of frame t-1, out = refined depth of frame t.
//   mask_out (H x W float, optional), pooled_out (Hq x Wq uint16, optional),
//   binary_out (Hq x Wq uint8, optional: pooled > floor(theta * s*s*255)).
// Readings: P5 (L1 over RGB, colours /255), P6 (dead zone theta in front of Eq. 1), P7 (quarter res
// per axis, box SUM then difference), P8 (window clipped, half-pixel centres, edge clamp), P17.
// --------------------------------------------------------------------------------------------------
int orc_refine(int32_t W, int32_t H, const uint8_t* rgb_cur, const uint8_t* rgb_prev, int32_t stride,
               const float* depth_cur, float* depth_state, float* mask_out, uint16_t* pooled_out,
               uint8_t* binary_out, float lambda_t, float beta, float theta, int32_t s, int32_t pool) {
    if (W <= 0 || H <= 0 || s <= 0 || pool <= 0 || (pool & 1) == 0) return -1;
    const int64_t N = (int64_t)W * H;
    if (!rgb_prev) {
        for (int64_t i = 0; i < N; ++i) {
            depth_state[i] = depth_cur[i];
            if (mask_out) mask_out[i] = 1.0f;
        }
        return 0;
    }
    const int Wq = (W + s - 1) / s, Hq = (H + s - 1) / s;
    int32_t* cq = new int32_t[(size_t)Wq * Hq];
    int32_t* pq = new int32_t[(size_t)Wq * Hq];
    float* Mq = new float[(size_t)Wq * Hq];
    // step 1-2: box sums of each image, L1 over RGB of the difference of the sums
    for (int yq = 0; yq < Hq; ++yq)
        for (int xq = 0; xq < Wq; ++xq) {
            int32_t c = 0;
            for (int ch = 0; ch < 3; ++ch) {
                int32_t sc = 0, sp = 0;
                for (int dy = 0; dy < s; ++dy)
                    for (int dx = 0; dx < s; ++dx) {
                        int y = yq * s + dy; if (y > H - 1) y = H - 1;
                        int x = xq * s + dx; if (x > W - 1) x = W - 1;
                        const int64_t o = ((int64_t)y * W + x) * stride + ch;
                        sc += rgb_cur[o];
                        sp += rgb_prev[o];
                    }
                const int32_t d = sc - sp;
                c += d < 0 ? -d : d;
            }
            cq[yq * Wq + xq] = c;
        }
    // max-pool over the pool x pool window clipped to the image
    const int r = pool / 2;
    for (int yq = 0; yq < Hq; ++yq)
        for (int xq = 0; xq < Wq; ++xq) {
            int32_t m = 0;
            for (int dy = -r; dy <= r; ++dy)
                for (int dx = -r; dx <= r; ++dx) {
                    const int y = yq + dy, x = xq + dx;
                    if (y < 0 || y >= Hq || x < 0 || x >= Wq) continue;
                    const int32_t v = cq[y * Wq + x];
                    if (v > m) m = v;
                }
            pq[yq * Wq + xq] = m;
        }
    // step 3: Eq. 1 on the pooled difference (colours in [0,1]: divide by s*s*255)
    const float norm = (float)(s * s * 255);
    const int32_t thr = (int32_t)std::floor((double)theta * (double)(s * s * 255) + 0.5e-3);
    for (int i = 0; i < Wq * Hq; ++i) {
        const float delta = (float)pq[i] / norm;
        float a = delta - theta;
        if (!(a > 0.0f)) a = 0.0f;
        const float b = a / lambda_t;
        float m = b + beta;
        if (m > 1.0f) m = 1.0f;
        Mq[i] = m;
        if (pooled_out) pooled_out[i] = (uint16_t)pq[i];
        if (binary_out) binary_out[i] = pq[i] > thr ? 1 : 0;
    }
    // step 4-5: bilinear upscale (half-pixel centres, edge clamp), then Eq. 2 with validity handling
    const float inv_s = 1.0f / (float)s;   // exact for s = 4
    for (int y = 0; y < H; ++y) {
        float sy = ((float)y + 0.5f) * inv_s - 0.5f;
        if (sy < 0.0f) sy = 0.0f;
        if (sy > (float)(Hq - 1)) sy = (float)(Hq - 1);
        const int y0 = (int)std::floor(sy);
        const float fy = sy - (float)y0;
        const int y1 = y0 + 1 < Hq ? y0 + 1 : Hq - 1;
        for (int x = 0; x < W; ++x) {
            float sx = ((float)x + 0.5f) * inv_s - 0.5f;
            if (sx < 0.0f) sx = 0.0f;
            if (sx > (float)(Wq - 1)) sx = (float)(Wq - 1);
            const int x0 = (int)std::floor(sx);
            const float fx = sx - (float)x0;
            const int x1 = x0 + 1 < Wq ? x0 + 1 : Wq - 1;
            const float a00 = Mq[y0 * Wq + x0], a01 = Mq[y0 * Wq + x1];
            const float a10 = Mq[y1 * Wq + x0], a11 = Mq[y1 * Wq + x1];
            const float top = fmaf(fx, a01 - a00, a00);
            const float bot = fmaf(fx, a11 - a10, a10);
            const float M = fmaf(fy, bot - top, top);
            const int64_t i = (int64_t)y * W + x;
            const float dc = depth_cur[i], dp = depth_state[i];
            const bool vc = dc > 0.0f, vp = dp > 0.0f;
            const float wc = vc ? M : 0.0f;
            const float wp = vp ? 1.0f - M : 0.0f;
            float out;
            if (wc + wp == 0.0f) out = 0.0f;
            else if (vc && vp) out = fmaf(M, dc - dp, dp);          // == M*D + (1-M)*D_prev, Eq. 2
            else out = vc ? dc : dp;
            depth_state[i] = out;
            if (mask_out) mask_out[i] = M;
        }
    }
    delete[] cq; delete[] pq; delete[] Mq;
    return 0;
}

// --------------------------------------------------------------------------------------------------
// O-W  Depth-variance fusion weight map of one input view (Eq. 11-12).
//   out: interleaved {depth, omega} per pixel (2 floats).  window = 0 -> omega = 1 where depth > 0.
// Readings: P11 (missing neighbours contribute clip^2; nu == 0 -> omega = 1; clip decoupled from tau).
// --------------------------------------------------------------------------------------------------
int orc_weight_map(int32_t W, int32_t H, const float* depth, float* out, float sigma0, float clip,
                   int32_t window) {
    if (W <= 0 || H <= 0 || window < 0 || (window > 0 && (window & 1) == 0)) return -1;
    const int r = window / 2;
    const float c2 = clip * clip;
    const float area = (float)(window * window);
    for (int q0 = 0; q0 < H; ++q0)
        for (int p0 = 0; p0 < W; ++p0) {
            const int64_t i = (int64_t)q0 * W + p0;
            const float D0 = depth[i];
            float omega;
            if (!(D0 > 0.0f)) {
                omega = 0.0f;
            } else if (window == 0) {
                omega = 1.0f;
            } else {
                float nu = 0.0f;
                for (int dq = -r; dq <= r; ++dq)
                    for (int dp = -r; dp <= r; ++dp) {
                        const int q = q0 + dq, p = p0 + dp;
                        float m = c2;
                        if (q >= 0 && q < H && p >= 0 && p < W) {
                            const float Dn = depth[(int64_t)q * W + p];
                            if (Dn > 0.0f) {
                                const float d = D0 - Dn;
                                const float dd = d * d;
                                m = dd < c2 ? dd : c2;
                            }
                        }
                        nu = nu + m;
                    }
                if (nu == 0.0f) {
                    omega = 1.0f;
                } else {
                    const float v = nu / area;
                    const float sd = sqrtf(v);
                    const float w = sigma0 / sd;
                    omega = w < 1.0f ? w : 1.0f;
                }
            }
            out[2 * i] = D0;
            out[2 * i + 1] = omega;
        }
    return 0;
}

// --------------------------------------------------------------------------------------------------
// Bin tables: tau_j = trunc_bins * local spacing (one-sided at the ends), or trunc_metric if > 0.
// Reading P3.  Computed in double, rounded to float.
// --------------------------------------------------------------------------------------------------
int orc_tau_table(int32_t D, const float* z, float trunc_bins, float trunc_metric, float* tau) {
    if (D < 2) return -1;
    for (int j = 0; j < D; ++j) {
        double sp;
        if (j == 0) sp = (double)z[1] - (double)z[0];
        else if (j == D - 1) sp = (double)z[D - 1] - (double)z[D - 2];
        else sp = ((double)z[j + 1] - (double)z[j - 1]) / 2.0;
        tau[j] = trunc_metric > 0.0f ? trunc_metric : (float)((double)trunc_bins * sp);
    }
    return 0;
}

// --------------------------------------------------------------------------------------------------
// Relative transform target pixel/depth -> view k homogeneous pixel:
//   p_world = R_t^T (z K_t^{-1} (uc, vc, 1)^T - t_t),  (x,y,w) = K_k (R_k p_world + t_k)
//   => (x,y,w) = z * Hm (uc,vc,1)^T + e,  Hm = K_k R_k R_t^T K_t^{-1},  e = K_k (t_k - R_k R_t^T t_t).
// Double arithmetic, plain left-to-right triple products, rounded to float at the end.
// --------------------------------------------------------------------------------------------------
int orc_relative(const OrcCamera* tgt, const OrcCamera* view, float* Hm_out, float* e_out) {
    double Rk[9], Rt[9], M1[9], M2[9], Hm[9], Kk[9], Kti[9];
    for (int i = 0; i < 9; ++i) { Rk[i] = view->R[i]; Rt[i] = tgt->R[i]; }
    // M1 = R_k * R_t^T
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            M1[3 * i + j] = Rk[3 * i + 0] * Rt[3 * j + 0] + Rk[3 * i + 1] * Rt[3 * j + 1] + Rk[3 * i + 2] * Rt[3 * j + 2];
    const double kk[9] = {(double)view->fx, 0.0, (double)view->cx, 0.0, (double)view->fy, (double)view->cy, 0.0, 0.0, 1.0};
    for (int i = 0; i < 9; ++i) Kk[i] = kk[i];
    const double fxt = tgt->fx, fyt = tgt->fy, cxt = tgt->cx, cyt = tgt->cy;
    const double kti[9] = {1.0 / fxt, 0.0, -cxt / fxt, 0.0, 1.0 / fyt, -cyt / fyt, 0.0, 0.0, 1.0};
    for (int i = 0; i < 9; ++i) Kti[i] = kti[i];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            M2[3 * i + j] = Kk[3 * i + 0] * M1[0 + j] + Kk[3 * i + 1] * M1[3 + j] + Kk[3 * i + 2] * M1[6 + j];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            Hm[3 * i + j] = M2[3 * i + 0] * Kti[0 + j] + M2[3 * i + 1] * Kti[3 + j] + M2[3 * i + 2] * Kti[6 + j];
    double d[3], e[3];
    const double tt[3] = {(double)tgt->t[0], (double)tgt->t[1], (double)tgt->t[2]};
    for (int i = 0; i < 3; ++i)
        d[i] = (double)view->t[i] - (M1[3 * i + 0] * tt[0] + M1[3 * i + 1] * tt[1] + M1[3 * i + 2] * tt[2]);
    for (int i = 0; i < 3; ++i)
        e[i] = Kk[3 * i + 0] * d[0] + Kk[3 * i + 1] * d[1] + Kk[3 * i + 2] * d[2];
    for (int i = 0; i < 9; ++i) Hm_out[i] = (float)Hm[i];
    for (int i = 0; i < 3; ++i) e_out[i] = (float)e[i];
    return 0;
}

// --------------------------------------------------------------------------------------------------
// O-I  Integrate (Eq. 9-10; accumulate mode: analogue of Eq. 13-14, reading P9).
//   rays: n_rays linear target-pixel indices (v*W_t + u), or NULL = all W_t*H_t pixels in order.
//   T, Wt: [n_rays][D] float, bin-fastest.  accumulate != 0: T/Wt hold the previous frame's values.
//   maps[k]: interleaved {depth, omega} of view k (orc_weight_map output).
//   half_storage != 0: results are rounded to binary16 (RNE) on store, as an fp16 volume would.
// --------------------------------------------------------------------------------------------------
int orc_integrate(const OrcCamera* tgt, int32_t D, const float* z, const float* tau, int32_t n_views,
                  const OrcCamera* views, const float* const* maps, int64_t n_rays, const int32_t* rays,
                  float* T, float* Wt, int32_t accumulate, float decay, float cap, int32_t half_storage) {
    if (D < 2 || n_views < 0) return -1;
    const int32_t Wd = tgt->width, Hd = tgt->height;
    if (!rays) n_rays = (int64_t)Wd * Hd;
    float (*Hm)[9] = new float[n_views > 0 ? n_views : 1][9];
    float (*ev)[3] = new float[n_views > 0 ? n_views : 1][3];
    for (int k = 0; k < n_views; ++k) orc_relative(tgt, &views[k], Hm[k], ev[k]);
    float (*b)[3] = new float[n_views > 0 ? n_views : 1][3];
    for (int64_t r = 0; r < n_rays; ++r) {
        const int32_t pix = rays ? rays[r] : (int32_t)r;
        const int32_t u = pix % Wd, v = pix / Wd;
        const float uc = (float)u + 0.5f, vc = (float)v + 0.5f;
        for (int k = 0; k < n_views; ++k)
            for (int a = 0; a < 3; ++a)
                b[k][a] = fmaf(Hm[k][3 * a + 0], uc, fmaf(Hm[k][3 * a + 1], vc, Hm[k][3 * a + 2]));
        for (int j = 0; j < D; ++j) {
            const float zj = z[j], tj = tau[j];
            float A = 0.0f, Wn = 0.0f;
            for (int k = 0; k < n_views; ++k) {
                const float x = fmaf(zj, b[k][0], ev[k][0]);
                const float y = fmaf(zj, b[k][1], ev[k][1]);
                const float w = fmaf(zj, b[k][2], ev[k][2]);      // z_k of Eq. 9
                if (w < 1e-6f) continue;
                const float rcp = 1.0f / w;
                const float px = x * rcp, py = y * rcp;
                const float fxp = std::floor(px), fyp = std::floor(py);
                if (!(fxp >= 0.0f) || !(fyp >= 0.0f) || !(fxp < (float)views[k].width) ||
                    !(fyp < (float)views[k].height)) continue;
                const int ix = (int)fxp, iy = (int)fyp;
                const float* m = maps[k] + 2 * ((int64_t)iy * views[k].width + ix);
                const float Dk = m[0], om = m[1];
                if (!(Dk > 0.0f)) continue;
                const float s = Dk - w;                              // reading P1
                if (s < -tj) continue;                               // omega_k = 0 if s_k < -tau
                const float c = s < tj ? s : tj;                     // clamp(s_k, -tau, tau)
                A = fmaf(om, c, A);
                Wn = Wn + om;
            }
            float* Tp = T + r * D + j;
            float* Wp = Wt + r * D + j;
            float To, Wo;
            if (!accumulate) {
                if (Wn > 0.0f) { To = A / Wn; Wo = Wn; } else { To = 0.0f; Wo = 0.0f; }
            } else {
                const float Wprev = decay * (*Wp);
                const float Wsum = Wprev + Wn;
                if (Wsum > 0.0f) To = fmaf(Wprev, *Tp, A) / Wsum; else To = 0.0f;
                Wo = Wsum < cap ? Wsum : cap;
            }
            if (half_storage) { To = round_f16(To); Wo = round_f16(Wo); }
            *Tp = To;
            *Wp = Wo;
        }
    }
    delete[] Hm; delete[] ev; delete[] b;
    return 0;
}

// --------------------------------------------------------------------------------------------------
// O-E  Extract ("change of sign in the value of s"; reading P13).
//   T, Wt: [n_rays][D]; outputs per ray: depth (0 = none), conf (0 = none), bin (-1 = none).
// --------------------------------------------------------------------------------------------------
int orc_extract(int64_t n_rays, int32_t D, const float* z, const float* T, const float* Wt,
                float* depth, float* conf, int32_t* bin) {
    for (int64_t r = 0; r < n_rays; ++r) {
        const float* Tr = T + r * D;
        const float* Wr = Wt + r * D;
        float d = 0.0f, c = 0.0f;
        int32_t jb = -1;
        for (int j = 0; j + 1 < D; ++j) {
            if (Wr[j] > 0.0f && Wr[j + 1] > 0.0f && Tr[j] > 0.0f && !(Tr[j + 1] > 0.0f)) {
                const float f = Tr[j] / (Tr[j] - Tr[j + 1]);
                d = fmaf(f, z[j + 1] - z[j], z[j]);
                c = fmaf(f, Wr[j + 1] - Wr[j], Wr[j]);
                jb = j;
                break;
            }
        }
        if (depth) depth[r] = d;
        if (conf) conf[r] = c;
        if (bin) bin[r] = jb;
    }
    return 0;
}

}  // extern "C"

// --------------------------------------------------------------------------------------------------
// O-M  The paper's own schedule: image-based TSDF evaluated on the fly along each
// target ray, no volume ("integrates depth along each ray on the fly and, thus, avoids creating
// an explicit 3D voxel grid"; "We advance along the ray with a step size of 0.8s until a surface
// intersection is detected. This is indicated by a change of sign in the value of s. We subsequently perform
// three steps of a bisection search to refine the intersection depth.").
//
// s(z) at target depth z: the per-sample arithmetic of O-I steps 1-4 with tau_j = tau (PAPER.md:341,
// tau = 0.02 m), normalised as in reading P2: s = sum(omega_k c_k) / sum(omega_k); "unobserved" if the sum of
// weights is 0.  Readings for what the paper leaves open (M1-M6):
//   M1 start at z = z_near, a ray is a miss once z > z_far or after max_evals evaluations of s;
//   M2 advance by max(step_scale * s, min_step) after a positive sample (step_scale = 0.8; min_step > 0
//      guarantees progress, since 0.8 s alone converges to the surface without ever crossing it);
//   M3 an unobserved sample advances like free space, by max(step_scale * tau, min_step);
//   M4 a crossing is a sample with s <= 0 whose PREVIOUS sample was observed and positive (no crossing
//      across an unobserved sample, as P13); a non-positive sample without such a predecessor advances by
//      min_step;
//   M5 bisection: n_bisect times m = 0.5 (a + b); s(m) > 0 -> a = m; s(m) <= 0 -> b = m; an unobserved
//      midpoint ends the refinement; depth = 0.5 (a + b);
//   M6 confidence = sum of weights at the last non-positive sample b; steps = evaluations of s.
// outputs per ray: depth (0 = miss), conf (0 = miss), steps.
// --------------------------------------------------------------------------------------------------
namespace {
struct OrcRayEval {
    int n_views;
    const OrcCamera* views;
    const float* const* maps;
    const float (*b)[3];
    const float (*ev)[3];
    float tau;
};

// one evaluation of Eq. 9-10 at target depth z: returns A = sum(omega c), Wn = sum(omega)
inline void orc_eval_s(const OrcRayEval& E, float z, float* A_out, float* W_out) {
    float A = 0.0f, Wn = 0.0f;
    for (int k = 0; k < E.n_views; ++k) {
        const float x = fmaf(z, E.b[k][0], E.ev[k][0]);
        const float y = fmaf(z, E.b[k][1], E.ev[k][1]);
        const float w = fmaf(z, E.b[k][2], E.ev[k][2]);          // z_k of Eq. 9
        if (w < 1e-6f) continue;
        const float rcp = 1.0f / w;
        const float px = x * rcp, py = y * rcp;
        const float fxp = std::floor(px), fyp = std::floor(py);
        if (!(fxp >= 0.0f) || !(fyp >= 0.0f) || !(fxp < (float)E.views[k].width) ||
            !(fyp < (float)E.views[k].height)) continue;
        const int ix = (int)fxp, iy = (int)fyp;
        const float* m = E.maps[k] + 2 * ((int64_t)iy * E.views[k].width + ix);
        const float Dk = m[0], om = m[1];
        if (!(Dk > 0.0f)) continue;
        const float s = Dk - w;                                  // reading P1
        if (s < -E.tau) continue;                                // omega_k = 0 if s_k < -tau
        const float c = s < E.tau ? s : E.tau;                   // clamp(s_k, -tau, tau)
        A = fmaf(om, c, A);
        Wn = Wn + om;
    }
    *A_out = A;
    *W_out = Wn;
}
}  // namespace

extern "C" int orc_raymarch(const OrcCamera* tgt, int32_t n_views, const OrcCamera* views,
                            const float* const* maps, int64_t n_rays, const int32_t* rays, float z_near,
                            float z_far, float tau, float step_scale, float min_step, int32_t max_evals,
                            int32_t n_bisect, float* depth, float* conf, int32_t* steps) {
    if (n_views < 0 || !(z_far > z_near) || !(tau > 0.0f) || !(min_step > 0.0f) || max_evals < 1 || n_bisect < 0)
        return -1;
    const int32_t Wd = tgt->width, Hd = tgt->height;
    if (!rays) n_rays = (int64_t)Wd * Hd;
    const int nv = n_views > 0 ? n_views : 1;
    float (*Hm)[9] = new float[nv][9];
    float (*ev)[3] = new float[nv][3];
    float (*b)[3] = new float[nv][3];
    for (int k = 0; k < n_views; ++k) orc_relative(tgt, &views[k], Hm[k], ev[k]);
    const float free_step = fmaxf(step_scale * tau, min_step);   // M3
    for (int64_t r = 0; r < n_rays; ++r) {
        const int32_t pix = rays ? rays[r] : (int32_t)r;
        const int32_t u = pix % Wd, v = pix / Wd;
        const float uc = (float)u + 0.5f, vc = (float)v + 0.5f;
        for (int k = 0; k < n_views; ++k)
            for (int a = 0; a < 3; ++a)
                b[k][a] = fmaf(Hm[k][3 * a + 0], uc, fmaf(Hm[k][3 * a + 1], vc, Hm[k][3 * a + 2]));
        const OrcRayEval E = {n_views, views, maps, b, ev, tau};
        float z = z_near, za = 0.0f, zb = 0.0f, Wb = 0.0f;
        bool prev_pos = false, hit = false;
        int32_t n = 0;
        while (n < max_evals && !(z > z_far)) {                   // M1
            float A, Wn;
            orc_eval_s(E, z, &A, &Wn);
            ++n;
            float step;
            if (Wn > 0.0f) {
                const float s = A / Wn;
                if (s > 0.0f) {
                    za = z; prev_pos = true;
                    step = fmaxf(step_scale * s, min_step);       // M2
                } else {
                    if (prev_pos) { zb = z; Wb = Wn; hit = true; break; }   // M4: change of sign
                    step = min_step;
                }
            } else {
                prev_pos = false;
                step = free_step;                                 // M3
            }
            z = z + step;
        }
        float d = 0.0f, c = 0.0f;
        if (hit) {
            for (int i = 0; i < n_bisect; ++i) {                  // M5
                const float m = 0.5f * (za + zb);
                float A, Wn;
                orc_eval_s(E, m, &A, &Wn);
                ++n;
                if (!(Wn > 0.0f)) break;
                const float s = A / Wn;
                if (s > 0.0f) za = m; else { zb = m; Wb = Wn; }
            }
            d = 0.5f * (za + zb);
            c = Wb;                                               // M6
        }
        if (depth) depth[r] = d;
        if (conf) conf[r] = c;
        if (steps) steps[r] = n;
    }
    delete[] Hm; delete[] ev; delete[] b;
    return 0;
}

// --------------------------------------------------------------------------------------------------
// O-T  Temporal fusion weight of the previous output depth (Eq. 3,
// PAPER.md:352-360 Eq. 13-14).  The rendered depth of the previous frame, D^{t-1}, enters the TSDF of frame t
// as one more depth view with its own pose (the previous target camera) and the per-pixel weight
//   omega_tmp^t = min(beta * omega_acc^t * max(1 - M^t, 0), eta)            (Eq. 13, eta = 15)
//   omega_acc^t = omega_tmp^{t-1} + sum_k omega_k^{t-1}                      (Eq. 14)
// omega_acc is the sum of ALL fusion weights at the previous frame's surface point, i.e. the confidence the
// raymarch / extract of frame t-1 returned (readings M6 / P13) when D^{t-2} took part in that frame's sum.
// M^t, the difference mask in the novel view: the paper forward-splats the K input masks M_k^t (Eq. 1) into the
// novel view and takes the maximum; reading F1 restates that as a gather: the surface point of pixel (u, v) of
// D^{t-1} is projected into every input view (A.1's projection, nearest pixel as P4) and M^t is the maximum of
// M_k^t over the views it lands in (0 if none; occlusion is not tested).  Invalid depth or omega_acc <= 0 -> 0.
//   prev: camera of D^{t-1};  masks[k]: fp32 height_k x width_k mask of view k (orc_refine's M).
// --------------------------------------------------------------------------------------------------
extern "C" int orc_temporal_weight(const OrcCamera* prev, const float* prev_depth, const float* prev_conf,
                                   int32_t n_views, const OrcCamera* views, const float* const* masks,
                                   float beta, float eta, float* weight_out) {
    if (n_views < 0) return -1;
    const int32_t Wd = prev->width, Hd = prev->height;
    const int nv = n_views > 0 ? n_views : 1;
    float (*Hm)[9] = new float[nv][9];
    float (*ev)[3] = new float[nv][3];
    for (int k = 0; k < n_views; ++k) orc_relative(prev, &views[k], Hm[k], ev[k]);
    for (int32_t v = 0; v < Hd; ++v)
        for (int32_t u = 0; u < Wd; ++u) {
            const int64_t i = (int64_t)v * Wd + u;
            const float d = prev_depth[i], acc = prev_conf[i];
            float wt = 0.0f;
            if (d > 0.0f && acc > 0.0f) {
                const float uc = (float)u + 0.5f, vc = (float)v + 0.5f;
                float Mmax = 0.0f;
                for (int k = 0; k < n_views; ++k) {
                    const float bx = fmaf(Hm[k][0], uc, fmaf(Hm[k][1], vc, Hm[k][2]));
                    const float by = fmaf(Hm[k][3], uc, fmaf(Hm[k][4], vc, Hm[k][5]));
                    const float bw = fmaf(Hm[k][6], uc, fmaf(Hm[k][7], vc, Hm[k][8]));
                    const float x = fmaf(d, bx, ev[k][0]);
                    const float y = fmaf(d, by, ev[k][1]);
                    const float w = fmaf(d, bw, ev[k][2]);
                    if (w < 1e-6f) continue;
                    const float rcp = 1.0f / w;
                    const float px = x * rcp, py = y * rcp;
                    const float fxp = std::floor(px), fyp = std::floor(py);
                    if (!(fxp >= 0.0f) || !(fyp >= 0.0f) || !(fxp < (float)views[k].width) ||
                        !(fyp < (float)views[k].height)) continue;
                    const float Mk = masks[k][(int64_t)(int)fyp * views[k].width + (int)fxp];
                    if (Mk > Mmax) Mmax = Mk;
                }
                const float stat = fmaxf(1.0f - Mmax, 0.0f);         // max(1 - M^t, 0)
                const float ba = beta * acc;
                const float t = ba * stat;
                wt = t < eta ? t : eta;                               // Eq. 13
            }
            weight_out[i] = wt;
        }
    delete[] Hm; delete[] ev;
    return 0;
}

// --------------------------------------------------------------------------------------------------
// O-F  Geometry features of the guidance depth for the blending network's input (
// PAPER.md:374-388, items 5-8 of A.4: "the dot product between each input-view ray direction, and the normals from
// the TSDF depth D^t", "the dot product between each input-view ray direction, and the target view direction",
// "the distance between the input and target cameras, repeated spatially", "the dot product between the input and
// target viewing directions, repeated spatially").  The paper gives no formulas; readings G1-G4:
//   G1 the surface point of target pixel (u, v): p = D (( uc - cx)/fx, (vc - cy)/fy, 1) in the target camera,
//      P = R_t^T (p - t_t) in the world;
//   G2 normal: n_c = +-(dx x dy), dx = p(u+1, v) - p(u-1, v) where both neighbours have depth, else the one-sided
//      difference with the neighbour that has, else undefined (same in v); oriented towards the camera (n_c . p <= 0),
//      normalised; n = R_t^T n_c.  Undefined (or zero cross product) -> both per-pixel features are 0;
//   G3 "input-view ray direction" at the pixel = unit vector from the input camera centre C_k = -R_k^T t_k to P;
//      "target view direction" at the pixel = unit vector from C_t to P;
//   G4 "viewing directions" = the cameras' optical axes (third rows of R); distance = |C_k - C_t|.
// out: [4 K][H][W] fp32, planar: channels [0, K) item 5, [K, 2K) item 6, [2K, 3K) item 7, [3K, 4K) item 8.
// --------------------------------------------------------------------------------------------------
namespace {
inline void orc_cam_point(const OrcCamera* c, const float* depth, int u, int v, float* p) {
    const float d = depth[(int64_t)v * c->width + u];
    const float uc = (float)u + 0.5f, vc = (float)v + 0.5f;
    p[0] = d * ((uc - c->cx) / c->fx);
    p[1] = d * ((vc - c->cy) / c->fy);
    p[2] = d;
}
inline bool orc_has(const OrcCamera* c, const float* depth, int u, int v) {
    return u >= 0 && v >= 0 && u < c->width && v < c->height && depth[(int64_t)v * c->width + u] > 0.0f;
}
// difference along one axis (du, dv): central, else one-sided, else false
inline bool orc_diff(const OrcCamera* c, const float* depth, int u, int v, int du, int dv, float* out) {
    const bool hp = orc_has(c, depth, u + du, v + dv), hm = orc_has(c, depth, u - du, v - dv);
    float a[3], b[3];
    if (hp && hm) { orc_cam_point(c, depth, u + du, v + dv, a); orc_cam_point(c, depth, u - du, v - dv, b); }
    else if (hp) { orc_cam_point(c, depth, u + du, v + dv, a); orc_cam_point(c, depth, u, v, b); }
    else if (hm) { orc_cam_point(c, depth, u, v, a); orc_cam_point(c, depth, u - du, v - dv, b); }
    else return false;
    for (int i = 0; i < 3; ++i) out[i] = a[i] - b[i];
    return true;
}
inline float orc_dot(const float* a, const float* b) { return fmaf(a[2], b[2], fmaf(a[1], b[1], a[0] * b[0])); }
// w = R^T q  (R row-major): w_i = R[0][i] q0 + R[1][i] q1 + R[2][i] q2
inline void orc_rt_mul(const float* R, const float* q, float* w) {
    for (int i = 0; i < 3; ++i) w[i] = fmaf(R[6 + i], q[2], fmaf(R[3 + i], q[1], R[i] * q[0]));
}
inline void orc_centre(const OrcCamera* c, float* C) {     // C = -R^T t, in double, rounded once
    for (int i = 0; i < 3; ++i)
        C[i] = (float)(-((double)c->R[i] * c->t[0] + (double)c->R[3 + i] * c->t[1] + (double)c->R[6 + i] * c->t[2]));
}
}  // namespace

extern "C" int orc_features(const OrcCamera* tgt, const float* depth, int32_t n_views, const OrcCamera* views, float* out) {
    if (n_views < 0) return -1;
    const int32_t W = tgt->width, H = tgt->height;
    const int64_t plane = (int64_t)W * H;
    float Ct[3];
    orc_centre(tgt, Ct);
    float (*Ck)[3] = new float[n_views > 0 ? n_views : 1][3];
    for (int k = 0; k < n_views; ++k) {
        orc_centre(&views[k], Ck[k]);
        const double dx = (double)Ck[k][0] - Ct[0], dy = (double)Ck[k][1] - Ct[1], dz = (double)Ck[k][2] - Ct[2];
        const float dist = (float)std::sqrt(dx * dx + dy * dy + dz * dz);                              // item 7
        const float axes = (float)((double)views[k].R[6] * tgt->R[6] + (double)views[k].R[7] * tgt->R[7] +
                                   (double)views[k].R[8] * tgt->R[8]);                                 // item 8
        for (int64_t i = 0; i < plane; ++i) {
            out[(2 * n_views + k) * plane + i] = dist;
            out[(3 * n_views + k) * plane + i] = axes;
        }
    }
    for (int v = 0; v < H; ++v)
        for (int u = 0; u < W; ++u) {
            const int64_t i = (int64_t)v * W + u;
            float n[3] = {0.0f, 0.0f, 0.0f}, P[3] = {0.0f, 0.0f, 0.0f};
            bool ok = orc_has(tgt, depth, u, v);
            if (ok) {
                float p[3], dx[3], dy[3];
                orc_cam_point(tgt, depth, u, v, p);
                ok = orc_diff(tgt, depth, u, v, 1, 0, dx) && orc_diff(tgt, depth, u, v, 0, 1, dy);
                if (ok) {
                    float c[3] = {dx[1] * dy[2] - dx[2] * dy[1], dx[2] * dy[0] - dx[0] * dy[2], dx[0] * dy[1] - dx[1] * dy[0]};
                    if (orc_dot(c, p) > 0.0f) { c[0] = -c[0]; c[1] = -c[1]; c[2] = -c[2]; }            // towards the camera
                    const float l2 = orc_dot(c, c);
                    ok = l2 > 0.0f;
                    if (ok) {
                        const float l = sqrtf(l2);
                        const float nc[3] = {c[0] / l, c[1] / l, c[2] / l};
                        orc_rt_mul(tgt->R, nc, n);
                        const float q[3] = {p[0] - tgt->t[0], p[1] - tgt->t[1], p[2] - tgt->t[2]};
                        orc_rt_mul(tgt->R, q, P);
                    }
                }
            }
            float rt[3] = {0.0f, 0.0f, 0.0f};
            if (ok) {
                const float d[3] = {P[0] - Ct[0], P[1] - Ct[1], P[2] - Ct[2]};
                const float l = sqrtf(orc_dot(d, d));
                ok = l > 0.0f;
                if (ok) { rt[0] = d[0] / l; rt[1] = d[1] / l; rt[2] = d[2] / l; }
            }
            for (int k = 0; k < n_views; ++k) {
                float f5 = 0.0f, f6 = 0.0f;
                if (ok) {
                    const float d[3] = {P[0] - Ck[k][0], P[1] - Ck[k][1], P[2] - Ck[k][2]};
                    const float l = sqrtf(orc_dot(d, d));
                    if (l > 0.0f) {
                        const float rk[3] = {d[0] / l, d[1] / l, d[2] / l};
                        f5 = orc_dot(rk, n);                                                            // item 5
                        f6 = orc_dot(rk, rt);                                                           // item 6
                    }
                }
                out[k * plane + i] = f5;
                out[(n_views + k) * plane + i] = f6;
            }
        }
    delete[] Ck;
    return 0;
}
