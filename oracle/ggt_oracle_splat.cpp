// ggt_oracle_splat.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT (second source file of libggt_oracle.so).
//
// Plain, slow, single-threaded CPU restatement of the paper's forward warping with pixel-sized 3D Gaussians
// (SURVEY.md 8(f) row f-3), written from /root/reference/PAPER.md.  Shares no code with the CUDA path.
//
// Passages followed:
//   PAPER.md:63-65 (3.1)  "for each pixel of an input I_k, we use the depth map D_k and pose to determine the 3D position
//                         of an isotropic, fully-opaque Gaussian.  The RGB color of each Gaussian is set to the underlying
//                         pixel value, and its scale is computed such that its projection in the source image I_k covers a
//                         single pixel.  This step produces a set of forward-rendered images {I_k} along with accumulated
//                         opacity of the Gaussians {alpha_k}, and depths {D_k} in the novel view."
//   PAPER.md:362-368 (A.3) scale, rotation, colour and opacity are computed analytically, one Gaussian per pixel.
//   PAPER.md:141          rendering is "the original 3D Gaussian splatting code [27]": EWA projection of each Gaussian
//                         to a 2D Gaussian, depth-sorted front-to-back alpha compositing per target pixel.
//   PAPER.md:92, 352-354  the difference masks M_k are splatted the same way (one more channel); the novel-view mask
//                         is their channel-wise maximum over the K views (taken by the caller: orc_temporal_weight_mask).
//
// The paper gives no formulas for the rasteriser; it cites [27].  What follows restates the published algorithm of [27]
// (its forward pass for opaque, isotropic Gaussians), with these readings (S1-S8):
//   S1 position   P = R_k^T (D K_k^-1 (u + 0.5, v + 0.5, 1)^T - t_k); in the target camera (x, y, w) = D H (uc, vc, 1)^T + e,
//                 H = K_t R_t R_k^T K_k^-1, e = K_t (t_t - R_t R_k^T t_k)  (PAPER.md:331's projection with the roles of
//                 the two cameras exchanged); centre mu = (x / w, y / w), sort key and depth value z = w.
//   S2 scale      3D standard deviation sigma = sigma_px * D / fx_k: its projection into the SOURCE image has a standard
//                 deviation of sigma_px pixels (default 0.5: one pixel from -1 sigma to +1 sigma).  A parameter.
//   S3 footprint  2D covariance Sigma' = sigma^2 J J^T + dilation I, J the Jacobian of the target's perspective
//                 projection at the centre ([27]'s EWA step; for an isotropic Gaussian the world-to-camera rotation
//                 cancels); dilation = 0.3 px^2 is [27]'s low-pass term.  A parameter.
//   S4 alpha      alpha = min(0.99, exp(q)), q = -1/2 d^T Sigma'^-1 d, d = centre - pixel centre; opacity 1 ("fully
//                 opaque"); a Gaussian contributes to a pixel iff q <= 0 and alpha >= 1/255 ([27]'s thresholds).
//   S5 order      per target pixel, contributing Gaussians are composited front to back in ascending z; equal z in
//                 ascending source pixel index (the order of [27]'s key sort is by depth only; the tie rule makes it total).
//   S6 compositing T = 1; for each: t' = T (1 - alpha); if t' < 1e-4 stop (that Gaussian is not added); C += c alpha T;
//                 T = t'.  Outputs: colour C (source units 0..255, premultiplied, no background), accumulated opacity
//                 1 - T, depth = (sum z alpha T) / (1 - T) (0 where nothing landed), mask = sum M alpha T.
//   S7 culling    Gaussians with D <= 0 or w < z_cull (default 0.2 m, [27]'s near cull) are dropped.
//   S8 exp        exp(q) is evaluated by the fp32 routine orc_exp_le0 below (2^n times a degree-7 polynomial, every
//                 operation stated), so that both implementations take the alpha >= 1/255 and T < 1e-4 decisions on
//                 identical bits (P14); its error against the true exponential is < 3e-7 relative (pinned).
// fp32 arithmetic in exactly the order written (compiled with -ffp-contract=off); fmaf only where written.
//
// Pins (tests/test_oracle_splat_pins.py): T23 orc_exp_le0 against numpy's exp; T24 one Gaussian: footprint, peak and
// 1/255 cut-off radius in closed form (fronto-parallel and off-axis covariance against an fp64 numerical Jacobian); T25
// coincident camera: image, depth and mask are reproduced, opacity saturates; T26 a dense fronto-parallel plane seen from
// a translated camera: opacity > 0.999, depth = plane depth, colour = the shifted image; T27 the nearer surface wins at an
// occlusion edge and the disoccluded strip stays empty; T28 all-pairs brute force in fp64 on a tiny case (no bounding
// boxes, no lists), including equal-depth ties.
// Parity unpinned (choices; parameters of the call): sigma_px (S2), dilation (S3), the thresholds 0.99, 1/255, 1e-4 and
// z_cull (S4, S6, S7 -- [27]'s published constants), the depth normalisation (S6), the tie rule (S5).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {
struct OrcCameraS {
    float fx, fy, cx, cy;
    float R[9];
    float t[3];
    int32_t width, height;
};

// exp(q) for q <= 0 in fp32 (reading S8): t = q log2(e); n = round-to-nearest-even(t) (magic-number addition);
// f = t - n in [-1/2, 1/2]; 2^f by the degree-7 Taylor polynomial of e^(f ln 2) in Horner form; times 2^n exactly.
// q < -80 returns 0 (2^n would be denormal; alpha is far below every threshold there).
inline float orc_exp_le0_impl(float q) {
    if (q < -80.0f) return 0.0f;
    const float t = q * 1.44269504f;
    const float big = 12582912.0f;                 // 1.5 * 2^23
    const float n = (t + big) - big;
    const float f = t - n;
    float p = 1.52527338e-5f;
    p = fmaf(p, f, 1.54035304e-4f);
    p = fmaf(p, f, 1.33335581e-3f);
    p = fmaf(p, f, 9.61812911e-3f);
    p = fmaf(p, f, 5.55041087e-2f);
    p = fmaf(p, f, 2.40226507e-1f);
    p = fmaf(p, f, 6.93147181e-1f);
    p = fmaf(p, f, 1.0f);
    const int32_t e = (int32_t)n + 127;            // n in [-116, 0]
    uint32_t bits = (uint32_t)e << 23;
    float s;
    std::memcpy(&s, &bits, 4);
    return p * s;
}

struct OrcGauss {
    float mx, my, z;       // centre in target pixels, depth key
    float ca, cb, cc;      // conic (inverse 2D covariance): q = -1/2 (ca dx^2 + cc dy^2) - cb dx dy
    float rad;             // conservative radius in pixels
    int32_t ok;
};

inline float orc_alpha(const OrcGauss& g, float pcx, float pcy, bool* contributes) {
    const float dx = g.mx - pcx, dy = g.my - pcy;
    const float t1 = dx * dx, t2 = dy * dy, t3 = dx * dy;
    const float s1 = g.ca * t1, s2 = g.cc * t2;
    const float s3 = s1 + s2;
    const float u = g.cb * t3;
    const float q = (-0.5f * s3) - u;
    if (q > 0.0f) { *contributes = false; return 0.0f; }
    float a = orc_exp_le0_impl(q);
    if (a > 0.99f) a = 0.99f;
    *contributes = a >= (1.0f / 255.0f);
    return a;
}
}  // namespace

extern "C" int orc_relative(const OrcCameraS* tgt, const OrcCameraS* view, float* Hm_out, float* e_out);   // ggt_oracle.cpp

extern "C" float orc_exp_le0(float q) { return orc_exp_le0_impl(q); }

// Per-Gaussian projection (readings S1-S3, S7) of source pixel (u, v) with depth D: exposed for the pins.
//   out[0..6] = mu_x, mu_y, z, conic a, b, c, radius; returns 1 if the Gaussian exists, else 0.
extern "C" int orc_splat_project(const OrcCameraS* tgt, const OrcCameraS* view, int32_t u, int32_t v, float D, float sigma_px,
                                 float dilation, float z_cull, float* out) {
    float Hm[9], ev[3];
    // roles exchanged: from the SOURCE view's pixel / depth into the TARGET camera
    orc_relative(view, tgt, Hm, ev);
    if (!(D > 0.0f)) return 0;
    const float uc = (float)u + 0.5f, vc = (float)v + 0.5f;
    const float bx = fmaf(Hm[0], uc, fmaf(Hm[1], vc, Hm[2]));
    const float by = fmaf(Hm[3], uc, fmaf(Hm[4], vc, Hm[5]));
    const float bw = fmaf(Hm[6], uc, fmaf(Hm[7], vc, Hm[8]));
    const float x = fmaf(D, bx, ev[0]), y = fmaf(D, by, ev[1]), w = fmaf(D, bw, ev[2]);
    if (!(w >= z_cull)) return 0;
    const float rw = 1.0f / w;
    const float mx = x * rw, my = y * rw;
    // camera-space X / z and Y / z of the centre in the target camera
    const float tx = (mx - tgt->cx) / tgt->fx, ty = (my - tgt->cy) / tgt->fy;
    const float sig = sigma_px * D / view->fx;                   // S2
    const float gx = tgt->fx * rw, gy = tgt->fy * rw;            // fx / z, fy / z
    const float s2 = sig * sig;
    // Sigma' = sigma^2 J J^T + dilation I,  J = [gx 0 -gx tx; 0 gy -gy ty]
    const float a = s2 * (gx * gx) * (1.0f + tx * tx) + dilation;
    const float b = s2 * (gx * gy) * (tx * ty);
    const float c = s2 * (gy * gy) * (1.0f + ty * ty) + dilation;
    const float det = a * c - b * b;
    if (!(det > 0.0f)) return 0;
    const float idet = 1.0f / det;
    const float mid = 0.5f * (a + c);
    float disc = mid * mid - det;
    if (disc < 0.0f) disc = 0.0f;
    const float lmax = mid + sqrtf(disc);
    // alpha >= 1/255 needs d^T Sigma'^-1 d <= 2 ln 255 = 11.083, hence |d|^2 <= 11.083 lmax: 3.34 sqrt(lmax) is conservative
    const float rad = 3.34f * sqrtf(lmax);
    out[0] = mx; out[1] = my; out[2] = w;
    out[3] = c * idet; out[4] = -b * idet; out[5] = a * idet;
    out[6] = rad;
    return 1;
}

// --------------------------------------------------------------------------------------------------
// O-S  Forward splat of ONE input view into the target view (readings S1-S8).
//   depth: fp32 H x W z-depth of the source view (<= 0 invalid); rgb: uint8 H x W x stride (optional); mask: fp32 H x W
//   (optional).  Outputs (each optional): out_rgb [3][Ht][Wt], out_alpha, out_depth, out_mask [Ht][Wt], fp32;
//   out_count [Ht][Wt] int32 = number of Gaussians that pass the alpha >= 1/255 test at the pixel (diagnostic).
// --------------------------------------------------------------------------------------------------
extern "C" int orc_splat_forward(const OrcCameraS* tgt, const OrcCameraS* view, const float* depth, const uint8_t* rgb,
                                 int32_t stride, const float* mask, float sigma_px, float dilation, float z_cull,
                                 float* out_rgb, float* out_alpha, float* out_depth, float* out_mask, int32_t* out_count) {
    const int W = view->width, H = view->height, Wt = tgt->width, Ht = tgt->height;
    if (W <= 0 || H <= 0 || Wt <= 0 || Ht <= 0) return -1;
    const int64_t N = (int64_t)W * H, Nt = (int64_t)Wt * Ht;
    std::vector<OrcGauss> gs((size_t)N);
    std::vector<std::vector<int32_t>> lists((size_t)Nt);
    for (int v = 0; v < H; ++v)
        for (int u = 0; u < W; ++u) {
            const int64_t i = (int64_t)v * W + u;
            float o[7];
            OrcGauss& g = gs[(size_t)i];
            g.ok = orc_splat_project(tgt, view, u, v, depth[i], sigma_px, dilation, z_cull, o);
            if (!g.ok) continue;
            g.mx = o[0]; g.my = o[1]; g.z = o[2]; g.ca = o[3]; g.cb = o[4]; g.cc = o[5]; g.rad = o[6];
            // candidate pixels: centres within the conservative radius (the alpha test decides)
            const float x0f = std::floor(g.mx - g.rad - 0.5f), x1f = std::ceil(g.mx + g.rad - 0.5f);
            const float y0f = std::floor(g.my - g.rad - 0.5f), y1f = std::ceil(g.my + g.rad - 0.5f);
            if (!(x1f >= 0.0f) || !(y1f >= 0.0f) || !(x0f <= (float)(Wt - 1)) || !(y0f <= (float)(Ht - 1))) continue;
            const int x0 = (int)std::max(x0f, 0.0f), x1 = (int)std::min(x1f, (float)(Wt - 1));
            const int y0 = (int)std::max(y0f, 0.0f), y1 = (int)std::min(y1f, (float)(Ht - 1));
            for (int py = y0; py <= y1; ++py)
                for (int px = x0; px <= x1; ++px) {
                    bool in;
                    orc_alpha(g, (float)px + 0.5f, (float)py + 0.5f, &in);
                    if (in) lists[(size_t)py * Wt + px].push_back((int32_t)i);
                }
        }
    for (int py = 0; py < Ht; ++py)
        for (int px = 0; px < Wt; ++px) {
            const int64_t p = (int64_t)py * Wt + px;
            std::vector<int32_t>& L = lists[(size_t)p];
            std::sort(L.begin(), L.end(), [&](int32_t a, int32_t b) {              // S5: ascending z, then index
                const float za = gs[(size_t)a].z, zb = gs[(size_t)b].z;
                return za < zb || (za == zb && a < b);
            });
            float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, Dacc = 0.0f, Macc = 0.0f;
            for (int32_t gi : L) {
                const OrcGauss& g = gs[(size_t)gi];
                bool in;
                const float a = orc_alpha(g, (float)px + 0.5f, (float)py + 0.5f, &in);
                if (!in) continue;
                const float tt = T * (1.0f - a);
                if (tt < 1e-4f) break;                                               // S6
                const float wgt = a * T;
                if (rgb) {
                    const uint8_t* c = rgb + (int64_t)gi * stride;
                    C0 = fmaf((float)c[0], wgt, C0); C1 = fmaf((float)c[1], wgt, C1); C2 = fmaf((float)c[2], wgt, C2);
                }
                Dacc = fmaf(g.z, wgt, Dacc);
                if (mask) Macc = fmaf(mask[gi], wgt, Macc);
                T = tt;
            }
            const float acc = 1.0f - T;
            if (out_rgb) { out_rgb[p] = C0; out_rgb[Nt + p] = C1; out_rgb[2 * Nt + p] = C2; }
            if (out_alpha) out_alpha[p] = acc;
            if (out_depth) out_depth[p] = acc > 0.0f ? Dacc / acc : 0.0f;
            if (out_mask) out_mask[p] = Macc;
            if (out_count) out_count[p] = (int32_t)L.size();
        }
    return 0;
}

// --------------------------------------------------------------------------------------------------
// Eq. 13 with the paper's own novel-view mask: omega_tmp = min(beta omega_acc max(1 - M^t, 0), eta)
// per pixel of D^{t-1}, M^t given (the channel-wise maximum of the K splatted masks).  depth <= 0 or omega_acc <= 0 -> 0.
// --------------------------------------------------------------------------------------------------
extern "C" int orc_temporal_weight_mask(int64_t n, const float* prev_depth, const float* prev_conf, const float* novel_mask,
                                        float beta, float eta, float* weight_out) {
    for (int64_t i = 0; i < n; ++i) {
        float wt = 0.0f;
        if (prev_depth[i] > 0.0f && prev_conf[i] > 0.0f) {
            const float stat = fmaxf(1.0f - novel_mask[i], 0.0f);
            const float ba = beta * prev_conf[i];
            const float t = ba * stat;
            wt = t < eta ? t : eta;
        }
        weight_out[i] = wt;
    }
    return 0;
}
