"""Pins of the forward-splat oracle (oracle/ggt_oracle_splat.cpp).

CPU only.  Expected values are closed forms of one Gaussian, invariants of dense pixel-sized Gaussians (coincident and
translated cameras, occlusion), and an all-pairs fp64 brute force written out below from explicit world geometry
(no bounding boxes, no lists, numpy's exp), T23-T28.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth


def cam(centre=(0, 0, 0), R=None, f=100.0, W=40, H=30, cx=None, cy=None):
    R = np.eye(3) if R is None else R
    return synth.camera_from_pose(centre, R, f, f, W / 2 if cx is None else cx, H / 2 if cy is None else cy, W, H)


# ---- T23: the fp32 exponential of reading S8 -------------------------------------------------------------------------
def test_T23_exp_le0_against_numpy():
    rng = np.random.default_rng(0)
    qs = -np.concatenate([rng.uniform(0, 12, 20000), np.linspace(0, 6, 4001), [5.5412636, 5.541263, 5.541265]]).astype(np.float32)
    got = np.array([oracle.exp_le0(float(q)) for q in qs], dtype=np.float64)
    ref = np.exp(qs.astype(np.float64))
    assert np.max(np.abs(got - ref) / ref) < 1e-6
    assert oracle.exp_le0(0.0) == 1.0 and oracle.exp_le0(-100.0) == 0.0
    # monotone on a fine grid around the 1/255 threshold (q = -ln 255 = -5.5413): the cut-off is a single crossing
    grid = np.float32(-5.5413) + np.arange(-2000, 2001, dtype=np.float32) * np.float32(1e-6)
    vals = np.array([oracle.exp_le0(float(q)) for q in grid])
    assert np.all(np.diff(vals) >= 0)


def test_T23_alpha_threshold_is_a_single_crossing_in_q():
    """alpha >= 1/255 (reading S4) as a threshold on q: with the fp32 exponential of S8 the decision is exactly
    q >= q* = -5.541263580322266 (0xC0B15208).  Checked on EVERY float of [-5.56, -5.52]; outside, exp(q) is more than
    2 % away from 1/255 and the exponential is good to 1e-6.  (The CUDA scatter passes use this form.)"""
    qstar = np.float32(-5.541263580322266)
    assert qstar.view(np.uint32) == 0xC0B15208
    thr = np.float32(1.0) / np.float32(255.0)
    bits = np.arange(int(np.float32(-5.52).view(np.uint32)), int(np.float32(-5.56).view(np.uint32)) + 1, dtype=np.uint32)
    qs = bits.view(np.float32)
    ge = np.array([np.float32(oracle.exp_le0(float(q))) >= thr for q in qs])
    assert np.array_equal(ge, qs >= qstar) and ge.any() and not ge.all()
    assert math.exp(-5.52) > 1.02 / 255 and math.exp(-5.56) < 0.99 / 255


# ---- T24: one Gaussian in closed form ------------------------------------------------------------------------------------
def test_T24_single_gaussian_footprint_and_peak():
    c = cam()
    u, v, D = 20, 15, 2.0                      # the pixel whose centre is the principal point (cx = 20, cy = 15) ... + 0.5
    c = cam(cx=20.5, cy=15.5)
    g = oracle.splat_project(c, c, u, v, D)
    assert g is not None
    assert abs(g[0] - 20.5) < 1e-5 and abs(g[1] - 15.5) < 1e-5 and abs(g[2] - D) < 1e-6
    # sigma' ^2 = sigma_px^2 + dilation = 0.25 + 0.3 on the axis: conic = 1 / 0.55, no cross term
    assert abs(g[3] - 1 / 0.55) < 1e-5 and abs(g[5] - 1 / 0.55) < 1e-5 and abs(g[4]) < 1e-6
    depth = np.zeros((30, 40), np.float32); depth[v, u] = D
    rgb = np.zeros((30, 40, 3), np.uint8); rgb[v, u] = (200, 100, 50)
    r = oracle.splat_forward(c, c, depth, rgb=rgb, mask=np.full((30, 40), 0.75, np.float32))
    a = r["alpha"]
    assert a[v, u] == np.float32(0.99)                                  # fully opaque, clipped at 0.99 ([27])
    for (dx, dy) in [(1, 0), (0, 1), (1, 1), (2, 0), (2, 1), (-1, -2)]:
        e = math.exp(-(dx * dx + dy * dy) / (2 * 0.55))
        assert abs(a[v + dy, u + dx] - e) < 2e-6 * max(e, 0.01), (dx, dy)
    # alpha >= 1/255 <=> d^2 <= 2 * 0.55 * ln 255 = 6.0955: the 21 integer offsets with dx^2 + dy^2 <= 6
    assert (a > 0).sum() == 21 and a[v + 2, u + 2] == 0 and r["count"].sum() == 21
    assert np.allclose(r["rgb"][:, v, u], np.array([200, 100, 50]) * 0.99, rtol=1e-6)
    assert abs(r["depth"][v, u] - D) < 1e-6 and abs(r["depth"][v, u + 2] - D) < 1e-6      # normalised by opacity (S6)
    assert abs(r["mask"][v, u] - 0.75 * 0.99) < 1e-6
    # scale (S2): seen from twice as close, the footprint's standard deviation doubles (dilation off)
    near = cam(centre=(0, 0, 1.0), cx=20.5, cy=15.5)
    g0 = oracle.splat_project(c, c, u, v, D, dilation=0.0)
    g1 = oracle.splat_project(near, c, u, v, D, dilation=0.0)
    assert abs(1 / g0[3] - 0.25) < 1e-6 and abs(1 / g1[3] - 1.0) < 1e-5 and abs(g1[2] - 1.0) < 1e-6
    # culling (S7): invalid depth, and a centre nearer than z_cull
    assert oracle.splat_project(c, c, u, v, 0.0) is None
    assert oracle.splat_project(cam(centre=(0, 0, 1.9)), c, u, v, D) is None          # w = 0.1 < 0.2


def test_T24_off_axis_covariance_against_numerical_jacobian():
    src = cam(centre=(0.3, -0.1, 0.0), R=synth.rot_yaw_pitch(0.1, -0.05), f=120.0, W=64, H=48)
    tgt = cam(centre=(-0.2, 0.15, 0.4), R=synth.rot_yaw_pitch(-0.2, 0.12), f=90.0, W=80, H=60)
    for (u, v, D) in [(5, 40, 1.7), (60, 3, 3.2), (31, 23, 0.9)]:
        g = oracle.splat_project(tgt, src, u, v, D)
        assert g is not None
        Ks = np.array([[src.fx, 0, src.cx], [0, src.fy, src.cy], [0, 0, 1.0]])
        P = src.R.astype(np.float64).T @ (D * np.linalg.inv(Ks) @ np.array([u + 0.5, v + 0.5, 1.0]) - src.t.astype(np.float64))

        def proj(Pw):
            q = tgt.R.astype(np.float64) @ Pw + tgt.t.astype(np.float64)
            return np.array([tgt.fx * q[0] / q[2] + tgt.cx, tgt.fy * q[1] / q[2] + tgt.cy]), q[2]
        mu, z = proj(P)
        assert np.allclose(g[:2], mu, atol=2e-4) and abs(g[2] - z) < 2e-6 * z
        sig = 0.5 * D / src.fx
        h = 1e-6
        J = np.stack([(proj(P + h * e)[0] - proj(P - h * e)[0]) / (2 * h) for e in np.eye(3)], axis=1)      # 2 x 3
        S = sig * sig * (J @ J.T) + 0.3 * np.eye(2)
        conic = np.linalg.inv(S)
        assert np.allclose([g[3], g[4], g[5]], [conic[0, 0], conic[0, 1], conic[1, 1]], rtol=2e-4, atol=1e-6)
        lmax = np.linalg.eigvalsh(S)[-1]
        assert g[6] >= math.sqrt(2 * math.log(255) * lmax)                  # the candidate radius is conservative


# ---- T25: coincident camera ---------------------------------------------------------------------------------------------
def test_T25_coincident_camera_reproduces_depth_and_constant_images():
    c = cam(W=36, H=28)
    rng = np.random.default_rng(3)
    H, W = 28, 36
    flat = np.full((H, W), 2.5, np.float32)
    rgb = np.empty((H, W, 3), np.uint8); rgb[:] = (37, 180, 255)
    r = oracle.splat_forward(c, c, flat, rgb=rgb, mask=np.full((H, W), 0.6, np.float32))
    inner = (slice(3, H - 3), slice(3, W - 3))
    assert r["alpha"][inner].min() > 0.999                                  # dense opaque Gaussians saturate (T < 1e-4 stop)
    assert np.allclose(r["depth"], 2.5, rtol=1e-6)                          # every contributor has z = 2.5
    for ch, val in enumerate((37, 180, 255)):
        assert np.allclose(r["rgb"][ch], val * r["alpha"], rtol=2e-6)
    assert np.allclose(r["mask"], 0.6 * r["alpha"], rtol=2e-6)
    # a general image and a smooth depth map: each output is a convex combination of the 5 x 5 neighbourhood, front first
    img = rng.integers(0, 256, (H, W, 3), dtype=np.uint8)
    yy, xx = np.mgrid[0:H, 0:W]
    dep = (2.0 + 0.01 * xx + 0.02 * yy).astype(np.float32)
    r = oracle.splat_forward(c, c, dep, rgb=img)
    for y in range(3, H - 3):
        for x in range(3, W - 3):
            nb = img[y - 2:y + 3, x - 2:x + 3].reshape(-1, 3).astype(np.float64)
            val = r["rgb"][:, y, x] / r["alpha"][y, x]
            assert np.all(val >= nb.min(0) - 1e-3) and np.all(val <= nb.max(0) + 1e-3)
    assert np.abs(r["depth"][inner] - dep[inner]).max() < 0.05              # within the neighbourhood's depth spread ...
    assert np.all(r["depth"][inner] <= dep[inner] + 1e-6)                   # ... and never behind the pixel's own surface point
    # invalid pixels leave holes that the neighbours' tails only partly fill
    hole = flat.copy(); hole[10:16, 12:20] = 0
    r = oracle.splat_forward(c, c, hole)
    assert r["alpha"][12:14, 15:17].max() == 0 and r["depth"][12, 15] == 0 and r["alpha"][10, 12] > 0.3


# ---- T26: a fronto-parallel plane from a translated camera -----------------------------------------------------------------
def test_T26_translated_camera_integer_disparity():
    W, H, f, D, b = 48, 20, 100.0, 2.0, 0.1               # disparity f b / D = 5 px exactly
    src = cam(W=W, H=H, f=f)
    tgt = cam(centre=(b, 0, 0), W=W, H=H, f=f)
    rgb = np.zeros((H, W, 3), np.uint8)
    rgb[:, :24] = (250, 10, 10); rgb[:, 24:] = (10, 10, 250)          # two wide stripes
    r = oracle.splat_forward(tgt, src, np.full((H, W), D, np.float32), rgb=rgb)
    a = r["alpha"]
    assert a[3:H - 3, 0:W - 5 - 3].min() > 0.999                        # the plane covers columns [-5, W - 5)
    assert a[:, W - 5 + 3:].max() == 0                                  # nothing lands right of it (beyond the tails)
    # (1 - T cancels where little has landed: the quotient is good to ~1e-7 / opacity)
    assert np.all(np.abs(r["depth"][a > 0] - D) <= 4e-7 * D / a[a > 0])
    # stripe interiors keep their colour, moved left by 5 px; the edge is at column 24 - 5 = 19
    assert np.allclose(r["rgb"][:, 5, 10] / a[5, 10], (250, 10, 10), atol=1e-3)
    assert np.allclose(r["rgb"][:, 5, 30] / a[5, 30], (10, 10, 250), atol=1e-3)
    mix = r["rgb"][0, 5, 16:23] / a[5, 16:23]
    assert mix[0] > 249.9 and mix[-1] < 10.1 and np.all(np.diff(mix) <= 1e-3)


# ---- T27: occlusion --------------------------------------------------------------------------------------------------------
def test_T27_nearer_surface_wins_and_disocclusion_stays_empty():
    W, H, f, b = 64, 16, 100.0, 0.1
    src = cam(W=W, H=H, f=f)
    tgt = cam(centre=(-b, 0, 0), W=W, H=H, f=f)            # moves right: near surface shifts +10 px, far one +3.33 px
    dep = np.empty((H, W), np.float32); dep[:, :32] = 1.0; dep[:, 32:] = 3.0
    mask = np.empty((H, W), np.float32); mask[:, :32] = 1.0; mask[:, 32:] = 0.6
    r = oracle.splat_forward(tgt, src, dep, mask=mask)
    # near surface lands on columns [10, 42), far surface on [35.3, 67.3): overlap [35.3, 42)
    ov = r["depth"][4:12, 37:40]
    assert np.abs(ov - 1.0).max() < 2e-3                    # the far Gaussians are behind T < 1e-4: no blend of 1 and 3
    assert np.abs(r["mask"][4:12, 37:40] - 1.0).max() < 2e-3
    assert np.abs(r["depth"][4:12, 48:60] - 3.0).max() < 1e-5
    # reversed baseline: the surfaces pull apart, the strip between them is disoccluded
    tgt2 = cam(centre=(b, 0, 0), W=W, H=H, f=f)            # near: [-10, 22), far: [28.7, ...)
    r2 = oracle.splat_forward(tgt2, src, dep)
    assert r2["alpha"][:, 25:26].max() == 0 and r2["depth"][5, 25] == 0
    assert r2["alpha"][5, 18] > 0.999 and r2["alpha"][5, 33] > 0.99      # (centres 1/3 px off the pixel centres: peak alpha 0.9)


# ---- T28: all-pairs fp64 brute force ---------------------------------------------------------------------------------------
def _brute_splat(tgt, src, depth, rgb, mask, sigma_px=0.5, dilation=0.3, z_cull=0.2):
    H, W = depth.shape
    Ht, Wt = tgt.height, tgt.width
    Ks = np.array([[src.fx, 0, src.cx], [0, src.fy, src.cy], [0, 0, 1.0]])
    Rs, ts = src.R.astype(np.float64), src.t.astype(np.float64)
    Rt, tt = tgt.R.astype(np.float64), tgt.t.astype(np.float64)
    G = []
    for v in range(H):
        for u in range(W):
            D = float(depth[v, u])
            if not D > 0:
                continue
            Pw = Rs.T @ (D * np.linalg.inv(Ks) @ np.array([u + 0.5, v + 0.5, 1.0]) - ts)
            q = Rt @ Pw + tt
            if q[2] < z_cull:
                continue
            mu = np.array([tgt.fx * q[0] / q[2] + tgt.cx, tgt.fy * q[1] / q[2] + tgt.cy])
            J = np.array([[tgt.fx / q[2], 0, -tgt.fx * q[0] / q[2] ** 2], [0, tgt.fy / q[2], -tgt.fy * q[1] / q[2] ** 2]])
            sig = sigma_px * D / src.fx
            S = sig * sig * (J @ J.T) + dilation * np.eye(2)
            G.append((q[2], v * W + u, mu, np.linalg.inv(S)))
    out = dict(rgb=np.zeros((3, Ht, Wt)), alpha=np.zeros((Ht, Wt)), depth=np.zeros((Ht, Wt)), mask=np.zeros((Ht, Wt)))
    fragile = np.zeros((Ht, Wt), bool)
    order = sorted(range(len(G)), key=lambda i: (np.float32(G[i][0]), G[i][1]))      # depth key as the fp32 both sides sort by
    for py in range(Ht):
        for px in range(Wt):
            pc = np.array([px + 0.5, py + 0.5])
            T, C, Dacc, Macc = 1.0, np.zeros(3), 0.0, 0.0
            for i in order:
                z, idx, mu, conic = G[i]
                d = mu - pc
                qv = -0.5 * d @ conic @ d
                a = min(0.99, math.exp(qv))
                if abs(a * 255.0 - 1.0) < 2e-4:
                    fragile[py, px] = True
                if a < 1.0 / 255.0:
                    continue
                t2 = T * (1 - a)
                if abs(t2 / 1e-4 - 1.0) < 2e-3:
                    fragile[py, px] = True
                if t2 < 1e-4:
                    break
                w = a * T
                C += rgb.reshape(-1, 3)[idx] * w
                Dacc += z * w
                Macc += mask.reshape(-1)[idx] * w
                T = t2
            acc = 1 - T
            out["rgb"][:, py, px] = C; out["alpha"][py, px] = acc
            out["depth"][py, px] = Dacc / acc if acc > 0 else 0.0
            out["mask"][py, px] = Macc
    return out, fragile


@pytest.mark.parametrize("case", ["rotated", "ties"])
def test_T28_all_pairs_bruteforce_fp64(case):
    rng = np.random.default_rng(11)
    W, H = 14, 11
    src = cam(centre=(0.05, -0.02, 0.0), R=synth.rot_yaw_pitch(0.03, -0.02), f=22.0, W=W, H=H)
    if case == "rotated":
        tgt = cam(centre=(-0.12, 0.06, 0.25), R=synth.rot_yaw_pitch(-0.08, 0.05), f=30.0, W=18, H=13)
        depth = rng.uniform(1.0, 3.0, (H, W)).astype(np.float32)          # a rough surface: many occlusions
        depth[rng.uniform(size=(H, W)) < 0.1] = 0
    else:
        src = cam(f=22.0, W=W, H=H)
        tgt = cam(centre=(0.07, 0.0, 0.0), f=22.0, W=18, H=13)             # parallel cameras: z = D exactly, ties everywhere
        depth = np.where(rng.uniform(size=(H, W)) < 0.5, 1.5, 2.25).astype(np.float32)
    rgb = rng.integers(0, 256, (H, W, 3), dtype=np.uint8)
    mask = rng.uniform(0.6, 1.0, (H, W)).astype(np.float32)
    r = oracle.splat_forward(tgt, src, depth, rgb=rgb, mask=mask)
    ref, fragile = _brute_splat(tgt, src, depth, rgb.astype(np.float64), mask.astype(np.float64))
    ok = ~fragile
    assert ok.mean() > 0.9
    assert np.abs(r["alpha"] - ref["alpha"])[ok].max() < 2e-5
    assert np.abs(r["rgb"] - ref["rgb"])[:, ok].max() < 255 * 2e-5
    assert np.abs(r["depth"] - ref["depth"])[ok].max() < 1e-4
    assert np.abs(r["mask"] - ref["mask"])[ok].max() < 2e-5
    assert (ref["alpha"] > 0.5).mean() > 0.3 and (ref["alpha"] == 0).any()


# ---- Eq. 13 with a given novel-view mask -----------------------------------------------------------------------------------
def test_temporal_weight_from_a_splatted_mask_closed_form():
    d = np.array([2.0, 2.0, 0.0, 2.0, 2.0, 2.0], np.float32)
    conf = np.array([4.0, 4.0, 4.0, 0.0, 40.0, 4.0], np.float32)
    M = np.array([0.6, 1.0, 0.6, 0.6, 0.0, 1.3], np.float32)
    w = oracle.temporal_weight_mask(d, conf, M, beta=0.5, eta=15.0)
    # min(beta omega_acc max(1 - M, 0), eta): 0.5*4*0.4 | M = 1 -> 0 | no depth | no weight | capped at eta | M > 1 -> 0
    assert np.allclose(w, [0.8, 0.0, 0.0, 0.0, 15.0, 0.0], atol=1e-6)


# ---- F1's gather and the paper's splat-and-max differ exactly where a surface point is occluded in an input view ------------
def test_splatted_mask_differs_from_the_gather_at_occluded_points():
    """Eq. 13's novel-view mask two ways (readings F1 and S1-S8).  A moving foreground strip (mask 1) in front
    of a static wall (mask 0.6), one input view 20 cm to the side of the camera of D^{t-1}.  For wall points that the
    strip hides from the input view, the gather (orc_temporal_weight) projects the wall point into the view and reads
    the STRIP's mask, so the static wall loses its temporal weight; the splat composites the view's own surfaces front
    to back, nothing of the view lands on those pixels, and the weight survives.  Everywhere else the two agree."""
    W, H, f = 96, 24, 100.0
    prev = cam(W=W, H=H, f=f)
    view = cam(centre=(0.2, 0, 0), W=W, H=H, f=f)
    scene = synth.Scene(3.0, [synth.Primitive("box", np.array([0.0, 0.0, 1.0]), np.array([0.08, 2.0, 0.001]), np.zeros(3), np.zeros(9))])
    d_prev = synth.raycast(prev, scene)[0].astype(np.float32)
    d_view = synth.raycast(view, scene)[0].astype(np.float32)
    m_view = np.where(d_view < 2.0, 1.0, 0.6).astype(np.float32)          # the strip moved, the wall did not
    conf = np.full((H, W), 4.0, np.float32)
    w_gather = oracle.temporal_weight(prev, d_prev, conf, [view], [m_view], beta=1.0, eta=15.0)
    sp = oracle.splat_forward(prev, view, d_view, mask=m_view)
    w_splat = oracle.temporal_weight_mask(d_prev, conf, sp["mask"], beta=1.0, eta=15.0)
    row = H // 2
    wall = d_prev[row] > 2.0
    # wall pixels of D^{t-1} whose surface point projects onto the strip in the input view: hidden from it
    x_in_view = (np.arange(W) + 0.5 - prev.cx) / f * 3.0 - 0.2              # world x of the wall point, relative to the view
    u_view = np.floor(x_in_view / 3.0 * f + view.cx).astype(int)
    hidden = wall & (u_view >= 0) & (u_view < W)
    hidden[hidden] = d_view[row, u_view[hidden]] < 2.0
    assert hidden.sum() >= 4
    assert np.allclose(w_gather[row, hidden], 0.0)                          # the gather read the occluder's mask (M = 1)
    inner = hidden & np.roll(hidden, 2) & np.roll(hidden, -2)               # away from the splats' 2-px tails
    assert inner.sum() >= 1 and np.allclose(w_splat[row, inner], 4.0)       # nothing of the view lands there: M = 0
    # a wall point both cameras see, far from the strip: both give beta * omega_acc * (1 - 0.6)
    far = wall & ~hidden & (np.abs(np.arange(W) - W // 2) > 30) & (u_view >= 3) & (u_view < W - 3)
    assert far.sum() > 10
    assert np.allclose(w_gather[row, far], 1.6, atol=1e-5) and np.allclose(w_splat[row, far], 4.0 * (1 - 0.6 * sp["alpha"][row, far]), atol=1e-4)
    assert np.abs(w_splat[row, far] - 1.6).max() < 0.01
