"""Pins of the oracle's temporal fusion weight (O-T: Eq. 3, Eq. 13-14) and of the
previous output depth used as one more TSDF view (-m "not gpu").  T15 Eq. 13 closed forms, T16 the novel-view mask
against an fp64 brute force with explicit world points, T17 the recursion of Eq. 14 through the full loop in closed
form, T18 the statistical effect (temporal variance of the output depth drops on a static scene)."""
import math

import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth

TAU, NEAR, FAR = 0.02, 0.5, 5.0


def rig4():
    rig = synth.grid_rig(96, 64)
    tgt = synth.camera_from_pose((0.03, -0.02, 0.0), np.eye(3), 72, 72, 48, 32, 96, 64)
    return tgt, [rig[i] for i in synth.nearest_views(tgt, rig, 4)]


def const_maps(cams, d, omega=1.0):
    out = []
    for c in cams:
        m = np.empty((c.height, c.width, 2), dtype=np.float32)
        m[..., 0] = d
        m[..., 1] = omega
        out.append(m)
    return out


# ---- T15: Eq. 13 closed forms --------------------------------------------------------------------------
@pytest.mark.parametrize("beta,acc,M,eta,expect", [
    (0.9, 4.0, 0.6, 15.0, 0.9 * 4.0 * 0.4),        # static region: Eq. 1's floor beta_mask = 0.6 -> 1 - M = 0.4
    (1.0, 4.0, 1.0, 15.0, 0.0),                    # dynamic region: the previous depth is ignored
    (1.0, 4.0, 1.3, 15.0, 0.0),                    # max(1 - M, 0)
    (1.0, 100.0, 0.6, 15.0, 15.0),                 # capped at eta
    (0.5, 19.0, 0.0, 15.0, 9.5),
])
def test_T15_eq13_closed_forms(beta, acc, M, eta, expect):
    tgt, views = rig4()
    d = np.full((tgt.height, tgt.width), 2.0, np.float32)
    c = np.full_like(d, acc)
    masks = [np.full((v.height, v.width), M, np.float32) for v in views]
    w = oracle.temporal_weight(tgt, d, c, views, masks, beta=beta, eta=eta)
    # at 2 m every pixel of this target projects into at least one of the 4 nearest rig cameras
    assert np.allclose(w, expect, rtol=1e-6, atol=1e-7)
    # invalid previous depth / no accumulated weight -> 0
    d2, c2 = d.copy(), c.copy()
    d2[3, 5] = 0.0; c2[7, 9] = 0.0
    w2 = oracle.temporal_weight(tgt, d2, c2, views, masks, beta=beta, eta=eta)
    assert w2[3, 5] == 0 and w2[7, 9] == 0
    # a surface point no input view sees has M^t = 0 (reading F1)
    far_cam = synth.camera_from_pose((50.0, 0, 0), np.eye(3), 72, 72, 48, 32, 96, 64)
    w3 = oracle.temporal_weight(far_cam, d, c, views, masks, beta=beta, eta=eta)
    assert np.allclose(w3, min(beta * acc, eta), rtol=1e-6)


# ---- T16: the novel-view mask against an fp64 brute force ----------------------------------------------
def test_T16_mask_gather_bruteforce_fp64():
    wl = synth.workload("C2", scale=0.1)
    tgt = synth.camera_from_pose((0.05, 0.02, -0.03), synth.rot_yaw_pitch(0.03, -0.02), 50, 50, 32, 18, 64, 36)
    views = [wl.rig[i] for i in synth.nearest_views(tgt, wl.rig, 4)]
    rng = np.random.default_rng(16)
    d = synth.raycast(tgt, wl.scene)[0].astype(np.float32)
    d[rng.uniform(size=d.shape) < 0.05] = 0
    acc = rng.uniform(0.5, 6.0, d.shape).astype(np.float32)
    masks = [rng.uniform(0.6, 1.0, (v.height, v.width)).astype(np.float32) for v in views]
    beta, eta = 0.8, 3.0
    w = oracle.temporal_weight(tgt, d, acc, views, masks, beta=beta, eta=eta)
    Kt = np.array([[tgt.fx, 0, tgt.cx], [0, tgt.fy, tgt.cy], [0, 0, 1]], dtype=np.float64)
    Kti = np.linalg.inv(Kt)
    n_checked = 0
    for v in range(tgt.height):
        for u in range(tgt.width):
            if not d[v, u] > 0:
                assert w[v, u] == 0
                continue
            p = tgt.R.astype(np.float64).T @ (float(d[v, u]) * (Kti @ np.array([u + 0.5, v + 0.5, 1.0])) - tgt.t.astype(np.float64))
            Mmax, fragile = 0.0, False
            for cam, m in zip(views, masks):
                Kk = np.array([[cam.fx, 0, cam.cx], [0, cam.fy, cam.cy], [0, 0, 1]], dtype=np.float64)
                x, y, z = Kk @ (cam.R.astype(np.float64) @ p + cam.t.astype(np.float64))
                if z < 1e-6:
                    continue
                px, py = x / z, y / z
                fragile |= min(abs(px - round(px)), abs(py - round(py))) < 2.0 ** -9
                ix, iy = math.floor(px), math.floor(py)
                if 0 <= ix < cam.width and 0 <= iy < cam.height:
                    Mmax = max(Mmax, float(m[iy, ix]))
            if fragile:
                continue
            expect = min(beta * float(acc[v, u]) * max(1.0 - Mmax, 0.0), eta)
            assert abs(w[v, u] - expect) <= 1e-5 * max(expect, 1e-3), (u, v, w[v, u], expect)
            n_checked += 1
    assert n_checked > 0.9 * (d > 0).sum()


# ---- T17: Eq. 14's recursion through the full loop, closed form ----------------------------------------
@pytest.mark.parametrize("beta,M,eta", [(1.0, 0.6, 15.0), (0.7, 0.0, 15.0), (1.0, 0.0, 6.0), (1.0, 1.0, 15.0)])
def test_T17_accumulated_weight_recursion(beta, M, eta):
    """Static fronto-parallel plane, omega_k = 1 for the V = 4 input views, constant mask M, target fixed: the
    confidence returned at frame t is omega_acc^{t+1} of Eq. 14, so
        conf_t = V + min(beta * conf_{t-1} * max(1 - M, 0), eta),  conf_0 = V
    wherever all views and the previous output see the surface, and the depth stays the plane's."""
    tgt, views = rig4()
    dplane = 2.0
    maps = const_maps(views, dplane)
    masks = [np.full((v.height, v.width), M, np.float32) for v in views]
    depth, conf, _ = oracle.raymarch(tgt, views, maps, NEAR, FAR, tau=TAU)
    inner = (conf == 4.0) & (depth > 0)
    assert inner.mean() > 0.5
    expect = 4.0
    for t in range(1, 8):
        w = oracle.temporal_weight(tgt, depth, conf, views, masks, beta=beta, eta=eta)
        rec = oracle.view_record(depth.reshape(tgt.height, tgt.width), w)
        depth, conf, _ = oracle.raymarch(tgt, views + [tgt], maps + [rec], NEAR, FAR, tau=TAU)
        expect = 4.0 + min(beta * expect * max(1.0 - M, 0.0), eta)
        assert np.allclose(conf[inner], expect, rtol=1e-5), (t, conf[inner][:3], expect)
        assert np.max(np.abs(depth[inner] - dplane)) <= 0.8 * TAU / 16 + 1e-6
    if M < 1.0 and beta * (1.0 - M) >= 1.0:
        assert expect == pytest.approx(4.0 + eta)          # the cap is reached and holds


# ---- T18: what the temporal view is for ----------------------------------------------------------------
def test_T18_temporal_view_reduces_frame_to_frame_variation():
    """Static scene, independent depth noise per frame (sigma 0.5 %), masks at Eq. 1's static floor 0.6: the marched
    depth with D^{t-1} fused in (Eq. 3) varies less from frame to frame than without, with the same mean."""
    wl = synth.workload("C1", scale=1.0)
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    views = [wl.rig[i] for i in vi]
    clean = [synth.raycast(c, wl.scene)[0].astype(np.float32) for c in views]
    masks = [np.full((v.height, v.width), 0.6, np.float32) for v in views]
    gt = wl.true_depth(tgt, 0).reshape(-1)
    plain, fused = [], []
    pd = pc = None
    for t in range(10):
        depths = [synth.noisy_depth(c, 180 + t, i, 0.005, 0.0) for i, c in enumerate(clean)]
        maps = [oracle.weight_map(d) for d in depths]
        d0, c0, _ = oracle.raymarch(tgt, views, maps, NEAR, 4.0, tau=TAU)
        plain.append(d0)
        if pd is None:
            pd, pc = d0, c0
        else:
            w = oracle.temporal_weight(tgt, pd, pc, views, masks, beta=1.0, eta=15.0)
            rec = oracle.view_record(pd.reshape(tgt.height, tgt.width), w)
            pd, pc, _ = oracle.raymarch(tgt, views + [tgt], maps + [rec], NEAR, 4.0, tau=TAU)
        fused.append(pd)
    plain, fused = np.array(plain[3:]), np.array(fused[3:])
    ok = np.all(plain > 0, axis=0) & np.all(fused > 0, axis=0) & (np.abs(plain.mean(0) - gt) < 0.05)
    assert ok.mean() > 0.6
    sp, sf = plain[:, ok].std(axis=0).mean(), fused[:, ok].std(axis=0).mean()
    assert sf < 0.75 * sp, (sf, sp)
    bp, bf = (plain[:, ok].mean(0) - gt[ok]).mean(), (fused[:, ok].mean(0) - gt[ok]).mean()
    assert abs(bf - bp) < 2e-3, (bp, bf)          # fusing D^{t-1} adds no bias of its own (the cut at -tau has one)
