"""Pins of the CPU oracle against what the paper and the mathematics fix.

CPU only (-m "not gpu").  Nothing here calls the CUDA path; expected values are closed forms,
invariants, library routines (numpy float16 conversion) or an independent brute-force fp64
restatement written out below with no hoisting.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])


# ------------------------------------------------------------------------------------------------
# helpers
# ------------------------------------------------------------------------------------------------
def const_maps(cams, d, omega=1.0):
    out = []
    for c in cams:
        m = np.empty((c.height, c.width, 2), dtype=np.float32)
        m[..., 0] = d
        m[..., 1] = omega
        out.append(m)
    return out


def run_oracle(target, z, views, maps, trunc_bins=2.0, trunc_metric=0.0, **kw):
    tau = oracle.tau_table(z, trunc_bins, trunc_metric)
    T, W = oracle.integrate(target, z, tau, views, maps, **kw)
    depth, conf, bins = oracle.extract(z, T, W)
    return T, W, depth, conf, bins, tau


# ------------------------------------------------------------------------------------------------
# binary16 emulation vs numpy's conversion (library routine)
# ------------------------------------------------------------------------------------------------
def test_f16_rounding_matches_numpy():
    rng = np.random.default_rng(5)
    xs = np.concatenate([
        rng.standard_normal(4000).astype(np.float32) * np.float32(10.0) ** rng.integers(-9, 5, 4000).astype(np.float32),
        np.array([0.0, -0.0, 1.0, 65504.0, 65519.9, 65520.0, 1e-8, 5.96e-8, 2.98e-8, 2.9802322e-8, 2.99e-8,
                  6.1e-5, 6.0975552e-05, 1.0009765625, 1.00048828125, 1.00146484375, 64.0, 0.333333],
                 dtype=np.float32)])
    with np.errstate(over="ignore"):
        ref = xs.astype(np.float16).astype(np.float32)
    got = np.array([oracle.round_f16(float(x)) for x in xs], dtype=np.float32)
    assert np.array_equal(ref.view(np.uint32), got.view(np.uint32))


# ------------------------------------------------------------------------------------------------
# T5 / T6: Eq. 1-2
# ------------------------------------------------------------------------------------------------
def test_T5_identical_images_give_beta():
    H, W = 32, 48
    rgb = (np.arange(H * W * 3) % 251).astype(np.uint8).reshape(H, W, 3)
    d = np.full((H, W), 2.0, np.float32)
    out, M, pq, bq = oracle.refine(rgb, rgb.copy(), d, d + 1.0, theta=0.0)
    assert np.all(pq == 0) and np.all(bq == 0)
    assert np.all(M == np.float32(GOLD["beta"]))
    # Eq. 2 with M = beta: 0.6*2 + 0.4*3 = 2.4
    assert np.allclose(out, 0.6 * 2.0 + 0.4 * 3.0, rtol=0, atol=1e-6)


@pytest.mark.parametrize("k", [1, 5, 10, 20, 28, 29, 40])
def test_T5_eq1_closed_form_uniform_change(k):
    H, W = 16, 16
    prev = np.full((H, W, 3), 100, np.uint8)
    cur = np.full((H, W, 3), 100 + k, np.uint8)
    d = np.ones((H, W), np.float32)
    _, M, pq, _ = oracle.refine(cur, prev, d, d, theta=0.0)
    assert np.all(pq == 3 * 16 * k)
    delta = 3.0 * k / 255.0                       # L1 over RGB of colours in [0,1]
    expect = min(delta / GOLD["lambda_t"] + GOLD["beta"], 1.0)   # Eq. 1
    assert np.allclose(M, expect, rtol=0, atol=2e-7)


def test_T5_single_block_pool_and_bilinear_ramp():
    H, W = 64, 64
    prev = np.full((H, W, 3), 50, np.uint8)
    cur = prev.copy()
    c = 7                                          # changed quarter-res cell (7,7)
    cur[4 * c:4 * c + 4, 4 * c:4 * c + 4, :] = 250   # block-mean L1 = 3*200/255 >> lambda_t*(1-beta)
    d = np.ones((H, W), np.float32)
    _, M, pq, bq = oracle.refine(cur, prev, d, d, theta=8.0 / 255.0)
    beta = np.float32(0.6)
    # pooled: 3x3 cells around c carry the block's value
    assert np.all(pq[c - 1:c + 2, c - 1:c + 2] == 3 * 16 * 200)
    assert pq.sum() == 9 * 3 * 16 * 200
    assert bq.sum() == 9
    row = M[4 * c + 1]                             # a row through the saturated core
    assert np.all(row[4 * c - 2:4 * c + 6] == 1.0)            # central 8 px
    for i, f in enumerate([1 / 8, 3 / 8, 5 / 8, 7 / 8]):       # 4-px linear ramps, 16-px support
        e = float(beta) + f * (1.0 - float(beta))
        assert abs(row[4 * c - 6 + i] - e) < 2e-7
        assert abs(row[4 * c + 9 - i] - e) < 2e-7
    assert np.all(row[:4 * c - 6] == beta) and np.all(row[4 * c + 10:] == beta)
    assert np.all(M[:4 * c - 6, :] == beta) and np.all(M[4 * c + 10:, :] == beta)
    # symmetric in x and y
    assert np.array_equal(M, M.T)


def test_T5_threshold_dead_zone():
    # L1 block difference just at / above 8/255 (pq = 128 / 129): binary mask flips exactly there
    H, W = 8, 8
    prev = np.zeros((H, W, 3), np.uint8)
    cur = prev.copy()
    cur[0:4, 0:4, 0] = 8                           # 16 px * 8 = 128  -> not above threshold
    d = np.ones((H, W), np.float32)
    _, M, pq, bq = oracle.refine(cur, prev, d, d, theta=8.0 / 255.0)
    assert pq.max() == 128 and bq.sum() == 0
    assert np.allclose(M, 0.6, atol=1e-6)
    cur[0, 0, 1] = 1                               # 129
    _, M, pq, bq = oracle.refine(cur, prev, d, d, theta=8.0 / 255.0)
    assert pq.max() == 129 and bq.sum() == 4       # 2x2 cells, all inside the clipped 3x3 window
    assert M.max() > 0.6


def test_T6_first_frame_and_full_mask_are_bit_exact():
    H, W = 16, 24
    rng = np.random.default_rng(1)
    d = rng.uniform(1, 3, (H, W)).astype(np.float32)
    prev_state = rng.uniform(1, 3, (H, W)).astype(np.float32)
    out, M, _, _ = oracle.refine(None, None, d, prev_state)
    assert np.array_equal(out, d) and np.all(M == 1.0)
    a = np.zeros((H, W, 3), np.uint8)
    b = np.full((H, W, 3), 255, np.uint8)
    out, M, _, _ = oracle.refine(b, a, d, prev_state)
    assert np.all(M == 1.0)
    assert np.array_equal(out, d)                  # fmaf(1, d - p, p) == d needs d-p+p == d: check
    # invalid handling (reading P17): single valid term wins, none -> 0
    d2 = d.copy(); d2[0, 0] = 0; ps = prev_state.copy(); ps[0, 1] = 0; d2[0, 2] = 0; ps[0, 2] = 0
    out, _, _, _ = oracle.refine(a, a, d2, ps)
    assert out[0, 0] == ps[0, 0] and out[0, 1] == d2[0, 1] and out[0, 2] == 0


def test_T6_ema_variance_ratio():
    H, W = 64, 64
    rgb = np.full((H, W, 3), 77, np.uint8)
    rng = np.random.default_rng(2)
    state = np.full((H, W), 2.0, np.float32)
    outs = []
    for t in range(60):
        d = (2.0 + 0.01 * rng.standard_normal((H, W))).astype(np.float32)
        state, _, _, _ = oracle.refine(rgb, rgb, d, state)
        if t >= 30:
            outs.append(state.copy())
    var = np.var(np.stack(outs) - 2.0)
    ratio = var / 1e-4
    assert abs(ratio - GOLD["ema_variance_ratio"]) < 0.03 * GOLD["ema_variance_ratio"]


# ------------------------------------------------------------------------------------------------
# T7: Eq. 11-12
# ------------------------------------------------------------------------------------------------
def test_T7_weight_closed_forms():
    H, W = 21, 21
    flat = np.full((H, W), 2.0, np.float32)
    m = oracle.weight_map(flat)
    assert np.all(m[3:-3, 3:-3, 1] == 1.0) and np.array_equal(m[..., 0], flat)
    # all 48 neighbours beyond the clip
    spike = flat.copy(); spike[10, 10] = 3.0
    m = oracle.weight_map(spike)
    assert abs(m[10, 10, 1] - GOLD["omega_all_clipped"]) < 1e-7
    assert abs(GOLD["omega_all_clipped"] - 0.001 * 7 / (0.02 * math.sqrt(48))) < 1e-9
    # neighbours of the spike see exactly one clipped neighbour: nu = clip^2 -> 0.001*7/0.02 = 0.35
    assert abs(m[10, 11, 1] - 0.35) < 1e-6
    # checkerboard +-a: 24 opposite-parity neighbours, each (2a)^2
    a = 0.004
    yy, xx = np.mgrid[0:H, 0:W]
    cb = (2.0 + a * (1 - 2 * ((xx + yy) & 1))).astype(np.float32)
    m = oracle.weight_map(cb)
    d2 = float(np.float32(cb[0, 0]) - np.float32(cb[0, 1])) ** 2
    expect = 0.001 / math.sqrt(24 * d2 / 49.0)
    assert abs(m[10, 10, 1] - expect) < 1e-6 * expect + 1e-7
    # border rule (P11): corner of a flat map has 33 missing neighbours
    m = oracle.weight_map(flat)
    assert abs(m[0, 0, 1] - 0.001 * 7 / (0.02 * math.sqrt(33))) < 1e-7
    # invalid centre -> omega 0; invalid neighbour counts as clip^2; window 0 -> 1
    hole = flat.copy(); hole[5, 5] = 0.0
    m = oracle.weight_map(hole)
    assert m[5, 5, 1] == 0.0 and abs(m[5, 6, 1] - 0.35) < 1e-6
    m0 = oracle.weight_map(hole, window=0)
    assert m0[5, 5, 1] == 0.0 and m0[..., 1].sum() == H * W - 1


# ------------------------------------------------------------------------------------------------
# T1: analytic scenes
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bins", ["uniform", "inverse"])
def test_T1_frontoparallel_plane_exact(bins):
    rig = synth.grid_rig(96, 64)
    tgt = synth.camera_from_pose((0.03, -0.02, 0.0), np.eye(3), 72, 72, 48, 32, 96, 64)
    vi = synth.nearest_views(tgt, rig, 4)
    z = synth.bins_uniform(0.5, 5, 48) if bins == "uniform" else synth.bins_inverse(0.5, 5, 48)
    for d in [0.9, 2.3456, 4.2]:
        views = [rig[i] for i in vi]
        T, W, depth, conf, bn, tau = run_oracle(tgt, z, views, const_maps(views, d))
        seen = depth > 0
        assert seen.mean() > 0.95
        assert np.max(np.abs(depth[seen] - d)) <= 4e-6 * d
        j = np.searchsorted(z, np.float32(d), side="left") - 1   # z_j < d <= z_{j+1}
        assert np.all(bn[seen] == j)
        assert np.all(conf[seen] <= 4.0 + 1e-6) and np.all(conf[seen] >= 1.0 - 1e-6)


def _interior(gt, px=3, rel=0.02):
    """Pixels >= px away from a ground-truth depth edge."""
    H, W = gt.shape
    edge = np.zeros_like(gt, dtype=bool)
    edge[:, 1:] |= np.abs(gt[:, 1:] - gt[:, :-1]) > rel * gt[:, 1:]
    edge[1:, :] |= np.abs(gt[1:, :] - gt[:-1, :]) > rel * gt[1:, :]
    edge[:, :-1] |= edge[:, 1:].copy()
    edge[:-1, :] |= edge[1:, :].copy()
    near = edge.copy()
    for _ in range(px):
        g = near.copy()
        g[1:, :] |= near[:-1, :]; g[:-1, :] |= near[1:, :]; g[:, 1:] |= near[:, :-1]; g[:, :-1] |= near[:, 1:]
        near = g
    return ~near


@pytest.mark.parametrize("name", ["C1", "C2"])
def test_T1_sphere_and_plane_scene_within_one_bin(name):
    wl = synth.workload(name, scale=1.0 if name == "C1" else 0.25)
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    views = [wl.rig[i] for i in vi]
    # noise-free analytic depth maps
    maps = [oracle.weight_map(synth.raycast(c, wl.scene)[0].astype(np.float32)) for c in views]
    T, W, depth, conf, bn, tau = run_oracle(tgt, wl.z_bins, views, maps)
    gt = wl.true_depth(tgt, 0)
    depth = depth.reshape(gt.shape)
    # interior = away from depth edges and seen by all views at the true depth
    inter = _interior(gt)
    conf_full = conf.reshape(gt.shape)
    jj = np.clip(np.searchsorted(wl.z_bins, gt.astype(np.float32)) - 1, 0, wl.z_bins.size - 2)
    spacing = (wl.z_bins[jj + 1] - wl.z_bins[jj]).astype(np.float64)
    Wvol = W.reshape(gt.shape + (-1,))
    allseen = np.take_along_axis(Wvol, jj[..., None], axis=2)[..., 0] > 0
    sel = inter & allseen & (gt > wl.z_bins[0]) & (gt < wl.z_bins[-1])
    assert sel.mean() > 0.5
    good = np.abs(depth - gt) <= spacing
    assert good[sel].mean() >= 0.99, good[sel].mean()
    # and far better than a bin on smooth surfaces in the median
    assert np.median(np.abs(depth - gt)[sel] / spacing[sel]) < 0.25


# ------------------------------------------------------------------------------------------------
# T2: coincident camera reproduces its own depth map
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bins", ["uniform", "inverse"])
def test_T2_coincident_camera_identity(bins):
    wl = synth.workload("C2", scale=0.2)
    cam = wl.rig[5]
    d = wl.view_inputs(0, 5)[0]                   # noisy, 2 % invalid
    n = 64
    z = synth.bins_uniform(0.5, 5, n) if bins == "uniform" else synth.bins_inverse(0.5, 5, n)
    T, W, depth, conf, bn, tau = run_oracle(cam, z, [cam], [oracle.weight_map(d)])
    depth = depth.reshape(d.shape)
    inrange = (d > z[0]) & (d <= z[-1])
    assert inrange.mean() > 0.9
    rel = np.abs(depth[inrange] - d[inrange]) / d[inrange]
    assert rel.max() <= 2e-6
    assert np.all(depth[d <= 0] == 0) and np.all(bn.reshape(d.shape)[d <= 0] == -1)
    assert np.all(depth[d > z[-1]] == 0)


# ------------------------------------------------------------------------------------------------
# T3: invariance to the order of the input views
# ------------------------------------------------------------------------------------------------
def test_T3_view_order_invariance():
    wl = synth.workload("C2", scale=0.2)
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    views = [wl.rig[i] for i in vi]
    maps = [oracle.weight_map(wl.view_inputs(0, i)[0]) for i in vi]
    T0, W0, d0, c0, b0, tau = run_oracle(tgt, wl.z_bins, views, maps)
    perm = [2, 0, 3, 1]
    T1, W1, d1, c1, b1, _ = run_oracle(tgt, wl.z_bins, [views[p] for p in perm], [maps[p] for p in perm])
    assert np.max(np.abs(T0 - T1) / tau[None, :]) <= 1e-5
    assert np.max(np.abs(W0 - W1)) <= 1e-5
    # bins identical except where the TSDF is within rounding of zero at the crossing
    diff = b0 != b1
    assert diff.mean() < 1e-4
    assert np.max(np.abs(d0 - d1)) <= 1e-4 * (wl.z_bins[-1] - wl.z_bins[0])


# ------------------------------------------------------------------------------------------------
# T4: brute force per voxel in double, explicit world point, no hoisting
# ------------------------------------------------------------------------------------------------
def _brute(target, z, tau, views, maps):
    """(T, W, fragile) for every voxel; direct restatement of PAPER.md:331-348 in fp64."""
    Wd, Hd, D = target.width, target.height, len(z)
    T = np.zeros((Hd * Wd, D)); Wt = np.zeros((Hd * Wd, D)); frag = np.zeros((Hd * Wd, D), bool)
    Kt = np.array([[target.fx, 0, target.cx], [0, target.fy, target.cy], [0, 0, 1]], dtype=np.float64)
    Kti = np.linalg.inv(Kt)
    Rt = target.R.astype(np.float64); tt = target.t.astype(np.float64)
    for v in range(Hd):
        for u in range(Wd):
            ray = Kti @ np.array([u + 0.5, v + 0.5, 1.0])
            for j in range(D):
                p = Rt.T @ (float(z[j]) * ray - tt)            # world point at z-depth z_j
                A = 0.0; Wn = 0.0; fr = False
                for cam, m in zip(views, maps):
                    Kk = np.array([[cam.fx, 0, cam.cx], [0, cam.fy, cam.cy], [0, 0, 1]], dtype=np.float64)
                    x, y, w = Kk @ (cam.R.astype(np.float64) @ p + cam.t.astype(np.float64))
                    if w < 1e-6:
                        continue
                    px, py = x / w, y / w
                    if min(abs(px - round(px)), abs(py - round(py))) < 2.0 ** -9:
                        fr = True
                    ix, iy = math.floor(px), math.floor(py)
                    if ix < 0 or iy < 0 or ix >= cam.width or iy >= cam.height:
                        continue
                    Dk, om = float(m[iy, ix, 0]), float(m[iy, ix, 1])
                    if Dk <= 0:
                        continue
                    s = Dk - w
                    if abs(s + float(tau[j])) < 1e-5:
                        fr = True
                    if s < -float(tau[j]):
                        continue
                    A += om * min(s, float(tau[j])); Wn += om
                r = v * Wd + u
                frag[r, j] = fr
                if Wn > 0:
                    T[r, j] = A / Wn; Wt[r, j] = Wn
    return T, Wt, frag


def test_T4_bruteforce_fp64_tiny_grid():
    rig = synth.arc_rig()
    # tiny cameras: shrink the C1 rig to 16x12
    def shrink(c):
        return synth.Camera(15, 15, 8, 6, c.R, c.t, 16, 12)
    views = [shrink(c) for c in rig]
    tgt = synth.camera_from_pose((0.02, 0.01, -1.9), synth.rot_yaw_pitch(0.02, -0.015), 15, 15, 8, 6, 16, 12)
    wl = synth.workload("C1")
    maps = [oracle.weight_map(synth.noisy_depth(synth.raycast(c, wl.scene)[0], 7, i, 0.005, 0.05))
            for i, c in enumerate(views)]
    z = synth.bins_uniform(0.5, 4.0, 16)
    tau = oracle.tau_table(z, 2.0)
    T, W = oracle.integrate(tgt, z, tau, views, maps)
    Tb, Wb, frag = _brute(tgt, z, tau, views, maps)
    ok = ~frag
    assert ok.mean() > 0.9
    assert np.max(np.abs(W - Wb)[ok] / np.maximum(Wb[ok], 1e-12)) <= 1e-5
    small = np.abs(Tb) < 1e-6
    rel = np.abs(T - Tb) / np.maximum(np.abs(Tb), 1e-12)
    assert np.max(rel[ok & ~small]) <= 1e-5 * 20   # cancellation in Dk - w: bound by tau-relative below
    assert np.max((np.abs(T - Tb) / tau[None, :])[ok]) <= 1e-5
    assert (Wb > 0).mean() > 0.3 and (Tb < 0).sum() > 10 and (Tb > 0).sum() > 10
    # tau table: 2 x local spacing, one-sided at the ends (reading P3)
    assert np.allclose(tau, 2 * (z[1] - z[0]), rtol=1e-5)


def test_relative_transform_against_direct_projection():
    rng = np.random.default_rng(3)
    tgt = synth.camera_from_pose((0.1, -0.2, 0.05), synth.rot_yaw_pitch(0.05, 0.03), 500, 480, 320, 180, 640, 360)
    view = synth.camera_from_pose((-0.3, 0.1, 0.0), synth.rot_yaw_pitch(-0.04, 0.01), 480, 490, 310, 185, 640, 360)
    Hm, e = oracle.relative(tgt, view)
    Kt = np.array([[tgt.fx, 0, tgt.cx], [0, tgt.fy, tgt.cy], [0, 0, 1]], dtype=np.float64)
    Kk = np.array([[view.fx, 0, view.cx], [0, view.fy, view.cy], [0, 0, 1]], dtype=np.float64)
    for _ in range(50):
        u, v, zz = rng.uniform(0, 640), rng.uniform(0, 360), rng.uniform(0.5, 5)
        p = tgt.R.astype(np.float64).T @ (zz * np.linalg.inv(Kt) @ np.array([u, v, 1.0]) - tgt.t.astype(np.float64))
        ref = Kk @ (view.R.astype(np.float64) @ p + view.t.astype(np.float64))
        got = zz * (Hm.astype(np.float64) @ np.array([u, v, 1.0])) + e
        assert np.allclose(ref, got, rtol=2e-6, atol=2e-4)


def test_tau_table_on_non_uniform_bins_hand_computed():
    """orc_tau_table on bins that are NOT uniform (reading P3): tau_j = trunc_bins x the local
    spacing (z[j+1] - z[j-1]) / 2, one-sided at the two ends.  Expected values are worked out by hand from the table
    below (dyadic numbers, so every step is exact): a wrong central difference (e.g. z[j+1] - z[j], or a missing / 2),
    a two-sided formula at the ends, or trunc_bins applied twice all fail."""
    z = np.array([0.5, 0.625, 1.0, 1.125, 2.0, 4.0], np.float32)
    #   spacings           one-sided 0.125 | (1.0-0.5)/2 | (1.125-0.625)/2 | (2-1)/2 | (4-1.125)/2 | one-sided 2.0
    local = np.array([0.125, 0.25, 0.25, 0.5, 1.4375, 2.0], np.float32)
    assert np.array_equal(oracle.tau_table(z, 2.0), 2.0 * local)
    assert np.array_equal(oracle.tau_table(z, 1.5), np.array([0.1875, 0.375, 0.375, 0.75, 2.15625, 3.0], np.float32))
    # trunc_metric > 0 overrides the spacing rule everywhere (tau = 0.02 m)
    assert np.array_equal(oracle.tau_table(z, 2.0, 0.02), np.full(6, np.float32(0.02)))
    # inverse-depth bins of C2-C5: 1/z uniform, so z[j+1] - z[j-1] = 2 d z[j+1] z[j-1] with d the inverse-depth step;
    # tau_j / (z[j+1] z[j-1]) must therefore be the constant 2 d in the interior (a one-sided difference z[j+1] - z[j]
    # would give d z[j+1] z[j] instead: off by the ratio z[j] / z[j-1], up to 7 % here)
    zi = synth.bins_inverse(0.5, 5.0, 64).astype(np.float64)
    tau = oracle.tau_table(zi.astype(np.float32), 2.0).astype(np.float64)
    d = (1.0 / 0.5 - 1.0 / 5.0) / 63
    # (the table is float32: the differences cancel ~5 bits, hence 2e-5; a wrong stencil is off by >= 1.4 %)
    assert np.allclose(tau[1:-1] / (zi[2:] * zi[:-2]), 2.0 * d, rtol=2e-5)
    assert np.isclose(tau[0], 2.0 * d * zi[0] * zi[1], rtol=2e-5) and np.isclose(tau[-1], 2.0 * d * zi[-1] * zi[-2], rtol=2e-5)


# ------------------------------------------------------------------------------------------------
# T8: behind-surface cut and clamp
# ------------------------------------------------------------------------------------------------
def test_T8_cut_and_clamp_sweep():
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 8, 8, 4, 4, 8, 8)
    tau_m = 0.25
    z = np.array([1.0, 1.75, 1.875, 2.0, 2.25, np.nextafter(np.float32(2.25), np.float32(3)), 3.0], np.float32)
    T, W, depth, conf, bn, tau = run_oracle(cam, z, [cam], const_maps([cam], 2.0), trunc_metric=tau_m)
    assert np.all(tau == np.float32(tau_m))
    t, w = T[27], W[27]
    assert t[0] == np.float32(tau_m) and w[0] == 1          # s = +1 saturates at +tau
    assert t[1] == np.float32(0.25) and t[2] == np.float32(0.125) and t[3] == 0.0
    assert t[4] == np.float32(-0.25) and w[4] == 1           # s = -tau exactly: kept
    assert t[5] == 0.0 and w[5] == 0 and w[6] == 0           # just below -tau: cut (omega_k = 0)
    assert np.all(bn == 2) and np.allclose(depth, 2.0, atol=1e-6)


# ------------------------------------------------------------------------------------------------
# T9: persistent running average
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("half", [False, True])
def test_T9_running_average_closed_form(half):
    rig = synth.grid_rig(32, 24)
    tgt = synth.camera_from_pose((0.0, 0.0, 0.0), np.eye(3), 24, 24, 16, 12, 32, 24)
    vi = synth.nearest_views(tgt, rig, 4)
    views = [rig[i] for i in vi]
    maps = const_maps(views, 2.0)
    z = synth.bins_uniform(1.0, 3.0, 9)                      # spacing 0.25 exactly
    tau = oracle.tau_table(z, 2.0)
    centre = np.array([12 * 32 + 16], np.int32)              # ray seen by all 4 views
    T = W = None
    for t in range(1, 25):
        T, W = oracle.integrate(tgt, z, tau, views, maps, rays=centre, T=T, Wt=W, accumulate=True,
                                decay=1.0, cap=64.0, half_storage=half)
        obs = z <= 2.0 + tau
        assert np.all(W[0][obs] == min(4 * t, 64))
        assert np.all(W[0][~obs] == 0)
        assert np.allclose(T[0][obs], np.clip(2.0 - z[obs], -tau[obs], tau[obs]), atol=1e-3 if half else 1e-6)
    # decay < 1: W -> V / (1 - gamma)
    T = W = None
    for t in range(200):
        T, W = oracle.integrate(tgt, z, tau, views, maps, rays=centre, T=T, Wt=W, accumulate=True,
                                decay=0.75, cap=1e9, half_storage=half)
    assert np.allclose(W[0][z <= 2.0 + tau], 4 / (1 - 0.75), rtol=2e-3 if half else 1e-5)
    # overwrite mode ignores history
    T2, W2 = oracle.integrate(tgt, z, tau, views, maps, rays=centre, T=T, Wt=W, accumulate=False)
    assert np.all(W2[0][z <= 2.0 + tau] == 4)


# ------------------------------------------------------------------------------------------------
# T10: extraction alone
# ------------------------------------------------------------------------------------------------
def test_T10_extract_synthetic_volume():
    z = synth.bins_inverse(0.5, 5, 40)
    tau = oracle.tau_table(z, 2.0)
    surf = np.array([0.7, 1.234, 2.5, 4.9, 0.5001], np.float64)
    T = np.clip(surf[:, None] - z[None, :].astype(np.float64), -tau, tau).astype(np.float32)
    W = np.ones_like(T)
    depth, conf, bn = oracle.extract(z, T, W)
    assert np.allclose(depth, surf, rtol=2e-6)
    for r, s in enumerate(surf):
        assert z[bn[r]] < s <= z[bn[r] + 1]
    assert np.all(conf == 1)
    # misses: all positive, all negative, zero weight at the crossing, gap across an unobserved bin
    Tm = np.stack([np.full(40, 0.1), np.full(40, -0.1), T[1], T[2]]).astype(np.float32)
    Wm = np.ones_like(Tm)
    Wm[2, bn[1] + 1] = 0
    Wm[3, bn[2]] = 0
    depth, conf, b2 = oracle.extract(z, Tm, Wm)
    assert np.all(b2 == -1) and np.all(depth == 0) and np.all(conf == 0)
    # first crossing wins; confidence interpolates W
    T2 = np.array([[0.2, 0.1, -0.1, 0.3, -0.3]], np.float32)
    W2 = np.array([[1, 2, 4, 1, 1]], np.float32)
    z2 = np.array([1, 2, 3, 4, 5], np.float32)
    depth, conf, b3 = oracle.extract(z2, T2, W2)
    assert b3[0] == 1 and abs(depth[0] - 2.5) < 1e-6 and abs(conf[0] - 3.0) < 1e-6
