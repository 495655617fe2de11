"""Pins of the oracle's raymarch (O-M, the paper's own schedule: PAPER.md:75, 348) against things other than itself
(-m "not gpu").  T11 closed-form scenes, T12 dense fp64 first-crossing brute force with explicit world points,
T13 coincident camera, T14 closed-form evaluation counts and miss cases."""
import math

import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth

TAU = 0.02
NEAR, FAR = 0.5, 5.0


def const_maps(cams, d, omega=1.0):
    out = []
    for c in cams:
        m = np.empty((c.height, c.width, 2), dtype=np.float32)
        m[..., 0] = d
        m[..., 1] = omega
        out.append(m)
    return out


def small_rig():
    rig = synth.grid_rig(96, 64)
    tgt = synth.camera_from_pose((0.03, -0.02, 0.0), np.eye(3), 72, 72, 48, 32, 96, 64)
    vi = synth.nearest_views(tgt, rig, 4)
    return tgt, [rig[i] for i in vi]


# ---- T11: closed-form scenes ---------------------------------------------------------------------------
@pytest.mark.parametrize("d", [0.9, 2.3456, 4.2])
def test_T11_frontoparallel_plane(d):
    """s(z) = d - z exactly (every view sees depth d), so the crossing is z = d; the final bracket is at most
    the last advance / 2^3 wide and the last advance is <= max(0.8 tau, min_step)."""
    tgt, views = small_rig()
    min_step = 1e-3
    depth, conf, steps = oracle.raymarch(tgt, views, const_maps(views, d), NEAR, FAR, tau=TAU, min_step=min_step)
    seen = depth > 0
    assert seen.mean() > 0.95
    # near the surface the advance is max(0.8 s, min_step) with s < tau: bracket <= 0.8 tau; after 3 halvings
    # the midpoint is within 0.8 tau / 16 of the crossing.  In practice the last advance is ~ min_step.
    assert np.max(np.abs(depth[seen] - d)) <= 0.8 * TAU / 16 + 1e-6
    assert np.median(np.abs(depth[seen] - d)) <= min_step / 8
    assert np.all(conf[seen] >= 1.0 - 1e-6) and np.all(conf[seen] <= 4.0 + 1e-6)
    assert np.all(depth[~seen] == 0) and np.all(conf[~seen] == 0)


def test_T11_sphere_scene_closed_form():
    """C1 (back plane + sphere), noise-free analytic inputs: the marched depth equals the closed-form ray-cast
    depth of the target view within tau on >= 99 % of interior pixels (tau is the band inside which the fused
    distance of several views may move the crossing)."""
    wl = synth.workload("C1", scale=1.0)
    tgt = wl.targets(0)[0]
    views = [wl.rig[i] for i in wl.views_for(tgt)]
    maps = [oracle.weight_map(synth.raycast(c, wl.scene)[0].astype(np.float32)) for c in views]
    depth, conf, steps = oracle.raymarch(tgt, views, maps, NEAR, 4.0, tau=TAU)
    gt = wl.true_depth(tgt, 0)
    depth = depth.reshape(gt.shape)
    edge = np.zeros_like(gt, dtype=bool)
    edge[:, 1:] |= np.abs(gt[:, 1:] - gt[:, :-1]) > 0.02 * gt[:, 1:]
    edge[1:, :] |= np.abs(gt[1:, :] - gt[:-1, :]) > 0.02 * gt[1:, :]
    near = edge.copy()
    for _ in range(4):
        g = near.copy()
        g[1:, :] |= near[:-1, :]; g[:-1, :] |= near[1:, :]; g[:, 1:] |= near[:, :-1]; g[:, :-1] |= near[:, 1:]
        near = g
    sel = ~near & (depth > 0)
    assert sel.mean() > 0.5
    err = np.abs(depth - gt)[sel]
    assert (err <= TAU).mean() >= 0.99, (err <= TAU).mean()
    assert np.median(err) < 0.25 * TAU


# ---- T12: dense fp64 brute force (explicit world points, no hoisting, no marching) ---------------------
def _s_fp64(target, views, maps, u, v, zs, tau):
    """Normalised Eq. 9-10 at target depths zs (array), restated in fp64 from PAPER.md:331-341 with explicit world
    points; NaN where unobserved."""
    zs = np.asarray(zs, dtype=np.float64)
    Kt = np.array([[target.fx, 0, target.cx], [0, target.fy, target.cy], [0, 0, 1]], dtype=np.float64)
    ray = np.linalg.inv(Kt) @ np.array([u + 0.5, v + 0.5, 1.0])
    p = (zs[:, None] * ray[None, :] - target.t.astype(np.float64)[None, :]) @ target.R.astype(np.float64)   # R^T (.)
    A = np.zeros_like(zs); Wn = np.zeros_like(zs)
    for cam, m in zip(views, maps):
        Kk = np.array([[cam.fx, 0, cam.cx], [0, cam.fy, cam.cy], [0, 0, 1]], dtype=np.float64)
        q = (p @ cam.R.astype(np.float64).T + cam.t.astype(np.float64)[None, :]) @ Kk.T
        x, y, w = q[:, 0], q[:, 1], q[:, 2]
        ok = w >= 1e-6
        ws = np.where(ok, w, 1.0)
        ix = np.floor(x / ws).astype(np.int64); iy = np.floor(y / ws).astype(np.int64)
        ok &= (ix >= 0) & (iy >= 0) & (ix < cam.width) & (iy < cam.height)
        ixc, iyc = np.clip(ix, 0, cam.width - 1), np.clip(iy, 0, cam.height - 1)
        Dk = m[iyc, ixc, 0].astype(np.float64); om = m[iyc, ixc, 1].astype(np.float64)
        sk = Dk - w
        ok &= (Dk > 0) & ~(sk < -tau)
        A += np.where(ok, om * np.minimum(sk, tau), 0.0); Wn += np.where(ok, om, 0.0)
    return np.where(Wn > 0, A / np.where(Wn > 0, Wn, 1.0), np.nan)


def _crossings(zs, sv):
    """Midpoints of consecutive observed samples with s > 0 followed by s <= 0."""
    i = np.nonzero((sv[:-1] > 0) & (sv[1:] <= 0))[0]
    return 0.5 * (zs[i] + zs[i + 1])


def test_T12_crossing_against_dense_fp64_scan():
    """On a tiny noisy scene the reported depth must be a genuine change of sign of the fp64 s(z) (a 2 um scan of
    +-(final bracket) around it finds + followed by <= 0), and it must be the FRONT-MOST one: a 0.1 mm scan of the
    whole ray has no crossing wider than the march can resolve in front of it."""
    wl = synth.workload("C1", scale=0.25)       # 16 x 12
    tgt = wl.targets(0)[0]
    views = [wl.rig[i] for i in wl.views_for(tgt)]
    maps = [oracle.weight_map(wl.view_inputs(0, i)[0]) for i in wl.views_for(tgt)]
    min_step = 1e-3
    depth, conf, steps = oracle.raymarch(tgt, views, maps, NEAR, 4.0, tau=TAU, min_step=min_step)
    half = 0.8 * TAU / 16 + 2e-5                # midpoint of a bracket <= 0.8 tau / 8 wide, + fp32 slack
    zs = np.arange(NEAR, 4.0, 1e-4)
    n_hit = n_first = 0
    rays = np.arange(0, tgt.width * tgt.height, 5)
    for r in rays:
        u, v = r % tgt.width, r // tgt.width
        sv = _s_fp64(tgt, views, maps, u, v, zs, TAU)
        coarse = _crossings(zs, sv)
        if depth[r] > 0:
            n_hit += 1
            zf = np.arange(depth[r] - half, depth[r] + half, 2e-6)
            fine = _crossings(zf, _s_fp64(tgt, views, maps, u, v, zf, TAU))
            assert fine.size > 0, "no change of sign of s near the reported depth (ray %d, %.6f)" % (r, depth[r])
            n_first += not np.any(coarse < depth[r] - half - 1e-4)
        else:
            # a miss may only have stepped over slivers: runs of s <= 0 shorter than the largest advance 0.8 tau
            # (nearest-pixel sampling of noisy maps makes s jump when the sampled pixel changes)
            for c in coarse:
                i = int(np.searchsorted(zs, c))
                run = 0
                while i + run < zs.size and sv[i + run] <= 0:
                    run += 1
                assert run * 1e-4 < 0.8 * TAU, (r, c, run)
    assert n_hit > 0.9 * rays.size
    # a crossing in front of the reported one can only be a sliver thinner than the march's advance (a few noisy
    # pixels); everywhere else the front-most surface is found
    assert n_first >= 0.95 * n_hit, (n_first, n_hit)


# ---- T13: coincident camera ----------------------------------------------------------------------------
def test_T13_coincident_camera_reproduces_its_depth():
    wl = synth.workload("C2", scale=0.1)
    cam = wl.rig[5]
    d = synth.noisy_depth(synth.raycast(cam, wl.scene)[0], 5, 0, 0.01, 0.02)
    m = oracle.weight_map(d)
    depth, conf, steps = oracle.raymarch(cam, [cam], [m], NEAR, FAR, tau=TAU, min_step=5e-4)
    depth = depth.reshape(d.shape)
    ok = (d > NEAR + TAU) & (d < FAR)
    # single view, same pixel: s(z) = D - z, crossing at D; bracket <= last advance / 8, midpoint within / 16
    assert np.all(depth[ok] > 0)
    assert np.max(np.abs(depth[ok] - d[ok])) <= 0.8 * TAU / 16 + 1e-6
    assert np.all(depth[d <= 0] == 0)
    assert np.allclose(conf.reshape(d.shape)[ok], m[..., 1][ok])


# ---- T14: evaluation counts and misses (1-D closed forms) ----------------------------------------------
def _march_1d(d, near, far, tau, scale, min_step, max_evals, n_bisect):
    """The march on the 1-D profile s(z) = min(d - z, tau) (one coincident view, omega = 1, plane at depth d),
    in fp32: free-space advances of scale * tau, a geometric approach inside the band, min_step at the end."""
    f = np.float32
    z, n, za = f(near), 0, None
    while n < max_evals and not z > f(far):
        s = min(f(d) - z, f(tau)); n += 1
        if s > 0:
            za = z; z = z + max(f(scale) * s, f(min_step))
        else:
            zb = z
            for _ in range(n_bisect):
                m = f(0.5) * (za + zb); n += 1
                if f(d) - m > 0: za = m
                else: zb = m
            return f(0.5) * (za + zb), n
    return f(0), n


@pytest.mark.parametrize("d,min_step", [(1.0, 1e-3), (2.71828, 1e-3), (4.9, 5e-4), (0.52, 2e-3)])
def test_T14_evaluation_count_and_depth_closed_form(d, min_step):
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 8, 6, 16, 12)
    depth, conf, steps = oracle.raymarch(cam, [cam], const_maps([cam], d), NEAR, FAR, tau=TAU, min_step=min_step)
    ed, en = _march_1d(d, NEAR, FAR, TAU, 0.8, min_step, 4096, 3)
    assert np.all(steps == en), (steps[:4], en)
    assert np.all(depth == ed)
    assert np.all(conf == 1.0)
    # orders of magnitude: (d - near - tau) / (0.8 tau) free-space advances, then ~log_5 + a few min_steps
    assert en >= (d - NEAR - TAU) / (0.8 * TAU)


def test_T14_misses():
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 8, 6, 16, 12)
    # nothing observed: free-space advances of 0.8 tau until z > z_far
    m = const_maps([cam], 0.0, 0.0)
    depth, conf, steps = oracle.raymarch(cam, [cam], m, NEAR, FAR, tau=TAU)
    z, n = np.float32(NEAR), 0
    while not z > np.float32(FAR):
        z = z + np.float32(0.8) * np.float32(TAU); n += 1
    assert np.all(depth == 0) and np.all(conf == 0) and np.all(steps == n)
    # surface beyond z_far: all positive, never crosses
    depth, conf, steps = oracle.raymarch(cam, [cam], const_maps([cam], 7.0), NEAR, FAR, tau=TAU)
    assert np.all(depth == 0) and np.all(steps == n)
    # evaluation budget
    depth, conf, steps = oracle.raymarch(cam, [cam], const_maps([cam], 4.0), NEAR, FAR, tau=TAU, max_evals=50)
    assert np.all(depth == 0) and np.all(steps == 50)
    # surface in front of z_near: first sample already <= 0, no positive predecessor -> creeps by min_step
    # through the band, then is cut (unobserved) to the end: a miss (M4)
    depth, conf, steps = oracle.raymarch(cam, [cam], const_maps([cam], 0.45), NEAR, FAR, tau=TAU)
    assert np.all(depth == 0)
    # view order does not change the front-most surface on a plane
    tgt, views = small_rig()
    a = oracle.raymarch(tgt, views, const_maps(views, 2.0), NEAR, FAR, tau=TAU)[0]
    b = oracle.raymarch(tgt, views[::-1], const_maps(views, 2.0), NEAR, FAR, tau=TAU)[0]
    assert np.max(np.abs(a - b)) <= 1e-5


def test_defaults_are_the_papers_constants():
    """The defaults of the oracle's raymarch / temporal weight and of the binding are the constants the paper prints
    (tests/golden/paper_constants.txt, each with its citation)."""
    import inspect
    import os
    from paper_2505_18932_b200 import binding
    gold = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if len(line) == 2:
                gold[line[0]] = float(line[1])
    o = inspect.signature(oracle.raymarch).parameters
    b = inspect.signature(binding.Context.ggt_raymarch_depth).parameters
    for sig in (o, b):
        assert sig["tau"].default == gold["tau_metric"]
        assert sig["step_scale"].default == gold["step_scale"]
        assert sig["n_bisect"].default == gold["n_bisect"]
    assert b["w_window"].default == gold["w_window"] and b["w_sigma0"].default == gold["w_sigma0"]
    assert b["w_clip"].default == gold["tau_metric"]          # Eq. 12's clip is the paper's tau
    assert inspect.signature(oracle.temporal_weight).parameters["eta"].default == gold["eta"]
    assert inspect.signature(binding.Context.ggt_temporal_weight).parameters["eta"].default == gold["eta"]
