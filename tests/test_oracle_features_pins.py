"""Pins of the oracle's network-input geometry features (O-F: PAPER.md:374-388, A.4 items 5-8) against closed forms
in fp64 (-m "not gpu"): T19 planes (normals exact, incl. one-sided differences at borders and holes), T20 sphere,
T21 the per-pixel dot products and the constant maps from explicit geometry, T22 undefined pixels."""
import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth


def cam_rays(cam):
    u = (np.arange(cam.width) + 0.5 - cam.cx) / cam.fx
    v = (np.arange(cam.height) + 0.5 - cam.cy) / cam.fy
    return np.stack(np.broadcast_arrays(u[None, :], v[:, None], np.ones((cam.height, cam.width))), axis=-1)   # z = 1


def plane_depth(cam, n, c):
    """z-depth of the plane n . X = c (camera coordinates) along every pixel ray."""
    return (c / (cam_rays(cam) @ np.asarray(n, dtype=np.float64))).astype(np.float32)


def centre(cam):
    return -np.asarray(cam.R, dtype=np.float64).T @ np.asarray(cam.t, dtype=np.float64)


def expected(cam, depth, normal_cam, views):
    """Items 5-8 in fp64 from explicit geometry, given the true camera-space unit normal per pixel (towards the camera)."""
    R, t = np.asarray(cam.R, np.float64), np.asarray(cam.t, np.float64)
    p = cam_rays(cam) * depth.astype(np.float64)[..., None]
    P = (p - t) @ R                      # R^T (p - t), row vectors
    n = normal_cam @ R
    rt = P - centre(cam); rt /= np.linalg.norm(rt, axis=-1, keepdims=True)
    K = len(views)
    out = np.zeros((4 * K,) + depth.shape)
    for k, vw in enumerate(views):
        rk = P - centre(vw); rk /= np.linalg.norm(rk, axis=-1, keepdims=True)
        out[k] = np.sum(rk * n, axis=-1)
        out[K + k] = np.sum(rk * rt, axis=-1)
        out[2 * K + k] = np.linalg.norm(centre(vw) - centre(cam))
        out[3 * K + k] = np.asarray(vw.R, np.float64)[2] @ R[2]
    return out


def setup(W=48, H=32):
    rig = synth.grid_rig(W, H)
    tgt = synth.camera_from_pose((0.03, -0.02, 0.05), synth.rot_yaw_pitch(0.05, -0.03), 40, 42, W / 2 + 1.5, H / 2 - 0.5, W, H)
    return tgt, [rig[i] for i in synth.nearest_views(tgt, rig, 4)]


# ---- T19: planes -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [(0.0, 0.0, 1.0), (0.3, -0.2, 1.0), (-0.5, 0.4, 0.8)])
def test_T19_plane_normals_and_features(n):
    tgt, views = setup()
    n = np.asarray(n) / np.linalg.norm(n)
    d = plane_depth(tgt, n, 2.5)
    f = oracle.features(tgt, d, views)
    ncam = np.broadcast_to(-n, d.shape + (3,))           # towards the camera: n_c . p < 0 since n . p = c > 0
    e = expected(tgt, d, ncam, views)
    # differences of points that lie on a plane are in the plane: the estimate is the plane's normal up to rounding of
    # the fp32 depths (relative 6e-8 on ~2.5 m against pixel footprints of ~6 cm: a few 1e-5 in the normal)
    assert np.max(np.abs(f - e)) < 2e-4
    # holes: a pixel whose neighbours are missing uses the one-sided differences and still gets the plane's normal
    d2 = d.copy()
    d2[10, 20] = 0; d2[11, 22] = 0; d2[15, 5:8] = 0
    f2 = oracle.features(tgt, d2, views)
    ok = d2 > 0
    assert np.max(np.abs(f2 - e)[:, ok]) < 2e-4
    assert np.all(f2[:8, ~ok] == 0)                       # no depth: items 5 and 6 are 0
    assert np.allclose(f2[8:, ~ok], e[8:, ~ok], atol=1e-6)   # the constant maps are constant


# ---- T20: sphere -------------------------------------------------------------------------------------------
def test_T20_sphere_normals():
    tgt, views = setup(96, 64)
    c, r = np.array([0.1, -0.05, 2.0]), 0.6              # sphere in camera coordinates
    rays = cam_rays(tgt)
    a = np.sum(rays * rays, -1); b = rays @ c; disc = b * b - a * (c @ c - r * r)
    hit = disc > 0
    z = np.where(hit, (b - np.sqrt(np.maximum(disc, 0))) / a, 0.0).astype(np.float32)
    f = oracle.features(tgt, z, views)
    p = rays * z.astype(np.float64)[..., None]
    ncam = (p - c) / r
    e = expected(tgt, z, ncam, views)
    # interior: all four neighbours on the sphere and away from the silhouette (finite differences: O(h^2) there)
    inter = hit.copy()
    inter[1:, :] &= hit[:-1, :]; inter[:-1, :] &= hit[1:, :]; inter[:, 1:] &= hit[:, :-1]; inter[:, :-1] &= hit[:, 1:]
    inter &= (-np.sum(ncam * p, -1) / np.linalg.norm(p, axis=-1)) > 0.5
    assert inter.sum() > 300
    assert np.max(np.abs(f[:4] - e[:4])[:, inter]) < 2e-2       # item 5 follows the analytic normal
    assert np.median(np.abs(f[:4] - e[:4])[:, inter]) < 2e-3
    assert np.max(np.abs(f[4:] - e[4:])[:, hit]) < 1e-5         # items 6-8 do not involve the normal


# ---- T21: values that need no surface model ----------------------------------------------------------------
def test_T21_constant_maps_and_ray_dots():
    wl = synth.workload("C2", scale=0.1)
    tgt = synth.camera_from_pose((0.05, 0.02, -0.03), synth.rot_yaw_pitch(0.03, -0.02), 50, 50, 32, 18, 64, 36)
    views = [wl.rig[i] for i in synth.nearest_views(tgt, wl.rig, 6)]
    d = synth.raycast(tgt, wl.scene)[0].astype(np.float32)
    f = oracle.features(tgt, d, views)
    K = len(views)
    e = expected(tgt, d, np.zeros(d.shape + (3,)), views)
    assert np.max(np.abs(f[2 * K:] - e[2 * K:])) < 1e-6
    defined = np.any(f[:K] != 0, axis=0)
    assert defined.mean() > 0.9
    assert np.max(np.abs(f[K:2 * K] - e[K:2 * K])[:, defined]) < 1e-5
    assert np.all(np.abs(f[:2 * K]) <= 1.0 + 1e-6)
    # the target's own camera as an input view: its ray IS the target view direction, and the normal faces it
    g = oracle.features(tgt, d, [tgt])
    assert np.max(np.abs(g[1] - 1.0)[defined]) < 1e-6 and np.all(g[0][defined] < 0) and np.all(g[2] == 0)
    assert np.max(np.abs(g[3] - 1.0)) < 1e-6


# ---- T22: undefined pixels ---------------------------------------------------------------------------------
def test_T22_undefined_pixels_are_zero():
    tgt, views = setup(16, 12)
    d = np.zeros((12, 16), np.float32)
    d[5, 7] = 2.0                                            # isolated: no neighbour in either axis
    d[2, 2:5] = 2.0                                          # a row segment: no vertical neighbour
    f = oracle.features(tgt, d, views)
    assert np.all(f[:8] == 0)
    d[3, 2:5] = 2.0                                          # now rows 2-3 x cols 2-4 have both
    f = oracle.features(tgt, d, views)
    assert np.all(f[0][2:4, 2:5] != 0) and f[0][5, 7] == 0
