"""CPU oracle of the geometry-guidance hot path — TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
The arithmetic lives in ggt_oracle.cpp (plain single-threaded C++, written from PAPER.md); this file
only compiles it with g++ and marshals numpy arrays.  It imports nothing from the CUDA package
except never: the two sides share no code.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ggt_oracle.cpp")
_SRCS = [_SRC, os.path.join(_HERE, "ggt_oracle_splat.cpp")]
_LIB = os.path.join(_HERE, "libggt_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2, contraction off, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
                               "-o", tmp] + _SRCS)
        os.replace(tmp, _LIB)
    return _LIB


class OrcCamera(ctypes.Structure):
    _fields_ = [("fx", ctypes.c_float), ("fy", ctypes.c_float), ("cx", ctypes.c_float),
                ("cy", ctypes.c_float), ("R", ctypes.c_float * 9), ("t", ctypes.c_float * 3),
                ("width", ctypes.c_int32), ("height", ctypes.c_int32)]


def _cam(c) -> OrcCamera:
    o = OrcCamera()
    o.fx, o.fy, o.cx, o.cy = c.fx, c.fy, c.cx, c.cy
    o.R[:] = [float(x) for x in np.asarray(c.R, dtype=np.float32).reshape(9)]
    o.t[:] = [float(x) for x in np.asarray(c.t, dtype=np.float32).reshape(3)]
    o.width, o.height = int(c.width), int(c.height)
    return o


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_round_f16.restype = ctypes.c_float
        _lib.orc_round_f16.argtypes = [ctypes.c_float]
        _lib.orc_exp_le0.restype = ctypes.c_float
        _lib.orc_exp_le0.argtypes = [ctypes.c_float]
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(ctypes.POINTER(ty)) if a is not None else None


def round_f16(x: float) -> float:
    return float(_load().orc_round_f16(ctypes.c_float(x)))


def refine(rgb_cur, rgb_prev, depth_cur, depth_state, lambda_t=0.7, beta=0.6, theta=0.0,
           downscale=4, pool=3, want_mask=True):
    """O-R. Returns (refined depth, mask or None, pooled uint16 or None, binary uint8 or None)."""
    lib = _load()
    H, W = depth_cur.shape
    depth_cur = np.ascontiguousarray(depth_cur, dtype=np.float32)
    state = np.array(depth_state, dtype=np.float32, order="C", copy=True)
    mask = np.empty((H, W), dtype=np.float32) if want_mask else None
    pooled = binary = None
    stride = 3
    if rgb_prev is not None:
        rgb_cur = np.ascontiguousarray(rgb_cur, dtype=np.uint8)
        rgb_prev = np.ascontiguousarray(rgb_prev, dtype=np.uint8)
        stride = rgb_cur.shape[2]
        Hq, Wq = -(-H // downscale), -(-W // downscale)
        pooled = np.empty((Hq, Wq), dtype=np.uint16)
        binary = np.empty((Hq, Wq), dtype=np.uint8)
    rc = lib.orc_refine(ctypes.c_int32(W), ctypes.c_int32(H), _p(rgb_cur, ctypes.c_uint8),
                        _p(rgb_prev, ctypes.c_uint8), ctypes.c_int32(stride),
                        _p(depth_cur, ctypes.c_float), _p(state, ctypes.c_float), _p(mask, ctypes.c_float),
                        _p(pooled, ctypes.c_uint16), _p(binary, ctypes.c_uint8),
                        ctypes.c_float(lambda_t), ctypes.c_float(beta), ctypes.c_float(theta),
                        ctypes.c_int32(downscale), ctypes.c_int32(pool))
    if rc != 0:
        raise ValueError("orc_refine rc=%d" % rc)
    return state, mask, pooled, binary


def weight_map(depth, sigma0=0.001, clip=0.02, window=7) -> np.ndarray:
    """O-W. Returns (H, W, 2) float32 interleaved {depth, omega}."""
    lib = _load()
    depth = np.ascontiguousarray(depth, dtype=np.float32)
    H, W = depth.shape
    out = np.empty((H, W, 2), dtype=np.float32)
    rc = lib.orc_weight_map(ctypes.c_int32(W), ctypes.c_int32(H), _p(depth, ctypes.c_float),
                            _p(out, ctypes.c_float), ctypes.c_float(sigma0), ctypes.c_float(clip),
                            ctypes.c_int32(window))
    if rc != 0:
        raise ValueError("orc_weight_map rc=%d" % rc)
    return out


def tau_table(z_bins, trunc_bins=2.0, trunc_metric=0.0) -> np.ndarray:
    lib = _load()
    z = np.ascontiguousarray(z_bins, dtype=np.float32)
    tau = np.empty_like(z)
    rc = lib.orc_tau_table(ctypes.c_int32(z.size), _p(z, ctypes.c_float), ctypes.c_float(trunc_bins),
                           ctypes.c_float(trunc_metric), _p(tau, ctypes.c_float))
    if rc != 0:
        raise ValueError("orc_tau_table rc=%d" % rc)
    return tau


def relative(target, view):
    lib = _load()
    Hm = np.empty(9, dtype=np.float32)
    e = np.empty(3, dtype=np.float32)
    t, v = _cam(target), _cam(view)
    lib.orc_relative(ctypes.byref(t), ctypes.byref(v), _p(Hm, ctypes.c_float), _p(e, ctypes.c_float))
    return Hm.reshape(3, 3), e


def integrate(target, z_bins, tau, views: Sequence, maps: Sequence[np.ndarray],
              rays: Optional[np.ndarray] = None, T: Optional[np.ndarray] = None,
              Wt: Optional[np.ndarray] = None, accumulate=False, decay=1.0, cap=64.0,
              half_storage=False):
    """O-I. Returns (T, W) arrays of shape (n_rays, D); n_rays = H_t*W_t when rays is None."""
    lib = _load()
    z = np.ascontiguousarray(z_bins, dtype=np.float32)
    tau = np.ascontiguousarray(tau, dtype=np.float32)
    D = z.size
    n_rays = int(target.width) * int(target.height) if rays is None else int(rays.size)
    if rays is not None:
        rays = np.ascontiguousarray(rays, dtype=np.int32)
    if T is None:
        T = np.zeros((n_rays, D), dtype=np.float32)
        Wt = np.zeros((n_rays, D), dtype=np.float32)
    else:
        T = np.array(T, dtype=np.float32, order="C", copy=True).reshape(n_rays, D)
        Wt = np.array(Wt, dtype=np.float32, order="C", copy=True).reshape(n_rays, D)
    V = len(views)
    cams = (OrcCamera * max(V, 1))(*[_cam(c) for c in views])
    maps = [np.ascontiguousarray(m, dtype=np.float32) for m in maps]
    ptrs = (ctypes.POINTER(ctypes.c_float) * max(V, 1))(*[_p(m, ctypes.c_float) for m in maps])
    t = _cam(target)
    rc = lib.orc_integrate(ctypes.byref(t), ctypes.c_int32(D), _p(z, ctypes.c_float), _p(tau, ctypes.c_float),
                           ctypes.c_int32(V), cams, ptrs, ctypes.c_int64(n_rays), _p(rays, ctypes.c_int32),
                           _p(T, ctypes.c_float), _p(Wt, ctypes.c_float), ctypes.c_int32(int(accumulate)),
                           ctypes.c_float(decay), ctypes.c_float(cap), ctypes.c_int32(int(half_storage)))
    if rc != 0:
        raise ValueError("orc_integrate rc=%d" % rc)
    return T, Wt


def extract(z_bins, T, Wt):
    """O-E. Returns (depth, conf, bin) per ray."""
    lib = _load()
    z = np.ascontiguousarray(z_bins, dtype=np.float32)
    T = np.ascontiguousarray(T, dtype=np.float32)
    Wt = np.ascontiguousarray(Wt, dtype=np.float32)
    n_rays, D = T.shape
    depth = np.empty(n_rays, dtype=np.float32)
    conf = np.empty(n_rays, dtype=np.float32)
    bins = np.empty(n_rays, dtype=np.int32)
    lib.orc_extract(ctypes.c_int64(n_rays), ctypes.c_int32(D), _p(z, ctypes.c_float), _p(T, ctypes.c_float),
                    _p(Wt, ctypes.c_float), _p(depth, ctypes.c_float), _p(conf, ctypes.c_float),
                    _p(bins, ctypes.c_int32))
    return depth, conf, bins


def raymarch(target, views: Sequence, maps: Sequence[np.ndarray], z_near, z_far, tau=0.02, step_scale=0.8,
             min_step=1e-3, max_evals=4096, n_bisect=3, rays: Optional[np.ndarray] = None):
    """O-M (the paper's own schedule). Returns (depth, conf, steps) per ray."""
    lib = _load()
    n_rays = int(target.width) * int(target.height) if rays is None else int(rays.size)
    if rays is not None:
        rays = np.ascontiguousarray(rays, dtype=np.int32)
    V = len(views)
    cams = (OrcCamera * max(V, 1))(*[_cam(c) for c in views])
    maps = [np.ascontiguousarray(m, dtype=np.float32) for m in maps]
    ptrs = (ctypes.POINTER(ctypes.c_float) * max(V, 1))(*[_p(m, ctypes.c_float) for m in maps])
    depth = np.empty(n_rays, dtype=np.float32)
    conf = np.empty(n_rays, dtype=np.float32)
    steps = np.empty(n_rays, dtype=np.int32)
    t = _cam(target)
    rc = lib.orc_raymarch(ctypes.byref(t), ctypes.c_int32(V), cams, ptrs, ctypes.c_int64(n_rays),
                          _p(rays, ctypes.c_int32), ctypes.c_float(z_near), ctypes.c_float(z_far),
                          ctypes.c_float(tau), ctypes.c_float(step_scale), ctypes.c_float(min_step),
                          ctypes.c_int32(max_evals), ctypes.c_int32(n_bisect), _p(depth, ctypes.c_float),
                          _p(conf, ctypes.c_float), _p(steps, ctypes.c_int32))
    if rc != 0:
        raise ValueError("orc_raymarch rc=%d" % rc)
    return depth, conf, steps


def temporal_weight(prev_cam, prev_depth, prev_conf, views: Sequence, masks: Sequence[np.ndarray], beta=1.0, eta=15.0):
    """O-T (Eq. 13-14). Returns the fp32 weight map of the previous output depth, shape of prev_depth."""
    lib = _load()
    H, W = int(prev_cam.height), int(prev_cam.width)
    d = np.ascontiguousarray(prev_depth, dtype=np.float32).reshape(H, W)
    c = np.ascontiguousarray(prev_conf, dtype=np.float32).reshape(H, W)
    V = len(views)
    cams = (OrcCamera * max(V, 1))(*[_cam(v) for v in views])
    masks = [np.ascontiguousarray(m, dtype=np.float32) for m in masks]
    ptrs = (ctypes.POINTER(ctypes.c_float) * max(V, 1))(*[_p(m, ctypes.c_float) for m in masks])
    out = np.empty((H, W), dtype=np.float32)
    t = _cam(prev_cam)
    rc = lib.orc_temporal_weight(ctypes.byref(t), _p(d, ctypes.c_float), _p(c, ctypes.c_float), ctypes.c_int32(V),
                                 cams, ptrs, ctypes.c_float(beta), ctypes.c_float(eta), _p(out, ctypes.c_float))
    if rc != 0:
        raise ValueError("orc_temporal_weight rc=%d" % rc)
    return out


def view_record(depth, weight) -> np.ndarray:
    """Interleaved {depth, omega} map of a view whose weights are given (e.g. temporal_weight) instead of Eq. 11-12."""
    depth = np.asarray(depth, dtype=np.float32)
    out = np.zeros(depth.shape + (2,), dtype=np.float32)
    ok = depth > 0
    out[..., 0] = depth
    out[..., 1] = np.where(ok, np.asarray(weight, dtype=np.float32).reshape(depth.shape), 0)
    return out


def features(target, depth, views: Sequence) -> np.ndarray:
    """O-F (PAPER.md:374-388 items 5-8). Returns (4 K, H, W) float32."""
    lib = _load()
    H, W = int(target.height), int(target.width)
    d = np.ascontiguousarray(depth, dtype=np.float32).reshape(H, W)
    V = len(views)
    cams = (OrcCamera * max(V, 1))(*[_cam(v) for v in views])
    out = np.empty((4 * V, H, W), dtype=np.float32)
    t = _cam(target)
    rc = lib.orc_features(ctypes.byref(t), _p(d, ctypes.c_float), ctypes.c_int32(V), cams, _p(out, ctypes.c_float))
    if rc != 0:
        raise ValueError("orc_features rc=%d" % rc)
    return out


# ---- f-3: forward warping with pixel-sized 3D Gaussians (ggt_oracle_splat.cpp) ---------------------------------------
def exp_le0(q: float) -> float:
    """The fp32 exponential both implementations use for alpha (reading S8), q <= 0."""
    return float(_load().orc_exp_le0(ctypes.c_float(q)))


def splat_project(target, view, u, v, D, sigma_px=0.5, dilation=0.3, z_cull=0.2):
    """One Gaussian: (mu_x, mu_y, z, conic a, b, c, radius) or None if it is culled (readings S1-S3, S7)."""
    lib = _load()
    out = np.zeros(7, dtype=np.float32)
    t, vw = _cam(target), _cam(view)
    ok = lib.orc_splat_project(ctypes.byref(t), ctypes.byref(vw), ctypes.c_int32(int(u)), ctypes.c_int32(int(v)),
                               ctypes.c_float(D), ctypes.c_float(sigma_px), ctypes.c_float(dilation),
                               ctypes.c_float(z_cull), _p(out, ctypes.c_float))
    return out if ok else None


def splat_forward(target, view, depth, rgb=None, mask=None, sigma_px=0.5, dilation=0.3, z_cull=0.2):
    """O-S. Returns dict(rgb (3,Ht,Wt) or None, alpha, depth, mask or None, count) of one view splatted into `target`."""
    lib = _load()
    H, W = int(view.height), int(view.width)
    Ht, Wt = int(target.height), int(target.width)
    depth = np.ascontiguousarray(depth, dtype=np.float32).reshape(H, W)
    stride = 3
    if rgb is not None:
        rgb = np.ascontiguousarray(rgb, dtype=np.uint8)
        stride = rgb.shape[2]
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.float32).reshape(H, W)
    o_rgb = np.empty((3, Ht, Wt), dtype=np.float32) if rgb is not None else None
    o_alpha = np.empty((Ht, Wt), dtype=np.float32)
    o_depth = np.empty((Ht, Wt), dtype=np.float32)
    o_mask = np.empty((Ht, Wt), dtype=np.float32) if mask is not None else None
    o_count = np.empty((Ht, Wt), dtype=np.int32)
    t, vw = _cam(target), _cam(view)
    rc = lib.orc_splat_forward(ctypes.byref(t), ctypes.byref(vw), _p(depth, ctypes.c_float), _p(rgb, ctypes.c_uint8),
                               ctypes.c_int32(stride), _p(mask, ctypes.c_float), ctypes.c_float(sigma_px),
                               ctypes.c_float(dilation), ctypes.c_float(z_cull), _p(o_rgb, ctypes.c_float),
                               _p(o_alpha, ctypes.c_float), _p(o_depth, ctypes.c_float), _p(o_mask, ctypes.c_float),
                               _p(o_count, ctypes.c_int32))
    if rc != 0:
        raise ValueError("orc_splat_forward rc=%d" % rc)
    return dict(rgb=o_rgb, alpha=o_alpha, depth=o_depth, mask=o_mask, count=o_count)


def temporal_weight_mask(prev_depth, prev_conf, novel_mask, beta=1.0, eta=15.0):
    """Eq. 13 with a given novel-view mask M^t (the paper's splat-and-max), per pixel of D^{t-1}."""
    lib = _load()
    d = np.ascontiguousarray(prev_depth, dtype=np.float32)
    c = np.ascontiguousarray(prev_conf, dtype=np.float32).reshape(d.shape)
    m = np.ascontiguousarray(novel_mask, dtype=np.float32).reshape(d.shape)
    out = np.empty_like(d)
    lib.orc_temporal_weight_mask(ctypes.c_int64(d.size), _p(d, ctypes.c_float), _p(c, ctypes.c_float), _p(m, ctypes.c_float),
                                 ctypes.c_float(beta), ctypes.c_float(eta), _p(out, ctypes.c_float))
    return out
