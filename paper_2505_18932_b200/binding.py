"""Thin ctypes binding of the C ABI in include/ggt.h — argument marshalling only.

Every step of the path runs in the CUDA kernels of libggt.so; torch is used for device memory and
streams.  There is no fallback: if the library is missing or there is no CUDA device, calls raise.
Function names mirror the C entry points (ggt_refine_depth, ggt_integrate, ggt_extract_depth, ...).
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libggt.so")

GGT_OK = 0
GGT_F32, GGT_F16 = 0, 1
GGT_OVERWRITE, GGT_ACCUMULATE = 0, 1
GGT_FRAME_RESULTS_ASYNC = 0x100
GGT_MAX_VIEWS = 16
GGT_PROFILE_STAGES = 5

EXPORTS = [
    "ggt_create", "ggt_destroy", "ggt_last_error", "ggt_launch_count", "ggt_profile_enable", "ggt_profile_collect", "ggt_selftest_arith", "ggt_workspace_bytes", "ggt_set_workspace",
    "ggt_volume_bytes", "ggt_volume_bind", "ggt_volume_unbind", "ggt_volume_reset", "ggt_volume_export",
    "ggt_volume_tables", "ggt_refine_depth", "ggt_refine_depth_static", "ggt_refine_depth_batch", "ggt_integrate", "ggt_integrate_batch", "ggt_integrate_extract_batch", "ggt_extract_depth", "ggt_integrate_extract",
    "ggt_raymarch_depth", "ggt_guidance_features", "ggt_temporal_weight", "ggt_integrate_weighted", "ggt_raymarch_depth_weighted",
    "ggt_frame_staging_bytes", "ggt_frame_host", "ggt_frame_host_results_wait",
    "ggt_splat_forward", "ggt_splat_reserve", "ggt_splat_status", "ggt_temporal_weight_mask",
]


class GgtError(RuntimeError):
    pass


class ggt_camera(ctypes.Structure):
    _fields_ = [("fx", ctypes.c_float), ("fy", ctypes.c_float), ("cx", ctypes.c_float), ("cy", ctypes.c_float),
                ("R", ctypes.c_float * 9), ("t", ctypes.c_float * 3),
                ("width", ctypes.c_int32), ("height", ctypes.c_int32)]


class ggt_refine_params(ctypes.Structure):
    _fields_ = [("lambda_t", ctypes.c_float), ("beta", ctypes.c_float), ("theta", ctypes.c_float),
                ("downscale", ctypes.c_int32), ("pool", ctypes.c_int32)]


class ggt_raymarch_params(ctypes.Structure):
    _fields_ = [("z_near", ctypes.c_float), ("z_far", ctypes.c_float), ("tau", ctypes.c_float),
                ("step_scale", ctypes.c_float), ("min_step", ctypes.c_float), ("max_evals", ctypes.c_int32),
                ("n_bisect", ctypes.c_int32), ("w_sigma0", ctypes.c_float), ("w_clip", ctypes.c_float),
                ("w_window", ctypes.c_int32)]


class ggt_splat_params(ctypes.Structure):
    _fields_ = [("sigma_px", ctypes.c_float), ("dilation", ctypes.c_float), ("z_cull", ctypes.c_float),
                ("reserved", ctypes.c_int32)]


class ggt_volume_desc(ctypes.Structure):
    _fields_ = [("width", ctypes.c_int32), ("height", ctypes.c_int32), ("bins", ctypes.c_int32),
                ("z_bins", ctypes.POINTER(ctypes.c_float)), ("trunc_bins", ctypes.c_float),
                ("trunc_metric", ctypes.c_float), ("w_sigma0", ctypes.c_float), ("w_clip", ctypes.c_float),
                ("w_window", ctypes.c_int32), ("weight_cap", ctypes.c_float), ("decay", ctypes.c_float),
                ("dtype", ctypes.c_int32)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libggt.so (built in-tree by paper_2505_18932_b200/build.py) and declare signatures."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GgtError("libggt.so not found at %s: run `python -m paper_2505_18932_b200.build` "
                       "(there is no CPU fallback)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, u32, f32p = ctypes.c_void_p, ctypes.c_int32, ctypes.c_uint32, ctypes.POINTER(ctypes.c_float)
    camp, descp = ctypes.POINTER(ggt_camera), ctypes.POINTER(ggt_volume_desc)
    lib.ggt_create.argtypes = [ctypes.POINTER(vp)]
    lib.ggt_destroy.argtypes = [vp]
    lib.ggt_last_error.argtypes = [vp]
    lib.ggt_last_error.restype = ctypes.c_char_p
    lib.ggt_launch_count.argtypes = [vp]
    lib.ggt_launch_count.restype = ctypes.c_int64
    lib.ggt_profile_enable.argtypes = [vp, i32]
    lib.ggt_profile_collect.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)]
    lib.ggt_selftest_arith.argtypes = [vp, ctypes.c_int64, vp, vp, vp, vp]
    lib.ggt_workspace_bytes.argtypes = [i32, i32, i32]
    lib.ggt_workspace_bytes.restype = ctypes.c_size_t
    lib.ggt_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.ggt_volume_bytes.argtypes = [descp]
    lib.ggt_volume_bytes.restype = ctypes.c_size_t
    lib.ggt_volume_bind.argtypes = [vp, descp, vp, ctypes.c_size_t, ctypes.POINTER(vp)]
    lib.ggt_volume_unbind.argtypes = [vp, vp]
    lib.ggt_volume_reset.argtypes = [vp, vp, vp]
    lib.ggt_volume_export.argtypes = [vp, vp, vp, vp, vp]
    lib.ggt_volume_tables.argtypes = [vp, f32p, f32p]
    lib.ggt_refine_depth.argtypes = [vp, i32, i32, vp, vp, i32, vp, vp, vp, vp, ctypes.POINTER(ggt_refine_params), vp]
    lib.ggt_refine_depth_static.argtypes = lib.ggt_refine_depth.argtypes
    lib.ggt_integrate.argtypes = [vp, vp, camp, i32, camp, ctypes.POINTER(vp), u32, vp]
    lib.ggt_extract_depth.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.ggt_integrate_extract.argtypes = [vp, vp, camp, i32, camp, ctypes.POINTER(vp), u32, vp, vp, vp, vp]
    lib.ggt_raymarch_depth.argtypes = [vp, camp, i32, camp, ctypes.POINTER(vp), ctypes.POINTER(ggt_raymarch_params), vp, vp,
                                       vp, vp]
    lib.ggt_raymarch_depth_weighted.argtypes = [vp, camp, i32, camp, ctypes.POINTER(vp), ctypes.POINTER(vp),
                                                ctypes.POINTER(ggt_raymarch_params), vp, vp, vp, vp]
    lib.ggt_integrate_weighted.argtypes = [vp, vp, camp, i32, camp, ctypes.POINTER(vp), ctypes.POINTER(vp), u32, vp]
    lib.ggt_temporal_weight.argtypes = [vp, camp, vp, vp, i32, camp, ctypes.POINTER(vp), ctypes.c_float, ctypes.c_float,
                                        vp, vp]
    lib.ggt_guidance_features.argtypes = [vp, camp, vp, i32, camp, vp, vp]
    lib.ggt_refine_depth_batch.argtypes = [vp, i32, i32, i32, ctypes.POINTER(vp), ctypes.POINTER(vp), i32, ctypes.POINTER(vp),
                                           ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp),
                                           ctypes.POINTER(ggt_refine_params), vp]
    lib.ggt_integrate_batch.argtypes = [vp, i32, ctypes.POINTER(vp), camp, i32, camp, ctypes.POINTER(vp), i32,
                                        ctypes.POINTER(i32), u32, vp]
    lib.ggt_integrate_extract_batch.argtypes = [vp, i32, ctypes.POINTER(vp), camp, i32, camp, ctypes.POINTER(vp), i32,
                                                ctypes.POINTER(i32), u32, ctypes.POINTER(vp), ctypes.POINTER(vp),
                                                ctypes.POINTER(vp), vp]
    lib.ggt_splat_forward.argtypes = [vp, camp, camp, vp, vp, i32, vp, ctypes.POINTER(ggt_splat_params), vp, vp, vp, vp, vp, vp]
    lib.ggt_splat_reserve.argtypes = [vp, ctypes.c_int64]
    lib.ggt_splat_status.argtypes = [vp, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64), vp]
    lib.ggt_temporal_weight_mask.argtypes = [vp, ctypes.c_int64, vp, vp, i32, ctypes.POINTER(vp), ctypes.c_float, ctypes.c_float,
                                             vp, vp]
    lib.ggt_frame_staging_bytes.argtypes = [descp, i32, i32, i32, i32]
    lib.ggt_frame_staging_bytes.restype = ctypes.c_size_t
    lib.ggt_frame_host_results_wait.argtypes = [vp, vp]
    lib.ggt_frame_host.argtypes = [vp, vp, camp, i32, camp, ctypes.POINTER(vp), ctypes.POINTER(vp),
                                   ctypes.POINTER(i32), i32, ctypes.POINTER(u32),
                                   ctypes.POINTER(ggt_refine_params), u32, vp, ctypes.c_size_t, vp, vp, vp]
    _lib = lib
    return lib


def to_camera(c) -> ggt_camera:
    """Marshal any object with fx, fy, cx, cy, R (3x3), t (3), width, height."""
    o = ggt_camera()
    o.fx, o.fy, o.cx, o.cy = float(c.fx), float(c.fy), float(c.cx), float(c.cy)
    o.R[:] = [float(x) for x in np.asarray(c.R, dtype=np.float32).reshape(9)]
    o.t[:] = [float(x) for x in np.asarray(c.t, dtype=np.float32).reshape(3)]
    o.width, o.height = int(c.width), int(c.height)
    return o


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _chk(t, dtype, numel=None, what="tensor", cuda=True):
    """Marshalling guard: the C ABI takes raw pointers, so dtype / device / layout / size are checked here."""
    if t is None:
        return None
    import torch
    want = getattr(torch, dtype)
    if t.dtype != want:
        raise GgtError("%s: dtype %s, expected %s" % (what, t.dtype, want))
    if cuda and not t.is_cuda:
        raise GgtError("%s: must be a CUDA tensor" % what)
    if not cuda and (t.is_cuda or not t.is_pinned()):
        raise GgtError("%s: must be a pinned host tensor" % what)
    if not t.is_contiguous():
        raise GgtError("%s: must be contiguous" % what)
    if numel is not None and t.numel() != int(numel):
        raise GgtError("%s: %d elements, expected %d" % (what, t.numel(), int(numel)))
    return t


def _chk_views(views, tensors, dtype="float32", what="depth"):
    for k, (c, t) in enumerate(zip(views, tensors)):
        _chk(t, dtype, int(c.width) * int(c.height), "%s of view %d" % (what, k))


def _stream() -> int:
    import torch
    return torch.cuda.current_stream().cuda_stream


def _refine_params(lambda_t=0.7, beta=0.6, theta=0.0, downscale=4, pool=3) -> ggt_refine_params:
    return ggt_refine_params(lambda_t, beta, theta, downscale, pool)


class Context:
    """ggt_ctx: one per (device, stream of use).  Owns no frame state."""

    def __init__(self):
        import torch
        if not torch.cuda.is_available():
            raise GgtError("no CUDA device: the ggt library has no CPU path")
        self.lib = load_library()
        h = ctypes.c_void_p()
        rc = self.lib.ggt_create(ctypes.byref(h))
        if rc != GGT_OK:
            raise GgtError("ggt_create: %s" % self.lib.ggt_last_error(None).decode())
        self.h = h
        self._ws = None

    def check(self, rc: int, what: str):
        if rc != GGT_OK:
            raise GgtError("%s failed (%d): %s" % (what, rc, self.lib.ggt_last_error(self.h).decode()))

    def close(self):
        if getattr(self, "h", None):
            self.lib.ggt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launch_count(self) -> int:
        return int(self.lib.ggt_launch_count(self.h))

    def ggt_profile_enable(self, enable: bool):
        self.check(self.lib.ggt_profile_enable(self.h, int(enable)), "ggt_profile_enable")

    def ggt_profile_collect(self):
        """{stage: (total ms, groups)} for refine / weight / integrate / extract since the last collect."""
        ms = (ctypes.c_double * GGT_PROFILE_STAGES)()
        n = (ctypes.c_int64 * GGT_PROFILE_STAGES)()
        self.check(self.lib.ggt_profile_collect(self.h, ms, n), "ggt_profile_collect")
        return {k: (ms[i], int(n[i])) for i, k in enumerate(("refine", "weight", "integrate", "extract", "raymarch"))}

    def ggt_selftest_arith(self, a, b):
        """(reciprocal, division, sqrt, x/49) mismatch counts of the kernels' arithmetic vs IEEE on cuda tensors a, b."""
        import torch
        out = torch.zeros(4, dtype=torch.int32, device="cuda")
        self.check(self.lib.ggt_selftest_arith(self.h, a.numel(), a.data_ptr(), b.data_ptr(), out.data_ptr(), _stream()),
                   "ggt_selftest_arith")
        r = out.cpu().numpy()
        return int(r[0]), int(r[1]), int(r[2]), int(r[3])

    def ggt_set_workspace(self, n_views: int, width: int, height: int):
        import torch
        n = self.lib.ggt_workspace_bytes(n_views, width, height)
        self._ws = torch.empty(n, dtype=torch.uint8, device="cuda")
        self.check(self.lib.ggt_set_workspace(self.h, self._ws.data_ptr(), n), "ggt_set_workspace")

    # ---- a1-a2 -------------------------------------------------------------------------------------
    def ggt_refine_depth(self, rgb_cur, rgb_prev, depth_cur, depth_state, mask_out=None, pooled_out=None,
                         lambda_t=0.7, beta=0.6, theta=0.0, downscale=4, pool=3):
        """In-place update of `depth_state` (torch fp32 HxW, cuda).  rgb_*: torch uint8 HxWx{3,4} or None."""
        H, W = depth_cur.shape
        stride = 3 if rgb_cur is None else int(rgb_cur.shape[2])
        for t, nm in ((rgb_cur, "rgb_cur"), (rgb_prev, "rgb_prev")):
            _chk(t, "uint8", H * W * stride, nm)
        for t, nm in ((depth_cur, "depth_cur"), (depth_state, "depth_state"), (mask_out, "mask_out")):
            _chk(t, "float32", H * W, nm)
        _chk(pooled_out, "uint16", ((H + 3) // 4) * ((W + 3) // 4), "pooled_out")
        prm = _refine_params(lambda_t, beta, theta, downscale, pool)
        rc = self.lib.ggt_refine_depth(self.h, W, H, _ptr(rgb_cur), _ptr(rgb_prev), stride, _ptr(depth_cur),
                                       _ptr(depth_state), _ptr(mask_out), _ptr(pooled_out), ctypes.byref(prm),
                                       _stream())
        self.check(rc, "ggt_refine_depth")

    def ggt_refine_depth_static(self, rgb_cur, rgb_prev, depth_cur, depth_state, mask_out=None, pooled_out=None,
                                lambda_t=0.7, beta=0.6, theta=0.0, downscale=4, pool=3):
        """ggt_refine_depth without any device allocation: scratch in the library's fixed 512 KB device array."""
        H, W = depth_cur.shape
        stride = 3 if rgb_cur is None else int(rgb_cur.shape[2])
        for t, nm in ((rgb_cur, "rgb_cur"), (rgb_prev, "rgb_prev")):
            _chk(t, "uint8", H * W * stride, nm)
        for t, nm in ((depth_cur, "depth_cur"), (depth_state, "depth_state"), (mask_out, "mask_out")):
            _chk(t, "float32", H * W, nm)
        _chk(pooled_out, "uint16", ((H + 3) // 4) * ((W + 3) // 4), "pooled_out")
        prm = _refine_params(lambda_t, beta, theta, downscale, pool)
        rc = self.lib.ggt_refine_depth_static(self.h, W, H, _ptr(rgb_cur), _ptr(rgb_prev), stride, _ptr(depth_cur),
                                              _ptr(depth_state), _ptr(mask_out), _ptr(pooled_out), ctypes.byref(prm),
                                              _stream())
        self.check(rc, "ggt_refine_depth_static")

    def ggt_refine_depth_batch(self, rgb_cur, rgb_prev, depth_cur, depth_state, mask_out=None, pooled_out=None,
                               lambda_t=0.7, beta=0.6, theta=0.0, downscale=4, pool=3):
        """ggt_refine_depth for a list of equally sized views in two launches; list entries may be None where allowed."""
        V = len(depth_cur)
        H, W = depth_cur[0].shape
        first = next((r for r in (rgb_cur or []) if r is not None), None)
        stride = 3 if first is None else int(first.shape[2])

        def arr(lst):
            if lst is None:
                return None
            return (ctypes.c_void_p * V)(*[None if t is None else t.data_ptr() for t in lst])
        for lst, dt, n in ((rgb_cur, "uint8", H * W * stride), (rgb_prev, "uint8", H * W * stride), (depth_cur, "float32", H * W),
                           (depth_state, "float32", H * W), (mask_out, "float32", H * W),
                           (pooled_out, "uint16", ((H + 3) // 4) * ((W + 3) // 4))):
            for t in (lst or []):
                _chk(t, dt, n, "ggt_refine_depth_batch argument")
        prm = _refine_params(lambda_t, beta, theta, downscale, pool)
        rc = self.lib.ggt_refine_depth_batch(self.h, V, W, H, arr(rgb_cur), arr(rgb_prev), stride, arr(depth_cur),
                                             arr(depth_state), arr(mask_out), arr(pooled_out), ctypes.byref(prm), _stream())
        self.check(rc, "ggt_refine_depth_batch")

    # ---- volume ------------------------------------------------------------------------------------
    def ggt_volume_bind(self, width, height, z_bins, dtype=GGT_F32, trunc_bins=2.0, trunc_metric=0.0,
                        w_sigma0=0.001, w_clip=0.02, w_window=7, weight_cap=64.0, decay=1.0) -> "Volume":
        return Volume(self, width, height, z_bins, dtype, trunc_bins, trunc_metric, w_sigma0, w_clip, w_window,
                      weight_cap, decay)

    # ---- a3-a6 -------------------------------------------------------------------------------------
    def _cams(self, target, views):
        V = len(views)
        arr = (ggt_camera * V)(*[to_camera(c) for c in views])
        return to_camera(target), arr

    def ggt_integrate(self, vol: "Volume", target, views: Sequence, depths: Sequence, flags=GGT_OVERWRITE):
        V = len(views)
        t, arr = self._cams(target, views)
        _chk_views(views, depths)
        ptrs = (ctypes.c_void_p * V)(*[d.data_ptr() for d in depths])
        rc = self.lib.ggt_integrate(self.h, vol.h, ctypes.byref(t), V, arr, ptrs, flags, _stream())
        self.check(rc, "ggt_integrate")

    def ggt_integrate_batch(self, vols, targets, rig_views, depths, view_index, flags=GGT_OVERWRITE):
        """n targets of one frame (volumes `vols`), each fusing the rig views listed in its row of `view_index`
        (n_targets x n_views ints); the weight maps of the rig views are computed once."""
        T, R = len(targets), len(rig_views)
        V = len(view_index[0])
        tarr = (ggt_camera * T)(*[to_camera(c) for c in targets])
        rarr = (ggt_camera * R)(*[to_camera(c) for c in rig_views])
        varr = (ctypes.c_void_p * T)(*[v.h for v in vols])
        _chk_views(rig_views, depths)
        ptrs = (ctypes.c_void_p * R)(*[d.data_ptr() for d in depths])
        idx = (ctypes.c_int32 * (T * V))(*[int(i) for row in view_index for i in row])
        rc = self.lib.ggt_integrate_batch(self.h, T, varr, tarr, R, rarr, ptrs, V, idx, flags, _stream())
        self.check(rc, "ggt_integrate_batch")

    def ggt_integrate_extract_batch(self, vols, targets, rig_views, depths, view_index, flags=GGT_OVERWRITE, depth=None,
                                    conf=None, bins=None):
        """ggt_integrate_batch with the zero-crossing search fused in; depth / conf / bins: lists of tensors (or None)."""
        T, R = len(targets), len(rig_views)
        V = len(view_index[0])
        tarr = (ggt_camera * T)(*[to_camera(c) for c in targets])
        rarr = (ggt_camera * R)(*[to_camera(c) for c in rig_views])
        varr = (ctypes.c_void_p * T)(*[v.h for v in vols])
        _chk_views(rig_views, depths)
        for lst, dt in ((depth, "float32"), (conf, "float32"), (bins, "int32")):
            for t, c in zip(lst or [], targets):
                _chk(t, dt, int(c.width) * int(c.height), "ggt_integrate_extract_batch output")
        ptrs = (ctypes.c_void_p * R)(*[d.data_ptr() for d in depths])
        idx = (ctypes.c_int32 * (T * V))(*[int(i) for row in view_index for i in row])

        def arr(lst):
            return None if lst is None else (ctypes.c_void_p * T)(*[None if t is None else t.data_ptr() for t in lst])
        rc = self.lib.ggt_integrate_extract_batch(self.h, T, varr, tarr, R, rarr, ptrs, V, idx, flags, arr(depth), arr(conf),
                                                  arr(bins), _stream())
        self.check(rc, "ggt_integrate_extract_batch")

    def ggt_integrate_extract(self, vol: "Volume", target, views, depths, flags=GGT_OVERWRITE, depth=None,
                              conf=None, bins=None):
        V = len(views)
        t, arr = self._cams(target, views)
        _chk_views(views, depths)
        self._chk_outputs(target, depth, conf, bins)
        ptrs = (ctypes.c_void_p * V)(*[d.data_ptr() for d in depths])
        rc = self.lib.ggt_integrate_extract(self.h, vol.h, ctypes.byref(t), V, arr, ptrs, flags, _ptr(depth),
                                            _ptr(conf), _ptr(bins), _stream())
        self.check(rc, "ggt_integrate_extract")

    # ---- a7 ----------------------------------------------------------------------------------------
    @staticmethod
    def _chk_outputs(target, depth, conf, ints):
        n = int(target.width) * int(target.height)
        _chk(depth, "float32", n, "depth output")
        _chk(conf, "float32", n, "confidence output")
        _chk(ints, "int32", n, "bin / steps output")

    def ggt_extract_depth(self, vol: "Volume", depth=None, conf=None, bins=None):
        self._chk_outputs(vol, depth, conf, bins)
        rc = self.lib.ggt_extract_depth(self.h, vol.h, _ptr(depth), _ptr(conf), _ptr(bins), _stream())
        self.check(rc, "ggt_extract_depth")

    # ---- f-1: the paper's own volume-free schedule ----------------------------------------------------
    def ggt_raymarch_depth(self, target, views, depths, z_near, z_far, depth=None, conf=None, steps=None, tau=0.02,
                           step_scale=0.8, min_step=1e-3, max_evals=4096, n_bisect=3, w_sigma0=0.001, w_clip=0.02,
                           w_window=7):
        V = len(views)
        t, arr = self._cams(target, views)
        _chk_views(views, depths)
        self._chk_outputs(target, depth, conf, steps)
        ptrs = (ctypes.c_void_p * V)(*[d.data_ptr() for d in depths])
        prm = ggt_raymarch_params(z_near, z_far, tau, step_scale, min_step, max_evals, n_bisect, w_sigma0, w_clip, w_window)
        rc = self.lib.ggt_raymarch_depth(self.h, ctypes.byref(t), V, arr, ptrs, ctypes.byref(prm), _ptr(depth), _ptr(conf),
                                         _ptr(steps), _stream())
        self.check(rc, "ggt_raymarch_depth")

    # ---- f-2: the previous output depth as one more view (Eq. 3, 13-14) ------------------------------
    def ggt_temporal_weight(self, prev_target, prev_depth, prev_conf, views, masks, weight_out, beta=1.0, eta=15.0):
        V = len(views)
        t, arr = self._cams(prev_target, views if V else [prev_target])
        n = int(prev_target.width) * int(prev_target.height)
        for x, nm in ((prev_depth, "prev_depth"), (prev_conf, "prev_conf"), (weight_out, "weight_out")):
            _chk(x, "float32", n, nm)
        _chk_views(views, masks, what="mask")
        ptrs = (ctypes.c_void_p * max(V, 1))(*[m.data_ptr() for m in masks])
        rc = self.lib.ggt_temporal_weight(self.h, ctypes.byref(t), prev_depth.data_ptr(), prev_conf.data_ptr(), V, arr, ptrs,
                                          beta, eta, weight_out.data_ptr(), _stream())
        self.check(rc, "ggt_temporal_weight")

    @staticmethod
    def _weight_ptrs(weights, V):
        if weights is None:
            return None
        return (ctypes.c_void_p * V)(*[None if w is None else w.data_ptr() for w in weights])

    def ggt_integrate_weighted(self, vol: "Volume", target, views, depths, weights, flags=GGT_OVERWRITE):
        V = len(views)
        t, arr = self._cams(target, views)
        _chk_views(views, depths)
        _chk_views(views, weights or [], what="weights")
        ptrs = (ctypes.c_void_p * V)(*[d.data_ptr() for d in depths])
        rc = self.lib.ggt_integrate_weighted(self.h, vol.h, ctypes.byref(t), V, arr, ptrs, self._weight_ptrs(weights, V), flags,
                                             _stream())
        self.check(rc, "ggt_integrate_weighted")

    def ggt_raymarch_depth_weighted(self, target, views, depths, weights, z_near, z_far, depth=None, conf=None, steps=None,
                                    tau=0.02, step_scale=0.8, min_step=1e-3, max_evals=4096, n_bisect=3, w_sigma0=0.001,
                                    w_clip=0.02, w_window=7):
        V = len(views)
        t, arr = self._cams(target, views)
        _chk_views(views, depths)
        _chk_views(views, weights or [], what="weights")
        self._chk_outputs(target, depth, conf, steps)
        ptrs = (ctypes.c_void_p * V)(*[d.data_ptr() for d in depths])
        prm = ggt_raymarch_params(z_near, z_far, tau, step_scale, min_step, max_evals, n_bisect, w_sigma0, w_clip, w_window)
        rc = self.lib.ggt_raymarch_depth_weighted(self.h, ctypes.byref(t), V, arr, ptrs, self._weight_ptrs(weights, V),
                                                  ctypes.byref(prm), _ptr(depth), _ptr(conf), _ptr(steps), _stream())
        self.check(rc, "ggt_raymarch_depth_weighted")

    # ---- f-3: forward warping with pixel-sized 3D Gaussians --------------------------------------------
    def ggt_splat_forward(self, target, view, depth, rgb=None, mask=None, out_rgb=None, out_alpha=None, out_depth=None,
                          out_mask=None, out_count=None, sigma_px=0.5, dilation=0.3, z_cull=0.2):
        t, arr = self._cams(target, [view])
        stride = 3 if rgb is None else int(rgb.shape[2])
        ns, nt = int(view.width) * int(view.height), int(target.width) * int(target.height)
        _chk(depth, "float32", ns, "depth"); _chk(rgb, "uint8", ns * stride, "rgb"); _chk(mask, "float32", ns, "mask")
        _chk(out_rgb, "float32", 3 * nt, "out_rgb"); _chk(out_alpha, "float32", nt, "out_alpha")
        _chk(out_depth, "float32", nt, "out_depth"); _chk(out_mask, "float32", nt, "out_mask"); _chk(out_count, "int32", nt, "out_count")
        prm = ggt_splat_params(sigma_px, dilation, z_cull, 0)
        rc = self.lib.ggt_splat_forward(self.h, ctypes.byref(t), arr, depth.data_ptr(), _ptr(rgb), stride, _ptr(mask),
                                        ctypes.byref(prm), _ptr(out_rgb), _ptr(out_alpha), _ptr(out_depth), _ptr(out_mask),
                                        _ptr(out_count), _stream())
        self.check(rc, "ggt_splat_forward")

    def ggt_splat_reserve(self, entries: int):
        self.check(self.lib.ggt_splat_reserve(self.h, int(entries)), "ggt_splat_reserve")

    def ggt_splat_status(self):
        """(entries of the last call, entries needed by an overflowed call or 0); synchronises the current stream."""
        last, need = ctypes.c_int64(), ctypes.c_int64()
        self.check(self.lib.ggt_splat_status(self.h, ctypes.byref(last), ctypes.byref(need), _stream()), "ggt_splat_status")
        return int(last.value), int(need.value)

    def ggt_temporal_weight_mask(self, prev_depth, prev_conf, masks, weight_out, beta=1.0, eta=15.0):
        K = len(masks)
        for x in [prev_depth, prev_conf, weight_out] + list(masks):
            _chk(x, "float32", prev_depth.numel(), "ggt_temporal_weight_mask argument")
        ptrs = (ctypes.c_void_p * K)(*[m.data_ptr() for m in masks])
        rc = self.lib.ggt_temporal_weight_mask(self.h, prev_depth.numel(), prev_depth.data_ptr(), prev_conf.data_ptr(), K, ptrs,
                                               beta, eta, weight_out.data_ptr(), _stream())
        self.check(rc, "ggt_temporal_weight_mask")

    # ---- f-4: network-input geometry features of the guidance depth ---------------------------------
    def ggt_guidance_features(self, target, depth, views, features):
        V = len(views)
        t, arr = self._cams(target, views)
        n = int(target.width) * int(target.height)
        _chk(depth, "float32", n, "depth")
        _chk(features, "float32", 4 * V * n, "features")
        rc = self.lib.ggt_guidance_features(self.h, ctypes.byref(t), depth.data_ptr(), V, arr, features.data_ptr(), _stream())
        self.check(rc, "ggt_guidance_features")

    # ---- end-to-end from host buffers -----------------------------------------------------------------
    def ggt_frame_host(self, vol: "Volume", target, views, host_rgb: Optional[Sequence], host_depth_in: Sequence,
                       slots: Sequence[int], slot_state: np.ndarray, staging, host_depth, host_conf,
                       flags=GGT_OVERWRITE, refine_params: Optional[ggt_refine_params] = None):
        """host_* are pinned CPU torch tensors; slot_state is a numpy uint32 array kept by the caller."""
        V = len(views)
        t, arr = self._cams(target, views)
        for k, c in enumerate(views):
            n = int(c.width) * int(c.height)
            _chk(host_depth_in[k], "float32", n, "host depth of view %d" % k, cuda=False)
            if host_rgb is not None:
                _chk(host_rgb[k], "uint8", 3 * n, "host colour of view %d" % k, cuda=False)
        nt = int(target.width) * int(target.height)
        _chk(host_depth, "float32", nt, "host_depth", cuda=False); _chk(host_conf, "float32", nt, "host_conf", cuda=False)
        _chk(staging, "uint8", None, "staging")
        rgbp = None
        if host_rgb is not None:
            rgbp = (ctypes.c_void_p * V)(*[None if r is None else r.data_ptr() for r in host_rgb])
        dp = (ctypes.c_void_p * V)(*[d.data_ptr() for d in host_depth_in])
        sl = (ctypes.c_int32 * V)(*[int(s) for s in slots])
        rc = self.lib.ggt_frame_host(
            self.h, vol.h, ctypes.byref(t), V, arr, rgbp, dp, sl, int(slot_state.size),
            slot_state.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)),
            ctypes.byref(refine_params) if refine_params is not None else None, flags, staging.data_ptr(),
            staging.numel(), _ptr(host_depth), _ptr(host_conf), _stream())
        self.check(rc, "ggt_frame_host")

    def ggt_frame_host_results_wait(self):
        """The current stream waits for the result copies of all GGT_FRAME_RESULTS_ASYNC calls made so far."""
        self.check(self.lib.ggt_frame_host_results_wait(self.h, _stream()), "ggt_frame_host_results_wait")


class Volume:
    """ggt_volume bound to a torch-owned uint8 storage tensor."""

    def __init__(self, ctx: Context, width, height, z_bins, dtype, trunc_bins, trunc_metric, w_sigma0, w_clip,
                 w_window, weight_cap, decay):
        import torch
        self.ctx = ctx
        self.z = np.ascontiguousarray(z_bins, dtype=np.float32)
        self.desc = ggt_volume_desc(int(width), int(height), int(self.z.size),
                                    self.z.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), trunc_bins, trunc_metric,
                                    w_sigma0, w_clip, int(w_window), weight_cap, decay, int(dtype))
        self.width, self.height, self.bins, self.dtype = int(width), int(height), int(self.z.size), int(dtype)
        n = ctx.lib.ggt_volume_bytes(ctypes.byref(self.desc))
        if n == 0:
            raise GgtError("ggt_volume_bytes: bad descriptor")
        self.nbytes = int(n)
        self.storage = torch.empty(n, dtype=torch.uint8, device="cuda")
        h = ctypes.c_void_p()
        ctx.check(ctx.lib.ggt_volume_bind(ctx.h, ctypes.byref(self.desc), self.storage.data_ptr(), n, ctypes.byref(h)),
                  "ggt_volume_bind")
        self.h = h

    def ggt_volume_reset(self):
        self.ctx.check(self.ctx.lib.ggt_volume_reset(self.ctx.h, self.h, _stream()), "ggt_volume_reset")

    def ggt_volume_export(self):
        """(T, W) torch fp32 tensors of shape (H_t*W_t, D), canonical bin-fastest layout."""
        import torch
        n = self.width * self.height
        T = torch.empty((n, self.bins), dtype=torch.float32, device="cuda")
        W = torch.empty((n, self.bins), dtype=torch.float32, device="cuda")
        self.ctx.check(self.ctx.lib.ggt_volume_export(self.ctx.h, self.h, T.data_ptr(), W.data_ptr(), _stream()),
                       "ggt_volume_export")
        return T, W

    def ggt_volume_tables(self):
        z = np.empty(self.bins, np.float32)
        tau = np.empty(self.bins, np.float32)
        self.ctx.lib.ggt_volume_tables(self.h, z.ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                                       tau.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
        return z, tau

    def close(self):
        if getattr(self, "h", None):
            self.ctx.lib.ggt_volume_unbind(self.ctx.h, self.h)
            self.h = None
