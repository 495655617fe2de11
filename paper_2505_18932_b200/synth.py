"""Seeded synthetic multi-camera inputs shaped like the paper's workloads.

This module is the ONE piece shared by the CPU oracle (`oracle/`) and the CUDA path: it produces
inputs (cameras, depth maps, colour images, depth-bin tables) and nothing else.  It contains none of
the method's arithmetic (no mask, no TSDF, no weights, no extraction): it is an analytic ray-caster
plus a counter-based random number generator.  numpy only, deterministic, seed-addressed.

Recipe (shapes from PAPER.md:149, 394-406 and BASELINE.json:configs):
  * counter-based RNG: u = splitmix64(seed ^ stream*GOLDEN ^ index) -> [0,1); Gaussian by Box-Muller;
  * un-normalised camera rays ((i+0.5-cx)/fx, (j+0.5-cy)/fy, 1): the ray parameter IS z-depth,
    which is what the paper's depth maps hold (Eq. 9 compares them with z_k);
  * nearest hit of a back plane, spheres and axis-aligned boxes; primitives move on straight lines;
  * depth noise D*(1 + sigma*n), invalid pixels D = 0 with probability p_inv;
  * uint8 procedural texture in object-local coordinates + integer sensor noise in {-1,0,1}.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence, Tuple

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


# --------------------------------------------------------------------------------------------------
# counter-based RNG
# --------------------------------------------------------------------------------------------------
def splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output step applied element-wise to uint64 counters."""
    with np.errstate(over="ignore"):
        z = (np.asarray(x, dtype=np.uint64) + _GOLDEN).astype(np.uint64)
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def _key(seed: int, stream: int) -> np.uint64:
    with np.errstate(over="ignore"):
        return np.uint64(seed) ^ (np.uint64(stream) * _GOLDEN)


def uniform(seed: int, stream: int, index) -> np.ndarray:
    """float64 uniform in [0,1) addressed by (seed, stream, index)."""
    idx = np.asarray(index, dtype=np.uint64)
    bits = splitmix64(splitmix64(idx ^ _key(seed, stream)))
    return (bits >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, index) -> np.ndarray:
    """float64 standard normal (Box-Muller on two counters of the same index)."""
    u1 = uniform(seed, 2 * stream + 1, index)
    u2 = uniform(seed, 2 * stream + 2, index)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


def stream_id(*parts: int) -> int:
    """Mix small integers (frame, view, purpose, ...) into one stream number."""
    s = 0x1234567
    for p in parts:
        s = (s * 1000003 + int(p) + 1) & 0x3FFFFFFFFFFF
    return s


# --------------------------------------------------------------------------------------------------
# cameras
# --------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Camera:
    """Pinhole camera, world -> camera x_cam = R p + t, pixel centres at +0.5.

    Values are stored as float32 (what both implementations receive)."""
    fx: float
    fy: float
    cx: float
    cy: float
    R: np.ndarray  # (3,3) float32 row-major
    t: np.ndarray  # (3,) float32
    width: int
    height: int

    def __post_init__(self):
        self.fx, self.fy = float(np.float32(self.fx)), float(np.float32(self.fy))
        self.cx, self.cy = float(np.float32(self.cx)), float(np.float32(self.cy))
        self.R = np.ascontiguousarray(self.R, dtype=np.float32).reshape(3, 3)
        self.t = np.ascontiguousarray(self.t, dtype=np.float32).reshape(3)

    @property
    def centre(self) -> np.ndarray:
        return -(self.R.astype(np.float64).T @ self.t.astype(np.float64))


def camera_from_pose(centre, R, fx, fy, cx, cy, width, height) -> Camera:
    R = np.asarray(R, dtype=np.float64)
    t = -R @ np.asarray(centre, dtype=np.float64)
    return Camera(fx, fy, cx, cy, R, t, width, height)


def rot_yaw_pitch(yaw: float, pitch: float) -> np.ndarray:
    """World->camera rotation for a camera yawed about y then pitched about x (radians)."""
    cy_, sy_ = math.cos(yaw), math.sin(yaw)
    cp_, sp_ = math.cos(pitch), math.sin(pitch)
    Ry = np.array([[cy_, 0, -sy_], [0, 1, 0], [sy_, 0, cy_]], dtype=np.float64)
    Rx = np.array([[1, 0, 0], [0, cp_, sp_], [0, -sp_, cp_]], dtype=np.float64)
    return Rx @ Ry


def look_at(centre, target=(0.0, 0.0, 0.0)) -> np.ndarray:
    """World->camera rotation whose +z axis points from `centre` to `target`, image y = world y."""
    c = np.asarray(centre, dtype=np.float64)
    f = np.asarray(target, dtype=np.float64) - c
    f /= np.linalg.norm(f)
    r = np.cross(np.array([0.0, 1.0, 0.0]), f)
    r /= np.linalg.norm(r)
    d = np.cross(f, r)
    return np.stack([r, d, f])


def grid_rig(width: int, height: int, n: int = 4, pitch: float = 0.2,
             focal_frac: float = 0.75) -> List[Camera]:
    """n x n planar rig, parallel axes looking down +z (BASELINE.json:configs[1]: 16 cameras, 20 cm)."""
    cams = []
    f = focal_frac * width
    for b in range(n):
        for a in range(n):
            c = ((a - (n - 1) / 2) * pitch, (b - (n - 1) / 2) * pitch, 0.0)
            cams.append(camera_from_pose(c, np.eye(3), f, f, width / 2, height / 2, width, height))
    return cams


def nearest_views(target: Camera, cams: Sequence[Camera], k: int,
                  exclude: Optional[int] = None) -> List[int]:
    """Indices of the k cameras whose centres are closest to the target's."""
    tc = target.centre
    d = [(float(np.sum((c.centre - tc) ** 2)), i) for i, c in enumerate(cams) if i != exclude]
    d.sort()
    return [i for _, i in d[:k]]


# --------------------------------------------------------------------------------------------------
# depth-bin tables (sample planes including both ends)
# --------------------------------------------------------------------------------------------------
def bins_uniform(near: float, far: float, n: int) -> np.ndarray:
    j = np.arange(n, dtype=np.float64)
    return (near + j * (far - near) / (n - 1)).astype(np.float32)


def bins_inverse(near: float, far: float, n: int) -> np.ndarray:
    j = np.arange(n, dtype=np.float64)
    inv = 1.0 / near + j * (1.0 / far - 1.0 / near) / (n - 1)
    return (1.0 / inv).astype(np.float32)


# --------------------------------------------------------------------------------------------------
# scene + ray-caster
# --------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Primitive:
    kind: str                 # "sphere" | "box"
    centre: np.ndarray        # (3,) at time 0
    size: np.ndarray          # sphere: (r,r,r); box: half-extents
    velocity: np.ndarray      # (3,) m/s
    phase: np.ndarray         # (9,) texture phases

    def centre_at(self, time: float) -> np.ndarray:
        return self.centre + self.velocity * time


@dataclasses.dataclass
class Scene:
    plane_z: float
    prims: List[Primitive]


def make_scene(seed: int, plane_z: float, n_spheres: int, n_boxes: int,
               sphere_r=(0.15, 0.4), box_h=(0.1, 0.3),
               cx=(-1.5, 1.5), cy=(-0.8, 0.8), cz=(1.5, 3.5), max_speed: float = 0.0) -> Scene:
    prims = []
    for i in range(n_spheres + n_boxes):
        u = uniform(seed, stream_id(77, i), np.arange(24))
        c = np.array([cx[0] + u[0] * (cx[1] - cx[0]), cy[0] + u[1] * (cy[1] - cy[0]),
                      cz[0] + u[2] * (cz[1] - cz[0])])
        if i < n_spheres:
            r = sphere_r[0] + u[3] * (sphere_r[1] - sphere_r[0])
            size, kind = np.array([r, r, r]), "sphere"
        else:
            size = box_h[0] + u[3:6] * (box_h[1] - box_h[0])
            kind = "box"
        v = (2.0 * u[6:9] - 1.0)
        v = v / max(np.linalg.norm(v), 1e-9) * (max_speed * u[9])
        prims.append(Primitive(kind, c, size, v, u[10:19] * 2.0 * math.pi))
    return Scene(plane_z, prims)


def _texture(local: np.ndarray, phase: np.ndarray) -> np.ndarray:
    """uint8 RGB from object-local coordinates: product of 3 sinusoids per channel."""
    out = np.empty(local.shape[:-1] + (3,), dtype=np.float64)
    x, y, z = local[..., 0], local[..., 1], local[..., 2]
    for c in range(3):
        p = phase[3 * c:3 * c + 3]
        f = 9.0 + 4.0 * c
        out[..., c] = np.sin(f * x + p[0]) * np.sin((f + 2.0) * y + p[1]) * np.sin((f - 3.0) * z + p[2])
    return np.clip(np.rint(127.5 + 110.0 * out), 0, 255).astype(np.uint8)


def raycast(cam: Camera, scene: Scene, time: float = 0.0, want_colour: bool = False
            ) -> Tuple[np.ndarray, Optional[np.ndarray]]:
    """Noise-free z-depth (float64, H x W) of the nearest hit and, optionally, uint8 RGB colour."""
    W, H = cam.width, cam.height
    R = cam.R.astype(np.float64)
    o = cam.centre
    ii = (np.arange(W, dtype=np.float64) + 0.5 - cam.cx) / cam.fx
    jj = (np.arange(H, dtype=np.float64) + 0.5 - cam.cy) / cam.fy
    Rt = R.T

    def dirs(x0, x1, y0, y1):
        gx, gy = np.meshgrid(ii[x0:x1], jj[y0:y1])
        dc = np.stack([gx, gy, np.ones_like(gx)], axis=-1)
        return dc @ Rt.T  # world direction per unit z-depth

    # back plane z_world = plane_z
    d_all = dirs(0, W, 0, H)
    with np.errstate(divide="ignore", invalid="ignore"):
        s = (scene.plane_z - o[2]) / d_all[..., 2]
    depth = np.where(s > 0, s, 0.0)
    rgb = None
    if want_colour:
        hit = o + d_all * depth[..., None]
        rgb = _texture(hit * 0.35, np.arange(9) * 0.7)
    del d_all

    for prim in scene.prims:
        c = prim.centre_at(time)
        # conservative pixel window from the bounding sphere projected into the camera
        rad = float(np.linalg.norm(prim.size)) if prim.kind == "box" else float(prim.size[0])
        cc = R @ (c - o)
        if cc[2] - rad <= 1e-3:
            x0, x1, y0, y1 = 0, W, 0, H
        else:
            zmin = cc[2] - rad
            # angular extent bound: |x/z| <= (|cx| + rad)/zmin style conservative box
            xs = [(cc[0] - rad) / zmin, (cc[0] + rad) / zmin, (cc[0] - rad) / (cc[2] + rad),
                  (cc[0] + rad) / (cc[2] + rad)]
            ys = [(cc[1] - rad) / zmin, (cc[1] + rad) / zmin, (cc[1] - rad) / (cc[2] + rad),
                  (cc[1] + rad) / (cc[2] + rad)]
            x0 = int(max(0, math.floor(min(xs) * cam.fx + cam.cx - 1)))
            x1 = int(min(W, math.ceil(max(xs) * cam.fx + cam.cx + 1)))
            y0 = int(max(0, math.floor(min(ys) * cam.fy + cam.cy - 1)))
            y1 = int(min(H, math.ceil(max(ys) * cam.fy + cam.cy + 1)))
            if x0 >= x1 or y0 >= y1:
                continue
        d = dirs(x0, x1, y0, y1)
        oc = o - c
        if prim.kind == "sphere":
            a = np.sum(d * d, axis=-1)
            b = d @ oc
            cq = float(oc @ oc) - prim.size[0] ** 2
            disc = b * b - a * cq
            ok = disc > 0
            sq = np.sqrt(np.where(ok, disc, 0.0))
            s = (-b - sq) / a
            ok &= s > 1e-6
        else:
            with np.errstate(divide="ignore", invalid="ignore"):
                inv = 1.0 / d
                t0 = (-prim.size - oc) * inv
                t1 = (prim.size - oc) * inv
            tn = np.max(np.minimum(t0, t1), axis=-1)
            tf = np.min(np.maximum(t0, t1), axis=-1)
            s = tn
            ok = (tn < tf) & (tn > 1e-6)
        sub = depth[y0:y1, x0:x1]
        closer = ok & ((s < sub) | (sub <= 0))
        sub[closer] = s[closer]
        if want_colour and np.any(closer):
            hit_local = (oc + d[closer] * s[closer][..., None])
            rgb[y0:y1, x0:x1][closer] = _texture(hit_local, prim.phase)
    return depth, rgb


def noisy_depth(depth: np.ndarray, seed: int, stream: int, sigma: float, p_invalid: float
                ) -> np.ndarray:
    """D*(1+sigma*n) with a fraction p_invalid of pixels set to 0; float32."""
    idx = np.arange(depth.size, dtype=np.uint64).reshape(depth.shape)
    out = depth.copy()
    if sigma > 0:
        out = out * (1.0 + sigma * normal(seed, stream, idx))
    if p_invalid > 0:
        out[uniform(seed, stream + 0x5555, idx) < p_invalid] = 0.0
    return np.ascontiguousarray(out, dtype=np.float32)


def noisy_colour(rgb: np.ndarray, seed: int, stream: int) -> np.ndarray:
    """Add integer sensor noise in {-1,0,1} per channel, clipped to uint8."""
    idx = np.arange(rgb.size, dtype=np.uint64).reshape(rgb.shape)
    n = np.floor(uniform(seed, stream + 0x3333, idx) * 3.0).astype(np.int16) - 1
    return np.clip(rgb.astype(np.int16) + n, 0, 255).astype(np.uint8)


# --------------------------------------------------------------------------------------------------
# the five workload configurations (BASELINE.json:configs[0..4] == C1..C5)
# --------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    rig: List[Camera]                 # all input cameras
    scene: Scene
    z_bins: np.ndarray                # float32 (D,)
    n_views: int                      # V
    n_frames: int
    fps: float
    sigma: float
    p_invalid: float
    colour: bool                      # colour images + ggt_refine_depth
    persistent: bool
    storage: str                      # "f32" | "f16"
    weight_cap: float
    trunc_bins: float = 2.0
    target_size: Tuple[int, int] = (0, 0)
    target_focal: float = 0.0
    n_targets: int = 1

    # ---- per-frame camera selection ------------------------------------------------------------
    def targets(self, frame: int) -> List[Camera]:
        raise NotImplementedError

    def views_for(self, target: Camera, exclude: Optional[int] = None) -> List[int]:
        return nearest_views(target, self.rig, self.n_views, exclude)

    # ---- per-frame inputs ------------------------------------------------------------------------
    def view_inputs(self, frame: int, view: int):
        """(depth float32 HxW, rgb uint8 HxWx3 or None) for rig camera `view` at `frame`."""
        cache = self.__dict__.setdefault("_cache", {})
        if (frame, view) in cache:
            return cache[(frame, view)]
        time = frame / self.fps
        d, rgb = raycast(self.rig[view], self.scene, time, want_colour=self.colour)
        st = stream_id(frame, view, 1)
        d = noisy_depth(d, self.seed, st, self.sigma, self.p_invalid)
        if rgb is not None:
            rgb = noisy_colour(rgb, self.seed, st)
        d.setflags(write=False)
        if rgb is not None:
            rgb.setflags(write=False)
        if len(cache) >= 48:              # bounded memo: both pipelines of a test ask for the same inputs
            cache.pop(next(iter(cache)))
        cache[(frame, view)] = (d, rgb)
        return d, rgb

    def true_depth(self, cam: Camera, frame: int) -> np.ndarray:
        """Noise-free ground-truth z-depth for any camera (test pins only)."""
        return raycast(cam, self.scene, frame / self.fps)[0]


class _C1(Workload):
    def targets(self, frame):
        return [camera_from_pose((0.0, 0.0, -2.0), np.eye(3), 60, 60, 32, 24, 64, 48)]

    def views_for(self, target, exclude=None):
        return [0, 1, 2, 3]


class _GridSingle(Workload):
    def targets(self, frame):
        u = uniform(self.seed, stream_id(901), np.arange(2))
        W, H = self.target_size
        c = ((u[0] - 0.5) * 0.2, (u[1] - 0.5) * 0.2, 0.0)
        return [camera_from_pose(c, np.eye(3), self.target_focal, self.target_focal, W / 2, H / 2, W, H)]


class _GridHeldOut(Workload):
    """C3: target = a rig camera held out of the inputs, index re-drawn every 10 frames."""

    def target_index(self, frame):
        u = uniform(self.seed, stream_id(902), np.arange(frame // 10 + 1))[-1]
        return int(u * len(self.rig)) % len(self.rig)

    def targets(self, frame):
        return [self.rig[self.target_index(frame)]]

    def views_for(self, target, exclude=None):
        idx = [i for i, c in enumerate(self.rig) if c is target]
        return nearest_views(target, self.rig, self.n_views, idx[0] if idx else exclude)


class _Lissajous(Workload):
    """C4: target moving on a smooth seeded path inside the rig, yaw/pitch <= 3 degrees."""

    def targets(self, frame):
        ph = uniform(self.seed, stream_id(903), np.arange(5)) * 2.0 * math.pi
        a = 2.0 * math.pi * frame / 60.0
        c = (0.25 * math.sin(a + ph[0]), 0.25 * math.sin(2 * a + ph[1]), 0.05 * math.sin(a + ph[2]))
        yaw = math.radians(3.0) * math.sin(a + ph[3])
        pitch = math.radians(3.0) * math.sin(2 * a + ph[4])
        W, H = self.target_size
        return [camera_from_pose(c, rot_yaw_pitch(yaw, pitch), self.target_focal, self.target_focal,
                                 W / 2, H / 2, W, H)]


class _StereoBatch(Workload):
    """C5: 4 seeded head positions x {-3.2, +3.2} cm in x -> 8 targets per frame."""

    def targets(self, frame):
        u = uniform(self.seed, stream_id(904), np.arange(12)).reshape(4, 3)
        W, H = self.target_size
        out = []
        for h in range(4):
            base = np.array([(u[h, 0] - 0.5) * 0.5, (u[h, 1] - 0.5) * 0.5, (u[h, 2] - 0.5) * 0.1])
            for eye in (-0.032, 0.032):
                c = base + np.array([eye, 0.0, 0.0])
                out.append(camera_from_pose(c, np.eye(3), self.target_focal, self.target_focal,
                                            W / 2, H / 2, W, H))
        return out[: self.n_targets]


def arc_rig() -> List[Camera]:
    """C1: 4 cameras on a 2 m-radius arc facing the origin, 15 cm arc spacing."""
    cams = []
    for i in range(4):
        phi = (i - 1.5) * 0.075
        c = (2.0 * math.sin(phi), 0.0, -2.0 * math.cos(phi))
        cams.append(camera_from_pose(c, look_at(c), 60, 60, 32, 24, 64, 48))
    return cams


def workload(name: str, scale: float = 1.0) -> Workload:
    """Build workload "C1".."C5".  `scale` < 1 shrinks image sizes (tests only; shapes otherwise kept)."""
    def sz(w, h):
        return (max(16, int(round(w * scale / 4)) * 4), max(16, int(round(h * scale / 4)) * 4))

    if name == "C1":
        seed = 1001
        u = uniform(seed, stream_id(900), np.arange(3))
        sphere = Primitive("sphere", (u - 0.5) * 0.6, np.array([0.4, 0.4, 0.4]), np.zeros(3),
                           np.arange(9) * 0.3)
        return _C1("C1", seed, arc_rig(), Scene(1.5, [sphere]), bins_uniform(0.5, 4.0, 32), 4, 1, 30.0,
                   0.005, 0.0, False, False, "f32", 64.0, target_size=(64, 48), target_focal=60.0)
    if name == "C2":
        W, H = sz(640, 360)
        return _GridSingle("C2", 1002, grid_rig(W, H), make_scene(1002, 4.5, 8, 4),
                           bins_inverse(0.5, 5.0, 64), 4, 1, 30.0, 0.01, 0.02, False, False, "f32", 64.0,
                           target_size=(W, H), target_focal=0.75 * W)
    if name == "C3":
        W, H = sz(1920, 1080)
        return _GridHeldOut("C3", 1003, grid_rig(W, H), make_scene(1003, 4.5, 8, 4, max_speed=0.5),
                            bins_inverse(0.5, 5.0, 128), 4, 30, 30.0, 0.01, 0.02, True, False, "f32",
                            64.0, target_size=(W, H), target_focal=0.75 * W)
    if name == "C4":
        W, H = sz(1920, 1080)
        return _Lissajous("C4", 1004, grid_rig(W, H), make_scene(1004, 4.5, 20, 12, max_speed=0.5),
                          bins_inverse(0.5, 5.0, 256), 8, 60, 30.0, 0.01, 0.02, False, True, "f16", 64.0,
                          target_size=(W, H), target_focal=0.75 * W)
    if name == "C5":
        W, H = sz(1920, 1080)
        tw, th = sz(2048, 2048)
        return _StereoBatch("C5", 1005, grid_rig(W, H), make_scene(1005, 4.5, 8, 4, max_speed=0.5),
                            bins_inverse(0.5, 5.0, 128), 6, 30, 30.0, 0.01, 0.02, True, True, "f32", 64.0,
                            target_size=(tw, th), target_focal=0.5 * tw, n_targets=8)
    raise ValueError(name)
