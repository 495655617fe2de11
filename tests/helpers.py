"""Shared test plumbing: run the oracle and the CUDA path on the same seeded inputs and compare.

Tolerances are BASELINE.json:north_star's: mask / zero-crossing bin bit-exact except where |tsdf| < 1e-6,
TSDF / weight within 1e-5 relative, depth within 1e-4 of the depth range.  Because both sides follow the
determinism contract (P14) the comparison is in practice bit-exact; the helpers report both.
"""
from __future__ import annotations

import numpy as np

import oracle
from paper_2505_18932_b200 import synth

REFINE = dict(lambda_t=0.7, beta=0.6, theta=8.0 / 255.0)


def sample_rays(width, height, every, seed):
    """Seeded subset of target pixels: ~1/every of them, plus the four corners and last row/col samples."""
    n = width * height
    if every <= 1:
        return None
    k = max(64, n // every)
    u = synth.uniform(seed, synth.stream_id(555), np.arange(k))
    idx = np.unique(np.concatenate([(u * n).astype(np.int64), [0, width - 1, n - width, n - 1]]))
    return idx.astype(np.int32)


class OraclePipeline:
    """Frame loop on the CPU oracle; integrate / extract restricted to a ray subset (rays independent)."""

    def __init__(self, wl: synth.Workload, rays_every: int = 1, use_refine=None):
        self.wl = wl
        self.state = {}      # rig camera index -> (refined depth, previous rgb)
        self.every = rays_every
        self.vol = {}        # target slot -> (T, W)
        self.use_refine = wl.colour if use_refine is None else use_refine
        self.tau = oracle.tau_table(wl.z_bins, wl.trunc_bins)

    def refine_view(self, frame, view):
        d, rgb = self.wl.view_inputs(frame, view)
        if not self.use_refine:
            return d, None, None
        prev = self.state.get(view)
        if prev is None:
            out, M, pq, _ = oracle.refine(None, None, d, d)
        else:
            out, M, pq, _ = oracle.refine(rgb, prev[1], d, prev[0], **REFINE)
        self.state[view] = (out, rgb)
        return out, M, pq

    def frame(self, frame):
        wl = self.wl
        res = []
        done = {}            # views already refined in this frame (each view is refined once per frame)
        for slot, tgt in enumerate(wl.targets(frame)):
            vi = wl.views_for(tgt)
            for v in vi:
                if v not in done:
                    done[v] = self.refine_view(frame, v)[0]
            depths = [done[v] for v in vi]
            maps = [oracle.weight_map(d) for d in depths]
            rays = sample_rays(tgt.width, tgt.height, self.every, wl.seed + slot)
            T, W = self.vol.get(slot, (None, None)) if wl.persistent else (None, None)
            T, W = oracle.integrate(tgt, wl.z_bins, self.tau, [wl.rig[v] for v in vi], maps, rays=rays, T=T, Wt=W,
                                    accumulate=wl.persistent, decay=1.0, cap=wl.weight_cap,
                                    half_storage=wl.storage == "f16")
            if wl.persistent:
                self.vol[slot] = (T, W)
            depth, conf, bins = oracle.extract(wl.z_bins, T, W)
            res.append(dict(target=tgt, views=vi, depths=depths, rays=rays, T=T, W=W, depth=depth, conf=conf, bins=bins))
        return res


class CudaPipeline:
    """The same frame loop through the C ABI (binding.Context)."""

    def __init__(self, wl: synth.Workload, fused=False, use_refine=None):
        import torch
        from paper_2505_18932_b200 import binding
        self.torch, self.binding = torch, binding
        self.wl = wl
        self.ctx = binding.Context()
        self.state = {}
        self.vols = {}
        self.fused = fused
        self.use_refine = wl.colour if use_refine is None else use_refine

    def volume(self, slot, tgt):
        b = self.binding
        if slot not in self.vols:
            v = self.ctx.ggt_volume_bind(tgt.width, tgt.height, self.wl.z_bins,
                                         dtype=b.GGT_F16 if self.wl.storage == "f16" else b.GGT_F32,
                                         trunc_bins=self.wl.trunc_bins, weight_cap=self.wl.weight_cap)
            v.ggt_volume_reset()
            self.vols[slot] = v
        return self.vols[slot]

    def refine_view(self, frame, view, want_mask=False):
        torch = self.torch
        d, rgb = self.wl.view_inputs(frame, view)
        dg = torch.from_numpy(d).cuda()
        if not self.use_refine:
            return dg, None, None
        rg = torch.from_numpy(rgb).cuda()
        H, W = d.shape
        mask = torch.empty((H, W), dtype=torch.float32, device="cuda") if want_mask else None
        pooled = torch.zeros(((H + 3) // 4, (W + 3) // 4), dtype=torch.uint16, device="cuda") if want_mask else None
        prev = self.state.get(view)
        if prev is None:
            st = torch.empty_like(dg)
            self.ctx.ggt_refine_depth(None, None, dg, st, mask_out=mask)
            pooled = None
        else:
            st = prev[0]
            self.ctx.ggt_refine_depth(rg, prev[1], dg, st, mask_out=mask, pooled_out=pooled, **REFINE)
        self.state[view] = (st, rg)
        return st, mask, pooled

    def frame(self, frame):
        torch, b = self.torch, self.binding
        wl = self.wl
        res = []
        done = {}            # views already refined in this frame (each view is refined once per frame)
        for slot, tgt in enumerate(wl.targets(frame)):
            vi = wl.views_for(tgt)
            for v in vi:
                if v not in done:
                    done[v] = self.refine_view(frame, v)[0]
            depths = [done[v] for v in vi]
            vol = self.volume(slot, tgt)
            n = tgt.width * tgt.height
            depth = torch.empty(n, dtype=torch.float32, device="cuda")
            conf = torch.empty(n, dtype=torch.float32, device="cuda")
            bins = torch.empty(n, dtype=torch.int32, device="cuda")
            flags = b.GGT_ACCUMULATE if wl.persistent else b.GGT_OVERWRITE
            views = [wl.rig[v] for v in vi]
            if self.fused:
                self.ctx.ggt_integrate_extract(vol, tgt, views, depths, flags, depth, conf, bins)
            else:
                self.ctx.ggt_integrate(vol, tgt, views, depths, flags)
                self.ctx.ggt_extract_depth(vol, depth, conf, bins)
            res.append(dict(target=tgt, views=vi, depths=depths, vol=vol, depth=depth, conf=conf, bins=bins))
        torch.cuda.synchronize()
        return res


def compare_frame(o, g, z_bins, tau, label=""):
    """Element-wise comparison of one target's oracle result `o` with the CUDA result `g`."""
    import torch
    rays = o["rays"]
    T, W = g["vol"].ggt_volume_export()
    if rays is not None:
        sel = torch.from_numpy(rays.astype(np.int64)).cuda()
        T, W = T[sel], W[sel]
        depth, conf, bins = g["depth"][sel], g["conf"][sel], g["bins"][sel]
    else:
        depth, conf, bins = g["depth"], g["conf"], g["bins"]
    T, W = T.cpu().numpy(), W.cpu().numpy()
    depth, conf, bins = depth.cpu().numpy(), conf.cpu().numpy(), bins.cpu().numpy()
    stats = {}
    # TSDF / weight: 1e-5 relative (absolute floor 1e-6 * tau for T near zero, north_star's exemption)
    dT = np.abs(T - o["T"])
    tolT = 1e-5 * np.abs(o["T"]) + 1e-6 * tau[None, :]
    stats["T_bad"] = int((dT > tolT).sum())
    stats["W_bad"] = int((np.abs(W - o["W"]) > 1e-5 * np.abs(o["W"])).sum())
    stats["T_bitexact"] = bool(np.array_equal(T.view(np.uint32), o["T"].view(np.uint32)))
    stats["W_bitexact"] = bool(np.array_equal(W.view(np.uint32), o["W"].view(np.uint32)))
    # zero-crossing bin: bit-exact except where |tsdf| < 1e-6 at the crossing pair
    diff = bins != o["bins"]
    if diff.any():
        r = np.nonzero(diff)[0]
        j = np.clip(np.maximum(bins[r], o["bins"][r]), 0, len(z_bins) - 2)
        near0 = (np.abs(o["T"][r, j]) < 1e-6) | (np.abs(o["T"][r, j + 1]) < 1e-6)
        stats["bin_bad"] = int((~near0).sum())
    else:
        stats["bin_bad"] = 0
    stats["bin_equal"] = bool(not diff.any())
    rng = float(z_bins[-1] - z_bins[0])
    same = ~diff
    stats["depth_bad"] = int((np.abs(depth - o["depth"])[same] > 1e-4 * rng).sum())
    stats["conf_bad"] = int((np.abs(conf - o["conf"])[same] > 1e-5 * np.abs(o["conf"][same]) + 1e-7).sum())
    stats["depth_bitexact"] = bool(np.array_equal(depth.view(np.uint32), o["depth"].view(np.uint32)))
    stats["hit_frac"] = float((o["bins"] >= 0).mean())
    stats["label"] = label
    return stats


def assert_parity(stats):
    assert stats["T_bad"] == 0 and stats["W_bad"] == 0, stats
    assert stats["bin_bad"] == 0, stats
    assert stats["depth_bad"] == 0 and stats["conf_bad"] == 0, stats
