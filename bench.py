#!/usr/bin/env python
"""bench.py — one JSON line for the geometry-guidance hot path on N B200s.

A step = one pass of the whole hot path over one target frame of the workload (default: C3 =
BASELINE.json:configs[2], 1920x1080 target, D = 128 inverse-depth bins, V = 4 input views of 1920x1080):
ggt_refine_depth on each of the V views, ggt_integrate (weight maps + fusion), ggt_extract_depth.
  value     Gvoxel.view/s = W_t*H_t*D*V per step / whole-step device time (inputs resident in HBM)
  e2e       same metric through ggt_frame_host with pinned HOST buffers (H2D of colour + depth, D2H of
            depth + confidence inside the timed region)
  roofline  dominant kernel (integrate main) timed with CUDA events on its stream via ggt_profile_*
  cpu_baseline  the oracle as it stands on one host core: one full step of the same workload
  extra     (rank 0, default workload only) compact legs for C4 and C5 (a few steps each, roofline fractions recomputed
            in the run), the fused call, the paper's own raymarch schedule, features, Eq. 3, the Gaussian forward splat
`--impl reference` times the oracle (tier contract: the reference arm is the oracle): full, unsampled steps.
"""
import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "Gvoxel·view TSDF updates/s"
UNIT = "Gvoxel·view/s"
REFINE = dict(lambda_t=0.7, beta=0.6, theta=8.0 / 255.0)
N_INPUT_FRAMES = 3          # distinct synthetic frames cycled through (prev/cur pairs)
# the roofline time per frame, max(T_bytes at the measured HBM peak, T_fma at peak FP32), as the
# survey derived it (its bytes assume an interleaved {T, W} volume; this build's planar layout moves fewer)
SURVEY_T_ROOF_MS = {"C2": 0.037, "C3": 0.66, "C4": 1.00, "C5": 15.9}
REFERENCE_BUDGET_S = 150.0  # --impl reference: full oracle steps are run while they fit this wall-clock budget


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C2", "C3", "C4", "C5"])
    ap.add_argument("--fused", action="store_true", help="use ggt_integrate_extract instead of integrate + extract")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the extra legs (C4 / C5 / raymarch / splat ...)")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)", {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (pynvml, ~5 ms period)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.005)

    def result(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ----------------------------------------------------------------------------------------------------
# workload set-up (inputs generated on the host by the seeded generator, then made resident in HBM)
# ----------------------------------------------------------------------------------------------------
_WL = {}


def _gen_view(name, frame, view):
    """Worker of the input-synthesis pool: one rig view of one frame (depth, colour)."""
    from paper_2505_18932_b200 import synth
    if name not in _WL:
        _WL[name] = synth.workload(name)
    d, rgb = _WL[name].view_inputs(frame, view)
    return np.array(d), (None if rgb is None else np.array(rgb))


def synth_pool():
    """Fork pool for the analytic ray-casts (CPU, seconds per 1080p view).  Created before CUDA is initialised."""
    import multiprocessing as mp
    world = max(1, int(os.environ.get("WORLD_SIZE", "1")))
    n = min(12, max(1, ((os.cpu_count() or 2) - 2) // world))
    return mp.get_context("fork").Pool(n) if n > 1 else None


class Inputs:
    def __init__(self, name, rank, world, n_frames=N_INPUT_FRAMES, pool=None):
        from paper_2505_18932_b200 import sharding, synth
        self.wl = wl = synth.workload(name)
        self.n_frames = n_frames
        self.frames = sharding.frames_for_rank(rank, world, n_frames)
        self.targets = wl.targets(self.frames[0])                  # C5: 8 targets per frame, else 1
        self.vis = [wl.views_for(t) for t in self.targets]
        self.target, self.vi = self.targets[0], self.vis[0]
        self.views = [wl.rig[v] for v in self.vi]
        self.view_ids = sorted(set(v for vi in self.vis for v in vi))     # each rig view is refined once per frame
        self.multi = len(self.targets) > 1
        jobs = [(name, f, v) for f in self.frames for v in self.view_ids]
        res = pool.starmap(_gen_view, jobs) if pool is not None else [_gen_view(*j) for j in jobs]
        got = dict(zip([(f, v) for _, f, v in jobs], res))
        self.data_by_view = [{v: got[(f, v)] for v in self.view_ids} for f in self.frames]
        self.data = [[d[v] for v in self.vi] for d in self.data_by_view]   # [frame][view] -> (depth, rgb)
        self.W, self.H = self.views[0].width, self.views[0].height
        self.V = len(self.vi)
        self.vv_per_step = float(sum(t.width * t.height * wl.z_bins.size * len(vi) for t, vi in zip(self.targets, self.vis)))

    def describe(self, world):
        wl, t = self.wl, self.target
        return {"workload": "%s (BASELINE.json:configs[%d]): target %dx%d, D=%d inverse-depth bins [0.5,5] m, V=%d views "
                            "of %dx%d from the 16-camera grid rig, %s %s volume, refine=%s"
                            % (wl.name, int(wl.name[1]) - 1, t.width, t.height, wl.z_bins.size, self.V, self.W, self.H,
                               wl.storage, "persistent" if wl.persistent else "overwrite", wl.colour),
                "targets_per_step": len(self.targets), "views": self.V, "bins": int(wl.z_bins.size),
                "parallelism": "independent target streams per GPU x%d (no data-path collective)" % world,
                "l2": "per-step traffic (volume %.2f GB written, its T plane read back) exceeds the 126 MB L2; no explicit flush"
                      % (t.width * t.height * wl.z_bins.size * (4 if wl.storage == "f16" else 8) / 1e9)}


class DeviceRun:
    """Device-resident inputs and the step function (all compute in libggt.so kernels)."""

    def __init__(self, inp, fused):
        import torch
        from paper_2505_18932_b200 import binding
        self.torch, self.b, self.inp, self.fused = torch, binding, inp, fused
        wl = inp.wl
        self.ctx = binding.Context()
        self.ctx.ggt_set_workspace(max(inp.V + 1, len(inp.view_ids)), max(inp.W, inp.target.width), max(inp.H, inp.target.height))   # + the previous output depth (Eq. 3 leg)
        self.vols = []
        for t in inp.targets:
            vol = self.ctx.ggt_volume_bind(t.width, t.height, wl.z_bins,
                                           dtype=binding.GGT_F16 if wl.storage == "f16" else binding.GGT_F32,
                                           trunc_bins=wl.trunc_bins, weight_cap=wl.weight_cap)
            vol.ggt_volume_reset()
            self.vols.append(vol)
        self.vol = self.vols[0]
        if inp.multi:          # [frame][rig view id] -> tensors; every view of the union is refined once per frame
            self.depth_by = [{v: torch.from_numpy(d[v][0]).cuda() for v in inp.view_ids} for d in inp.data_by_view]
            self.rgb_by = [{v: torch.from_numpy(d[v][1]).cuda() for v in inp.view_ids} for d in inp.data_by_view]
            self.state_by = {v: self.depth_by[0][v].clone() for v in inp.view_ids}
            pos = {v: i for i, v in enumerate(inp.view_ids)}
            self.rig_views = [wl.rig[v] for v in inp.view_ids]
            self.view_index = [[pos[v] for v in vi] for vi in inp.vis]
        self.depth_in = [[torch.from_numpy(d).cuda() for d, _ in fr] for fr in inp.data]
        self.rgb_in = [[torch.from_numpy(r).cuda() if r is not None else None for _, r in fr] for fr in inp.data]
        self.state = [self.depth_in[0][k].clone() for k in range(inp.V)]
        n = inp.target.width * inp.target.height
        self.depth = torch.empty(n, dtype=torch.float32, device="cuda")
        self.conf = torch.empty(n, dtype=torch.float32, device="cuda")
        self.flags = binding.GGT_ACCUMULATE if wl.persistent else binding.GGT_OVERWRITE
        self.i = 0

    def step(self):
        inp, ctx = self.inp, self.ctx
        cur = 1 + self.i % (inp.n_frames - 1)
        prev = cur - 1
        self.i += 1
        if inp.multi:
            ids = inp.view_ids
            ctx.ggt_refine_depth_batch([self.rgb_by[cur][v] for v in ids], [self.rgb_by[prev][v] for v in ids],
                                       [self.depth_by[cur][v] for v in ids], [self.state_by[v] for v in ids], **REFINE)
            # the 8 targets of the frame in one batched call: the weight maps of the rig views are computed once
            ctx.ggt_integrate_batch(self.vols, inp.targets, self.rig_views, [self.state_by[v] for v in ids], self.view_index,
                                    self.flags)
            for ti in range(len(inp.targets)):
                ctx.ggt_extract_depth(self.vols[ti], self.depth, self.conf)
            return
        if inp.wl.colour:
            ctx.ggt_refine_depth_batch(self.rgb_in[cur], self.rgb_in[prev], self.depth_in[cur], self.state, **REFINE)
            depths = self.state
        else:
            depths = self.depth_in[cur]
        if self.fused:
            ctx.ggt_integrate_extract(self.vol, inp.target, inp.views, depths, self.flags, self.depth, self.conf)
        else:
            ctx.ggt_integrate(self.vol, inp.target, inp.views, depths, self.flags)
            ctx.ggt_extract_depth(self.vol, self.depth, self.conf)


class HostRun:
    """End-to-end through ggt_frame_host: pinned host inputs/outputs, copies inside the timed region."""

    def __init__(self, inp, dev: DeviceRun):
        import ctypes
        import torch
        self.torch, self.inp, self.dev = torch, inp, dev
        wl = inp.wl
        self.rgb = [[torch.from_numpy(r).pin_memory() if r is not None else None for _, r in fr] for fr in inp.data]
        self.dep = [[torch.from_numpy(d).pin_memory() for d, _ in fr] for fr in inp.data]
        n = inp.target.width * inp.target.height
        self.outs = [(torch.empty(n, dtype=torch.float32).pin_memory(), torch.empty(n, dtype=torch.float32).pin_memory())
                     for _ in range(2)]          # two result buffers: the pipelined leg alternates between them
        self.out_d, self.out_c = self.outs[0]
        nb = dev.ctx.lib.ggt_frame_staging_bytes(ctypes.byref(dev.vol.desc), inp.V, inp.V, inp.W, inp.H)
        self.staging = torch.empty(nb, dtype=torch.uint8, device="cuda")
        self.slot_state = np.zeros(inp.V, np.uint32)
        self.prm = dev.b.ggt_refine_params(REFINE["lambda_t"], REFINE["beta"], REFINE["theta"], 4, 3) if wl.colour else None
        self.h2d = inp.V * (inp.W * inp.H * 4 + (inp.W * inp.H * 3 if wl.colour else 0))
        self.d2h = 2 * n * 4
        self.i = 0

    def step(self, async_results=False):
        inp, dev = self.inp, self.dev
        cur = self.i % inp.n_frames
        self.i += 1
        dev.ctx.ggt_frame_host(dev.vol, inp.target, inp.views, self.rgb[cur] if inp.wl.colour else None, self.dep[cur],
                               list(range(inp.V)), self.slot_state, self.staging, *self.outs[self.i & 1],
                               flags=dev.flags | (dev.b.GGT_FRAME_RESULTS_ASYNC if async_results else 0), refine_params=self.prm)


def timed(torch, dist, fn, steps, warmup):
    """W untimed steps, then exactly K steps between barrier + synchronize, CUDA events on the current stream."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return e0.elapsed_time(e1)


def device_peaks(torch, sampler):
    """SM count and maximum SM clock read on the box: the FP32 and issue-slot peaks derive from them."""
    props = torch.cuda.get_device_properties(torch.cuda.current_device())
    sms = int(props.multi_processor_count)
    mhz = sampler.max_mhz if sampler is not None and sampler.max_mhz else None
    src = "NVML max SM clock"
    if not mhz:
        mhz = float(getattr(props, "clock_rate", 1965000)) / 1e3
        src = "cudaDeviceProp.clockRate"
    hz = float(mhz) * 1e6
    return {"sm_count": sms, "sm_max_mhz": float(mhz), "clock_source": src,
            "fp32_tflops": sms * 128 * 2 * hz / 1e12, "issue_per_s": sms * 4 * hz}


def stage_profile(torch, dev, steps):
    """Per-stage device time of `steps` steps (events around each kernel group on the launching stream)."""
    dev.ctx.ggt_profile_enable(True)
    torch.cuda.synchronize()
    for _ in range(steps):
        dev.step()
    torch.cuda.synchronize()
    prof = dev.ctx.ggt_profile_collect()
    dev.ctx.ggt_profile_enable(False)
    return prof, {k: (v[0] / max(steps, 1)) for k, v in prof.items()}


def roofline_of(inp, prof, stage_ms, fused, hbm_peak, peak_src, peaks):
    """Roofline object of the dominant kernel (k_integrate) plus the north_star quantity integrate + extract."""
    t, wl = inp.target, inp.wl
    voxels = t.width * t.height * wl.z_bins.size
    vox_bytes = voxels * (4 if wl.storage == "f16" else 8)
    map_bytes = inp.V * inp.W * inp.H * 8
    integ_bytes = vox_bytes * (2 if wl.persistent else 1) + map_bytes      # algorithmic: DESIGN.md "Roofline"
    integ_ms = prof["integrate"][0] / max(prof["integrate"][1], 1)
    achieved = integ_bytes / (integ_ms / 1e3) / 1e9 if integ_ms > 0 else 0.0
    nt = len(inp.targets)
    # extract searches the T plane only (half of the volume) and fetches W for the crossing candidates
    path_bytes = (integ_bytes + (0 if fused else vox_bytes // 2) + 2 * t.width * t.height * 4) * nt
    path_ms = stage_ms["integrate"] + stage_ms["extract"]
    vv = inp.vv_per_step
    flops = 16.0 * vv + 12.0 * voxels * nt                               # 16 per voxel.view + 8 + 4 per voxel
    t_bytes_ms = path_bytes / (hbm_peak * 1e9) * 1e3
    t_fma_ms = flops / (peaks["fp32_tflops"] * 1e12) * 1e3
    t_roof = max(t_bytes_ms, t_fma_ms)
    s_roof = SURVEY_T_ROOF_MS.get(wl.name)
    roof = {"bound": "hbm", "kernel": "k_integrate (ggt_integrate main kernel)", "achieved": achieved, "peak": hbm_peak,
            "unit": "GB/s", "frac": achieved / hbm_peak, "traffic": None, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": integ_bytes, "ms_per_launch": integ_ms,
            "integrate_plus_extract": {"bytes": path_bytes, "ms": path_ms,
                                       "frac": (path_bytes / (path_ms / 1e3) / 1e9 / hbm_peak) if path_ms > 0 else 0.0,
                                       "t_bytes_ms": t_bytes_ms, "t_fma_ms": t_fma_ms,
                                       "frac_of_max_tbytes_tfma": t_roof / path_ms if path_ms > 0 else 0.0,
                                       "survey_t_roof_ms": s_roof,
                                       "frac_of_survey_t_roof": (s_roof / path_ms) if path_ms > 0 and s_roof else None},
            "alu": {"flop_per_voxel_view": 16, "achieved_tflops": 16 * vv / nt / (integ_ms / 1e3) / 1e12 if integ_ms > 0 else 0.0,
                    "peak_tflops_at_max_clock": peaks["fp32_tflops"], "sm_count": peaks["sm_count"],
                    "sm_max_mhz": peaks["sm_max_mhz"], "clock_source": peaks["clock_source"]}}
    traffic_file = os.path.join(ROOT, "profiles", "traffic_integrate.json")
    if os.path.exists(traffic_file):
        with open(traffic_file) as fh:
            tj = json.load(fh)
        roof["traffic"] = tj.get(wl.name + ("_fused" if fused else ""))
        roof["traffic_source"] = "profiles/traffic_integrate.json (ncu --set full capture of this kernel; not measured in this run)"
        if roof["traffic"] and integ_ms > 0:
            # DRAM bytes actually moved over this run's kernel time: k_integrate leaves out what it can prove away (views
            # that cannot see a stretch of bins; plane words of unseen bins whose bits do not change are not rewritten), so
            # on wide-angle targets it moves fewer bytes than the algorithmic count and `frac` is an effective rate
            roof["dram_frac"] = roof["traffic"] / (integ_ms / 1e3) / 1e9 / hbm_peak
            if roof["traffic"] < 0.9 * integ_bytes:
                roof["note"] = ("the kernel moves %.2f GB per launch against %.2f GB algorithmic (bins that no view sees and that were "
                                "never observed are read but not rewritten): frac is an effective rate, dram_frac the real one"
                                % (roof["traffic"] / 1e9, integ_bytes / 1e9))
        wi = tj.get(wl.name + "_warp_instructions")
        if wi and not fused and integ_ms > 0:
            # the kernel's practical limit: one warp instruction per SM sub-partition per clock; the instruction count is
            # the ncu-measured one of the committed profile (static for this workload)
            roof["issue"] = {"warp_instructions_per_launch": wi, "peak_warp_instructions_per_s": peaks["issue_per_s"],
                             "frac": wi / peaks["issue_per_s"] / (integ_ms / 1e3)}
    return roof, integ_ms


# ----------------------------------------------------------------------------------------------------
# the oracle, timed as it stands on the host cores (cpu_baseline leg and --impl reference)
# ----------------------------------------------------------------------------------------------------
def oracle_step(inp, cur=1, ray_every=1):
    """One step of the whole path on the CPU oracle, single-threaded: refine + weight maps of the V views, integrate +
    extract of the target (every ray when ray_every = 1).  Returns the wall time and its parts."""
    import oracle
    wl, tgt = inp.wl, inp.target
    t0 = time.perf_counter()
    depths = []
    for k in range(inp.V):
        d, rgb = inp.data[cur][k]
        if wl.colour:
            dp, rp = inp.data[cur - 1][k]
            d = oracle.refine(rgb, rp, d, dp, want_mask=False, **REFINE)[0]
        depths.append(d)
    t1 = time.perf_counter()
    maps = [oracle.weight_map(d) for d in depths]
    t2 = time.perf_counter()
    n = tgt.width * tgt.height
    rays = None if ray_every <= 1 else np.arange(ray_every // 2, n, ray_every, dtype=np.int32)
    tau = oracle.tau_table(wl.z_bins, wl.trunc_bins)
    T, W = oracle.integrate(tgt, wl.z_bins, tau, inp.views, maps, rays=rays, accumulate=wl.persistent,
                            cap=wl.weight_cap, half_storage=wl.storage == "f16")
    oracle.extract(wl.z_bins, T, W)
    t3 = time.perf_counter()
    return t3 - t0, {"refine_s": t1 - t0, "weight_s": t2 - t1, "integrate_extract_s": t3 - t2,
                     "rays": n if rays is None else int(rays.size)}


def cpu_baseline(inp):
    oracle_step(inp, ray_every=64)               # the same untimed page-in pass the reference arm makes
    full, parts = oracle_step(inp)
    return {"value": inp.vv_per_step / full / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "one full %s step, nothing sampled or extrapolated: refine + weight maps of all %d views, integrate + extract "
                      "of all %d target rays; %.1f s of CPU work (refine %.1f, weight maps %.1f, integrate + extract %.1f); host has "
                      "%d cores, the oracle is single-threaded"
                      % (inp.wl.name, inp.V, parts["rays"], full, parts["refine_s"], parts["weight_s"], parts["integrate_extract_s"],
                         os.cpu_count() or 0),
            "ms_per_step": full * 1e3}


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores (rank 0 only), same metric / config; every timed step is a full,
    unsampled step; as many of the requested steps as fit REFERENCE_BUDGET_S are run."""
    if rank != 0:
        return
    t_start = time.perf_counter()
    pool = synth_pool()
    inp = Inputs(args.workload, 0, 1, pool=pool)
    if pool is not None:
        pool.close()
    if inp.multi:
        print(json.dumps({"impl": "reference", "unavailable": "the oracle leg runs the single-target workloads (C2-C4)"}))
        return
    warm = min(args.warmup, 1)
    for _ in range(warm):
        oracle_step(inp, ray_every=64)           # pages the library and the inputs in; not timed
    times, parts = [], None
    while len(times) < max(1, args.steps):
        if times and (time.perf_counter() - t_start) + 1.1 * max(times) > REFERENCE_BUDGET_S:
            break
        dt, parts = oracle_step(inp, cur=1 + len(times) % (inp.n_frames - 1))
        times.append(dt)
    ms = float(np.mean(times)) * 1e3
    value = inp.vv_per_step / (ms / 1e3) / 1e9
    sample = ("each step: one full %s step of the oracle, single-threaded, nothing sampled or extrapolated (refine + weight maps of "
              "all %d views, integrate + extract of all %d rays); %d of the requested %d steps run within the %.0f s budget"
              % (inp.wl.name, inp.V, parts["rays"], len(times), args.steps, REFERENCE_BUDGET_S))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": len(times),
            "steps_requested": args.steps, "steps_run": len(times), "warmup": warm, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": inp.describe(1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "wall_s": time.perf_counter() - t_start}
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------------------
def fused_batch_frame(dev, d8, c8):
    inp, ids = dev.inp, dev.inp.view_ids
    dev.ctx.ggt_refine_depth_batch([dev.rgb_by[1][v] for v in ids], [dev.rgb_by[0][v] for v in ids],
                                   [dev.depth_by[1][v] for v in ids], [dev.state_by[v] for v in ids], **REFINE)
    dev.ctx.ggt_integrate_extract_batch(dev.vols, inp.targets, dev.rig_views, [dev.state_by[v] for v in ids],
                                        dev.view_index, dev.flags, depth=d8, conf=c8)


def compact_leg(torch, name, pool, hbm_peak, peak_src, peaks, steps, warmup):
    """extra.C4 / extra.C5: a few steps of another BASELINE.json config with its roofline fractions recomputed in the run."""
    inp = Inputs(name, 0, 1, n_frames=2, pool=pool)
    dev = DeviceRun(inp, False)
    for _ in range(warmup):
        dev.step()
    launches0 = dev.ctx.launch_count
    ms = timed(torch, None, dev.step, steps, 0) / steps
    launches = (dev.ctx.launch_count - launches0) // steps
    prof, stage_ms = stage_profile(torch, dev, steps)
    roof, integ_ms = roofline_of(inp, prof, stage_ms, False, hbm_peak, peak_src, peaks)
    out = {"config": inp.describe(1)["workload"], "steps": steps, "warmup": warmup, "ms_per_step": ms,
           "ms_per_target": ms / len(inp.targets), "gvoxel_view_per_s": inp.vv_per_step / (ms / 1e3) / 1e9,
           "stages_ms": {"refine_all_views": stage_ms["refine"], "weight_maps": stage_ms["weight"],
                         "integrate": stage_ms["integrate"], "extract": stage_ms["extract"]},
           "k_integrate_ms_per_launch": integ_ms, "gpu_launches_per_step": int(launches), "roofline": roof}
    if inp.multi:
        d8 = [torch.empty_like(dev.depth) for _ in inp.targets]
        c8 = [torch.empty_like(dev.conf) for _ in inp.targets]
        out["fused_batch_frame_ms"] = timed(torch, None, lambda: fused_batch_frame(dev, d8, c8), steps, 1) / steps
    else:
        depths = dev.depth_in[1]
        fused_fn = lambda: dev.ctx.ggt_integrate_extract(dev.vol, inp.target, inp.views, depths, dev.flags, dev.depth, dev.conf)
        out["fused_integrate_extract_ms"] = timed(torch, None, fused_fn, steps, 1) / steps
    del dev
    torch.cuda.empty_cache()
    return out


def splat_leg(torch, binding, wl, k):
    """f-3 at PAPER.md Table 4's shape: K = 4 views of 1352x1014 forward-splatted into a 1352x1014 target."""
    from paper_2505_18932_b200 import synth
    rig = synth.grid_rig(1352, 1014)
    tgt = rig[5]
    vi = synth.nearest_views(tgt, rig, 4, exclude=5)
    ctx = binding.Context()
    ins = []
    for i in vi:
        d, rgb = synth.raycast(rig[i], wl.scene, 0.0, want_colour=True)
        ins.append((rig[i], torch.from_numpy(synth.noisy_depth(d, 1352, i, 0.01, 0.02)).cuda(), torch.from_numpy(rgb).cuda(),
                    torch.full(d.shape, 0.7, dtype=torch.float32, device="cuda")))
    n = 1352 * 1014
    outs = [(torch.empty((3, 1014, 1352), device="cuda"), torch.empty(n, device="cuda"), torch.empty(n, device="cuda"),
             torch.empty(n, device="cuda")) for _ in vi]

    def fn():
        for (cam, d, rgb, m), (o_rgb, o_a, o_d, o_m) in zip(ins, outs):
            ctx.ggt_splat_forward(tgt, cam, d, rgb=rgb, mask=m, out_rgb=o_rgb, out_alpha=o_a, out_depth=o_d, out_mask=o_m)
    ms = timed(torch, None, fn, k, 2) / k
    last, need = ctx.ggt_splat_status()
    return {"call": "ggt_splat_forward x 4 views (PAPER.md:63-67, 362-368): K = 4 views of 1352x1014 into a 1352x1014 target, colour + "
                    "opacity + depth + mask each (the resolution of PAPER.md Table 4's 10 ms forward-splatting stage, GPU not stated)",
            "ms_per_frame_4_views": ms, "ms_per_view": ms / 4, "list_entries_last_view": last, "overflow": need,
            "coverage_last_view": float((outs[-1][1] > 0.5).float().mean().item()), "paper_ms": 10.0}


def main():
    args = parse_args()
    from paper_2505_18932_b200 import sharding
    rank, local_rank, world = sharding.env_rank()
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    # input synthesis (CPU ray-casts) in a fork pool, before CUDA is initialised in this process
    pool = synth_pool()
    inp = Inputs(args.workload, rank, world, pool=pool)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        torch.cuda.set_device(local_rank)
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist = dist_mod
    else:
        torch.cuda.set_device(0)
    import __graft_entry__
    if rank == 0:
        __graft_entry__.build()
    if dist is not None:
        dist.barrier()

    dev = DeviceRun(inp, args.fused)
    host = HostRun(inp, dev) if not inp.multi else None
    hbm_peak, peak_src, _ = measured_peaks()

    # ---- headline: device-resident inputs --------------------------------------------------------------
    sampler = ClockSampler(physical_gpu_index(local_rank))
    peaks = device_peaks(torch, sampler)
    for _ in range(args.warmup):
        dev.step()
    launches_w = dev.ctx.launch_count
    sampler.start()                                 # keeps sampling through the stage-profile and e2e legs below: the
    ms_local = timed(torch, dist, dev.step, args.steps, 0)     # timed region alone lasts only K ms
    samples_timed = len(sampler.samples)
    gpu_launches = dev.ctx.launch_count - launches_w
    red = sharding.reduce_timing(ms_local, inp.vv_per_step * args.steps, device="cuda" if dist is not None else None)
    ms_per_step = red["ms"] / args.steps
    value = red["units"] / (red["ms"] / 1e3) / 1e9

    # ---- per-stage device time of the same step (events around each kernel group, same stream) ---------
    prof, stage_ms = stage_profile(torch, dev, args.steps)
    roofline, integ_ms = roofline_of(inp, prof, stage_ms, args.fused, hbm_peak, peak_src, peaks)
    t, wl = inp.target, inp.wl

    # ---- e2e: host buffers through ggt_frame_host, result needed on the host every step ----------------
    if inp.multi:
        e2e = {"value": None, "unit": UNIT, "note": "ggt_frame_host takes one target per call; the e2e leg runs on the single-target workloads (default C3)"}
    else:
        def e2e_step():
            host.step()
            torch.cuda.current_stream().synchronize()
        e2e_steps = max(3, min(args.steps, 50))
        ms_e2e_local = timed(torch, dist, e2e_step, e2e_steps, max(3, min(args.warmup, 5)))
        red_e = sharding.reduce_timing(ms_e2e_local, inp.vv_per_step * e2e_steps, device="cuda" if dist is not None else None)
        e2e = {"value": red_e["units"] / (red_e["ms"] / 1e3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": host.h2d,
               "d2h_bytes_per_step": host.d2h, "ms_per_step": red_e["ms"] / e2e_steps, "steps": e2e_steps,
               "api": "ggt_frame_host (pinned host buffers, stream synchronised every step)"}
        # the same call without the per-step synchronise: ggt_frame_host uploads frame n + 1 on its own copy stream
        # while frame n's integrate / extract run; results alternate between two pinned buffers, one sync at the end
        # (GGT_FRAME_RESULTS_ASYNC: the result copies run on the context's own stream out of alternating device buffers;
        # the timed region ends once the stream has waited for the last of them)
        left = [3 + e2e_steps]

        def pipe_step():
            host.step(async_results=True)
            left[0] -= 1
            if left[0] == 0:
                dev.ctx.ggt_frame_host_results_wait()
        ms_pipe_local = timed(torch, dist, pipe_step, e2e_steps, 3)
        red_p = sharding.reduce_timing(ms_pipe_local, inp.vv_per_step * e2e_steps, device="cuda" if dist is not None else None)
        e2e["pipelined"] = {"value": red_p["units"] / (red_p["ms"] / 1e3) / 1e9, "unit": UNIT, "ms_per_step": red_p["ms"] / e2e_steps,
                            "note": "same per-step copies, no host synchronise between steps, result copies on the context's stream "
                                    "(GGT_FRAME_RESULTS_ASYNC; throughput of an online stream)"}

    sampler.stop_flag = True
    sampler.join(timeout=2)
    clocks = sampler.result()
    clocks["samples_in_timed_region"] = samples_timed
    clocks["window"] = "the K timed steps, the per-stage pass of K steps and the e2e legs (GPU under load throughout)"
    extra = {}
    do_extra = rank == 0 and not args.no_extra
    # ---- C5 only: the same frame with the zero-crossing search fused into the batch (no volume re-read) ---------
    if do_extra and inp.multi:
        d8 = [torch.empty_like(dev.depth) for _ in inp.targets]
        c8 = [torch.empty_like(dev.conf) for _ in inp.targets]
        kf = max(3, min(args.steps, 10))
        ms_ff = timed(torch, None, lambda: fused_batch_frame(dev, d8, c8), kf, 2) / kf
        extra["fused_batch_frame"] = {"call": "ggt_refine_depth_batch + ggt_integrate_extract_batch (8 targets, no volume re-read)",
                                      "ms_per_frame": ms_ff}

    # ---- extra legs (not the headline): fused integrate+extract, and the paper's own volume-free schedule ------
    if do_extra and not inp.multi:
        k = max(3, min(args.steps, 20))
        depths = dev.state if wl.colour else dev.depth_in[1]
        fused_fn = lambda: dev.ctx.ggt_integrate_extract(dev.vol, inp.target, inp.views, depths, dev.flags, dev.depth, dev.conf)
        ms_f = timed(torch, None, fused_fn, k, 3) / k
        extra["fused_integrate_extract"] = {"ms_per_call": ms_f, "includes": "weight maps + fused integrate/extract kernel (no volume re-read)",
                                            "gvoxel_view_per_s": inp.vv_per_step / (ms_f / 1e3) / 1e9}
        # the same inputs seen by cameras that do NOT share H (a real rig: every camera with its own rotation): view i
        # yawed by 4 (i - 1.5) degrees, every second one pitched by 2 degrees.  The cameras only change the projection the
        # kernel evaluates (the depth maps stay those of the parallel rig: this leg times the march, it renders nothing)
        from paper_2505_18932_b200 import synth as _synth
        turned = [_synth.camera_from_pose(c.centre, _synth.rot_yaw_pitch(math.radians(4.0 * (i - 1.5)), math.radians(2.0 * (i % 2))),
                                          c.fx, c.fy, c.cx, c.cy, c.width, c.height) for i, c in enumerate(inp.views)]
        np_fn = lambda: dev.ctx.ggt_integrate(dev.vol, inp.target, turned, depths, dev.flags)
        for _ in range(3):                                       # the first launch of this kernel loads it
            np_fn()
        dev.ctx.ggt_profile_enable(True)
        timed(torch, None, np_fn, k, 0)
        prof_n = dev.ctx.ggt_profile_collect()
        dev.ctx.ggt_profile_enable(False)
        extra["non_parallel_rig"] = {"call": "ggt_integrate on the step's inputs with every view rotated on its own (no shared H: per-view w and 1/w)",
                                     "k_integrate_ms_per_launch": prof_n["integrate"][0] / max(prof_n["integrate"][1], 1),
                                     "parallel_rig_k_integrate_ms_per_launch": integ_ms}
        n_t = t.width * t.height
        steps_out = torch.zeros(n_t, dtype=torch.int32, device="cuda")
        zn, zf = float(wl.z_bins[0]), float(wl.z_bins[-1])
        rm_fn = lambda: dev.ctx.ggt_raymarch_depth(inp.target, inp.views, depths, zn, zf, depth=dev.depth, conf=dev.conf, steps=steps_out)
        dev.ctx.ggt_profile_enable(True)
        ms_r = timed(torch, None, rm_fn, k, 3) / k
        prof_r = dev.ctx.ggt_profile_collect()
        dev.ctx.ggt_profile_enable(False)
        evals = float(steps_out.sum().item())
        k_ms = prof_r["raymarch"][0] / max(prof_r["raymarch"][1], 1)
        extra["paper_schedule_raymarch"] = {
            "call": "ggt_raymarch_depth (PAPER.md:75, 348: on-the-fly TSDF, advance 0.8 s, 3 bisection steps; tau 0.02 m, "
                    "min_step 1e-3 m), same inputs as the step, no volume",
            "ms_per_call": ms_r, "kernel_ms": k_ms, "evaluations_per_ray_mean": evals / n_t,
            "gsample_view_per_s": evals * inp.V / (k_ms / 1e3) / 1e9 if k_ms > 0 else None,
            "hit_fraction": float((dev.depth > 0).float().mean().item())}
        # the paper's Table 4 shape for the same schedule: target and K = 4 views of 1352 x 1014
        from paper_2505_18932_b200 import synth as _synth
        rig_p = _synth.grid_rig(1352, 1014)
        tgt_p = rig_p[5]
        vi_p = _synth.nearest_views(tgt_p, rig_p, 4, exclude=5)
        views_p = [rig_p[i] for i in vi_p]
        dep_p = [torch.from_numpy(_synth.noisy_depth(_synth.raycast(c, wl.scene)[0], 1352, i, 0.01, 0.02)).cuda()
                 for i, c in enumerate(views_p)]
        n_p = 1352 * 1014
        d_p, c_p = torch.empty(n_p, device="cuda"), torch.empty(n_p, device="cuda")
        s_p = torch.zeros(n_p, dtype=torch.int32, device="cuda")
        ctx_p = dev.b.Context()            # its own context: the step's caller-sized workspace does not fit these views
        rmp_fn = lambda: ctx_p.ggt_raymarch_depth(tgt_p, views_p, dep_p, zn, zf, depth=d_p, conf=c_p, steps=s_p)
        ms_rp = timed(torch, None, rmp_fn, k, 3) / k
        extra["paper_table4_shape"] = {
            "call": "ggt_raymarch_depth, target and K = 4 views of 1352x1014 (the resolution of PAPER.md Table 4's 6 ms TSDF "
                    "stage, GPU not stated), synthetic scene of this workload, weight maps included",
            "ms_per_call": ms_rp, "evaluations_per_ray_mean": float(s_p.sum().item()) / n_p,
            "hit_fraction": float((d_p > 0).float().mean().item())}
        del dep_p, d_p, c_p, s_p, ctx_p
        # f-4: network-input geometry features of the guidance depth just produced
        feats = torch.empty((4 * inp.V, t.height, t.width), dtype=torch.float32, device="cuda")
        gdepth = dev.depth.clone()
        ft_fn = lambda: dev.ctx.ggt_guidance_features(inp.target, gdepth, inp.views, feats)
        ms_ft = timed(torch, None, ft_fn, k, 3) / k
        ft_bytes = n_t * (4 + 16 * inp.V)
        extra["guidance_features"] = {"call": "ggt_guidance_features (PAPER.md:374-388 items 5-8), [4K][H][W] fp32", "ms_per_call": ms_ft,
                                      "algorithmic_bytes": ft_bytes, "frac_of_hbm_peak": ft_bytes / (ms_ft / 1e3) / 1e9 / hbm_peak}
        del feats
        # Eq. 3 (f-2): the previous output depth as a (V+1)-th view with Eq. 13's weight, masks from ggt_refine_depth
        Hv, Wv = inp.H, inp.W
        masks = [torch.full((Hv, Wv), 0.6, dtype=torch.float32, device="cuda") for _ in range(inp.V)]
        if wl.colour:
            for kk in range(inp.V):
                st = dev.depth_in[0][kk].clone()
                dev.ctx.ggt_refine_depth(dev.rgb_in[1][kk], dev.rgb_in[0][kk], dev.depth_in[1][kk], st, mask_out=masks[kk], **REFINE)
        prev_d, prev_c = dev.depth.clone(), dev.conf.clone()
        wmap = torch.empty(n_t, dtype=torch.float32, device="cuda")
        tw_fn = lambda: dev.ctx.ggt_temporal_weight(inp.target, prev_d, prev_c, inp.views, masks, wmap, beta=1.0, eta=15.0)
        ms_tw = timed(torch, None, tw_fn, k, 3) / k
        views5, depths5 = list(inp.views) + [inp.target], list(depths) + [prev_d]
        rm5_fn = lambda: dev.ctx.ggt_raymarch_depth_weighted(inp.target, views5, depths5, [None] * inp.V + [wmap], zn, zf,
                                                            depth=dev.depth, conf=dev.conf, steps=steps_out)
        ms_r5 = timed(torch, None, rm5_fn, k, 3) / k
        extra["paper_temporal_fusion_eq3"] = {
            "call": "ggt_temporal_weight (Eq. 13-14) + ggt_raymarch_depth_weighted with D^{t-1} as view V+1 (Eq. 3)",
            "temporal_weight_ms": ms_tw, "raymarch_weighted_ms_per_call": ms_r5, "views": inp.V + 1,
            "evaluations_per_ray_mean": float(steps_out.sum().item()) / n_t}
        del masks, prev_d, prev_c, wmap
        # f-3: the Gaussian forward splat at Table 4's shape
        extra["gaussian_forward_splat"] = splat_leg(torch, dev.b, wl, max(3, min(args.steps, 10)))

    # ---- the other 1080p / batched configs, a few steps each (default workload, one GPU) -------------------------
    if do_extra and world == 1 and args.workload == "C3":
        host = None
        dev.vols, dev.vol = [], None           # release the C3 volume before the 34 GB of C5
        torch.cuda.empty_cache()
        for name, ks in (("C4", 5), ("C5", 3)):
            try:
                extra[name] = compact_leg(torch, name, pool, hbm_peak, peak_src, peaks, ks, 3)
            except Exception as exc:           # a leg that cannot run (e.g. memory) is reported, never silently dropped
                extra[name] = {"error": repr(exc)}
    if pool is not None:
        pool.close()

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if wl.storage == "f32" else "f32 compute, f16 storage", "data": "synthetic",
                "config": inp.describe(world), "clocks": clocks, "e2e": e2e, "gpu_launches": int(gpu_launches),
                "roofline": roofline,
                "stages_ms": {"refine_all_views": stage_ms["refine"], "weight_maps": stage_ms["weight"],
                              "integrate": stage_ms["integrate"], "extract": stage_ms["extract"],
                              "note": "per-step device time per stage (CUDA events on the launching stream)"},
                "ms_per_1080p_target_frame": ms_per_step,
                "integrate_gvoxel_view_per_s": inp.vv_per_step / len(inp.targets) / (integ_ms / 1e3) / 1e9 if integ_ms > 0 else None,
                "ms_per_target": ms_per_step / len(inp.targets),
                "paper_context": "PAPER.md Table 4: TSDF stage 6 ms/frame, forward splatting 10 ms at 1352x1014, K=4, GPU not stated",
                "extra": extra}
        if not args.no_cpu_baseline and world == 1 and not inp.multi:
            line["cpu_baseline"] = cpu_baseline(inp)
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
