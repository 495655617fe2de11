"""GPU-vs-oracle parity through the C ABI (-m gpu): the five BASELINE.json configs plus edge cases.

Every case feeds the same seeded synthetic inputs (paper_2505_18932_b200.synth) to the oracle and to
libggt.so and compares element by element with north_star's tolerances (tests/helpers.py).  Small /
scaled cases compare every ray; full-size cases compare a seeded ray subset (rays are independent).
"""
import ctypes

import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth
import helpers

pytestmark = pytest.mark.gpu


def run_config(name, scale, frames, every, fused=False, expect_hits=0.5):
    wl = synth.workload(name, scale=scale)
    op = helpers.OraclePipeline(wl, rays_every=every)
    gp = helpers.CudaPipeline(wl, fused=fused)
    all_stats = []
    for f in frames:
        ores, gres = op.frame(f), gp.frame(f)
        for slot, (o, g) in enumerate(zip(ores, gres)):
            st = helpers.compare_frame(o, g, wl.z_bins, op.tau, label="%s f%d t%d" % (name, f, slot))
            helpers.assert_parity(st)
            all_stats.append(st)
    assert np.mean([s["hit_frac"] for s in all_stats]) > expect_hits
    return all_stats


# ---- the kernel's own reciprocal / division against IEEE (determinism contract P14) -----------------------
def test_fast_reciprocal_and_division():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    # every float from 1e-6 (the validity threshold on w) up to 2^24, in chunks
    lo = int(np.float32(1e-6).view(np.uint32)) & ~1
    hi = int(np.float32(16777216.0).view(np.uint32))
    g = torch.Generator(device="cuda").manual_seed(7)
    total = 0
    for start in range(lo, hi, 1 << 26):
        bits = torch.arange(start, min(start + (1 << 26), hi), dtype=torch.int32, device="cuda")
        b = bits.view(torch.float32)
        # numerators: |a| <= 16 * b-ish magnitudes as in a weighted mean, random sign, plus exact zeros
        a = (torch.rand(b.shape, generator=g, device="cuda") * 2 - 1) * b * 0.3
        a[::97] = 0.0
        r, q, sq, c49 = ctx.ggt_selftest_arith(a, b)
        assert r == 0 and q == 0 and sq == 0 and c49 == 0, (start, r, q, sq, c49)
        total += b.numel()
    assert total > 3e8
    # weights and numerators in the ranges the TSDF tail sees: Wn in [0.05, 16], |A| <= tau * Wn
    b = torch.rand(1 << 24, generator=g, device="cuda") * 16 + 0.05
    a = (torch.rand(1 << 24, generator=g, device="cuda") * 2 - 1) * b * 0.25
    assert ctx.ggt_selftest_arith(a, b) == (0, 0, 0, 0)
    # quotients up to magnitude 1 (unit vectors: |v_i| <= |v|), denominators over 12 decades
    b = torch.exp(torch.rand(1 << 24, generator=g, device="cuda") * 28.0 - 14.0)
    a = (torch.rand(1 << 24, generator=g, device="cuda") * 2 - 1) * b
    a[::5] = b[::5]
    assert ctx.ggt_selftest_arith(a, b) == (0, 0, 0, 0)
    # the ranges Eq. 11-12 sees: nu in [1e-16, 49 * clip^2], nu / 49, its square root
    b = torch.exp(torch.rand(1 << 24, generator=g, device="cuda") * 34.0 - 37.0)            # 1e-16 .. 0.05
    a = torch.full_like(b, 0.001)
    assert ctx.ggt_selftest_arith(a, b) == (0, 0, 0, 0)


# ---- refine (a1-a2) ---------------------------------------------------------------------------------
@pytest.mark.parametrize("W,H,stride", [(64, 48, 3), (200, 136, 3), (203, 131, 3), (132, 70, 4), (1920, 1080, 3)])
def test_refine_parity(W, H, stride):
    import torch
    from paper_2505_18932_b200 import binding
    rng = np.random.default_rng(W * 1000 + H)
    prev = rng.integers(0, 256, (H, W, stride), dtype=np.uint8)
    cur = prev.copy()
    # static noise of +-1 everywhere, a few changed blobs of varying strength, one saturated region
    cur = np.clip(cur.astype(np.int16) + rng.integers(-1, 2, cur.shape), 0, 255).astype(np.uint8)
    for _ in range(12):
        x, y = rng.integers(0, W), rng.integers(0, H)
        w, h, amp = rng.integers(2, 40), rng.integers(2, 40), rng.integers(2, 120)
        blk = cur[y:y + h, x:x + w].astype(np.int16) + amp
        cur[y:y + h, x:x + w] = np.clip(blk, 0, 255).astype(np.uint8)
    d = rng.uniform(0.5, 5, (H, W)).astype(np.float32)
    s = rng.uniform(0.5, 5, (H, W)).astype(np.float32)
    d[rng.uniform(size=(H, W)) < 0.05] = 0
    s[rng.uniform(size=(H, W)) < 0.05] = 0
    for theta in (0.0, 8.0 / 255.0):
        o_out, o_M, o_pq, _ = oracle.refine(cur, prev, d, s, theta=theta)
        ctx = binding.Context()
        st = torch.from_numpy(s.copy()).cuda()
        M = torch.empty((H, W), dtype=torch.float32, device="cuda")
        pq = torch.zeros(((H + 3) // 4, (W + 3) // 4), dtype=torch.uint16, device="cuda")
        ctx.ggt_refine_depth(torch.from_numpy(cur).cuda(), torch.from_numpy(prev).cuda(), torch.from_numpy(d).cuda(),
                             st, mask_out=M, pooled_out=pq, theta=theta)
        torch.cuda.synchronize()
        assert np.array_equal(pq.cpu().numpy(), o_pq)                                   # integer: bit-exact
        assert np.array_equal(M.cpu().numpy().view(np.uint32), o_M.view(np.uint32))     # mask: bit-exact
        assert np.array_equal(st.cpu().numpy().view(np.uint32), o_out.view(np.uint32))
        assert (o_M == 1).any() and (o_M < 1).any()
    # first frame
    st = torch.zeros((H, W), dtype=torch.float32, device="cuda")
    ctx.ggt_refine_depth(None, None, torch.from_numpy(d).cuda(), st, mask_out=M)
    assert np.array_equal(st.cpu().numpy(), d) and bool((M == 1).all())


# ---- the five configs --------------------------------------------------------------------------------
def test_C1_full():
    st = run_config("C1", 1.0, [0], 1)
    assert st[0]["T_bitexact"] and st[0]["W_bitexact"] and st[0]["bin_equal"] and st[0]["depth_bitexact"], st


def test_C2_full():
    st = run_config("C2", 1.0, [0], 1)
    assert st[0]["T_bitexact"] and st[0]["W_bitexact"] and st[0]["bin_equal"], st


def test_C2_fused_equals_separate():
    run_config("C2", 0.5, [0], 1, fused=True)


def test_C3_scaled_video_all_rays():
    # 480x272, 12 frames: covers the target re-draw at frame 10 and the per-camera refine history
    run_config("C3", 0.25, list(range(12)), 1)


def test_C3_full_size_sampled():
    run_config("C3", 1.0, [0, 1, 2], 64)


def test_C4_scaled_persistent_fp16_all_rays():
    st = run_config("C4", 0.25, list(range(8)), 1)
    assert all(s["T_bitexact"] and s["W_bitexact"] for s in st), st


def test_C4_full_size_sampled():
    run_config("C4", 1.0, [0, 1, 2], 64)


def test_C5_scaled_batched_targets_all_rays():
    run_config("C5", 0.125, [0, 1, 2], 1, expect_hits=0.2)   # 90-degree targets see beyond the rig's coverage


def test_C5_full_size_sampled():
    # 8 persistent fp32 volumes of 2048 x 2048 x 128 (34.4 GB), 1/512 of the rays, 2 frames
    run_config("C5", 1.0, [0, 1], 512, expect_hits=0.2)


def test_fused_persistent_fp16_matches():
    run_config("C4", 0.25, [0, 1, 2], 1, fused=True)


# ---- edge cases ------------------------------------------------------------------------------------------
def _simple(n_views, D, dtype_name, W=70, H=37, invalid=False, seed=11, accumulate=False, frames=1, fused=False):
    """Random rig around the origin, arbitrary (ragged) sizes and view counts."""
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C2", scale=0.2)
    rig = synth.grid_rig(W + 13, H + 6)
    tgt = synth.camera_from_pose((0.04, -0.03, 0.01), synth.rot_yaw_pitch(0.02, 0.01), 0.8 * W, 0.8 * W, W / 2, H / 2, W, H)
    vi = synth.nearest_views(tgt, rig, n_views)
    views = [rig[i] for i in vi]
    z = synth.bins_inverse(0.5, 5, D)
    tau = oracle.tau_table(z, 2.0)
    ctx = binding.Context()
    vol = ctx.ggt_volume_bind(W, H, z, dtype=binding.GGT_F16 if dtype_name == "f16" else binding.GGT_F32)
    vol.ggt_volume_reset()
    T = Wt = None
    for f in range(frames):
        depths = []
        for i, c in enumerate(views):
            d = synth.noisy_depth(synth.raycast(c, wl.scene)[0], seed + f, i, 0.01, 0.03)
            if invalid:
                d[:] = 0
            depths.append(d)
        maps = [oracle.weight_map(d) for d in depths]
        T, Wt = oracle.integrate(tgt, z, tau, views, maps, T=T if accumulate else None, Wt=Wt if accumulate else None,
                                 accumulate=accumulate, half_storage=dtype_name == "f16")
        od, oc, ob = oracle.extract(z, T, Wt)
        gd = [torch.from_numpy(d).cuda() for d in depths]
        n = W * H
        depth = torch.empty(n, dtype=torch.float32, device="cuda")
        conf = torch.empty(n, dtype=torch.float32, device="cuda")
        bins = torch.empty(n, dtype=torch.int32, device="cuda")
        flags = binding.GGT_ACCUMULATE if accumulate else binding.GGT_OVERWRITE
        if fused:
            ctx.ggt_integrate_extract(vol, tgt, views, gd, flags, depth, conf, bins)
        else:
            ctx.ggt_integrate(vol, tgt, views, gd, flags)
            ctx.ggt_extract_depth(vol, depth, conf, bins)
        o = dict(rays=None, T=T, W=Wt, depth=od, conf=oc, bins=ob)
        g = dict(vol=vol, depth=depth, conf=conf, bins=bins)
        st = helpers.compare_frame(o, g, z, tau)
        helpers.assert_parity(st)
    return st, ob


@pytest.mark.parametrize("n_views", [1, 2, 3, 5, 7, 9, 16])
def test_view_counts(n_views):
    st, _ = _simple(n_views, 24, "f32")
    assert st["T_bitexact"]


@pytest.mark.parametrize("n_views", [3, 5, 6, 7, 9, 12])
@pytest.mark.parametrize("dtype_name,accumulate,fused", [("f16", True, False), ("f32", True, True), ("f16", False, True)])
def test_view_counts_all_kernel_variants(n_views, dtype_name, accumulate, fused):
    """odd view counts run the pipelined march with a ragged last unit: every storage / mode / fused variant"""
    _simple(n_views, 22, dtype_name, accumulate=accumulate, frames=2 if accumulate else 1, fused=fused)


@pytest.mark.parametrize("D,dtype_name", [(2, "f32"), (3, "f32"), (33, "f32"), (5, "f16"), (33, "f16"), (130, "f16")])
def test_ragged_bins(D, dtype_name):
    _simple(4, D, dtype_name)


def test_all_invalid_inputs_give_empty_volume():
    st, ob = _simple(4, 16, "f32", invalid=True)
    assert np.all(ob == -1)


@pytest.mark.parametrize("dtype_name", ["f32", "f16"])
def test_accumulate_small(dtype_name):
    _simple(4, 20, dtype_name, accumulate=True, frames=4)


def test_max_bins_and_error_codes():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    z = synth.bins_inverse(0.5, 5, 1024)
    vol = ctx.ggt_volume_bind(33, 9, z)
    vol.ggt_volume_reset()
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 16.5, 4.5, 33, 9)
    d = torch.full((9, 33), 2.0, device="cuda")
    ctx.ggt_integrate(vol, cam, [cam], [d])
    depth = torch.empty(33 * 9, device="cuda")
    ctx.ggt_extract_depth(vol, depth)
    assert torch.allclose(depth, torch.full_like(depth, 2.0), rtol=2e-6)
    # errors: too many bins, mismatching target, bad flags, zero views
    with pytest.raises(binding.GgtError):
        ctx.ggt_volume_bind(8, 8, synth.bins_inverse(0.5, 5, 1025))
    with pytest.raises(binding.GgtError):
        ctx.ggt_volume_bind(8, 8, np.array([1.0, 0.9, 2.0], np.float32))
    other = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 16, 4, 32, 8)
    with pytest.raises(binding.GgtError):
        ctx.ggt_integrate(vol, other, [cam], [d])
    with pytest.raises(binding.GgtError):
        ctx.ggt_integrate(vol, cam, [cam], [d], flags=7)
    with pytest.raises(binding.GgtError):
        ctx.ggt_refine_depth(None, None, d, d.clone(), downscale=2)
    assert "downscale" in ctx.lib.ggt_last_error(ctx.h).decode()


def test_frame_host_matches_device_path():
    """ggt_frame_host (host buffers, copies inside) gives what the device-pointer calls give."""
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C3", scale=0.25)
    gp = helpers.CudaPipeline(wl)
    ctx = binding.Context()
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    views = [wl.rig[v] for v in vi]
    H, W = views[0].height, views[0].width
    vol = ctx.ggt_volume_bind(tgt.width, tgt.height, wl.z_bins)
    n_slots = len(wl.rig)
    nbytes = ctx.lib.ggt_frame_staging_bytes(ctypes.byref(vol.desc), n_slots, len(vi), W, H)
    staging = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    state = np.zeros(n_slots, np.uint32)
    hd = torch.empty(tgt.height * tgt.width, dtype=torch.float32).pin_memory()
    hc = torch.empty(tgt.height * tgt.width, dtype=torch.float32).pin_memory()
    prm = binding.ggt_refine_params(0.7, 0.6, 8.0 / 255.0, 4, 3)
    for f in range(3):
        ref = gp.frame(f)[0]
        ins = [wl.view_inputs(f, v) for v in vi]
        rgb = [torch.from_numpy(r).pin_memory() for _, r in ins]
        dep = [torch.from_numpy(d).pin_memory() for d, _ in ins]
        ctx.ggt_frame_host(vol, tgt, views, rgb, dep, vi, state, staging, hd, hc, refine_params=prm)
        torch.cuda.synchronize()
        assert torch.equal(hd, ref["depth"].cpu()) and torch.equal(hc, ref["conf"].cpu())
    assert (hd > 0).float().mean() > 0.5


def test_frame_host_pipelined_without_host_sync():
    """Frames enqueued back to back with no synchronise in between (ggt_frame_host uploads frame n + 1 on its own copy
    stream while frame n computes) give, frame by frame, what the device-pointer calls give."""
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C3", scale=0.25)
    gp = helpers.CudaPipeline(wl)
    ctx = binding.Context()
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    views = [wl.rig[v] for v in vi]
    H, W = views[0].height, views[0].width
    vol = ctx.ggt_volume_bind(tgt.width, tgt.height, wl.z_bins)
    n_slots = len(wl.rig)
    nbytes = ctx.lib.ggt_frame_staging_bytes(ctypes.byref(vol.desc), n_slots, len(vi), W, H)
    staging = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    state = np.zeros(n_slots, np.uint32)
    prm = binding.ggt_refine_params(0.7, 0.6, 8.0 / 255.0, 4, 3)
    F = 6
    n = tgt.height * tgt.width
    outs = [(torch.empty(n, dtype=torch.float32).pin_memory(), torch.empty(n, dtype=torch.float32).pin_memory()) for _ in range(F)]
    ins = [[wl.view_inputs(f, v) for v in vi] for f in range(F)]
    rgb = [[torch.from_numpy(r).pin_memory() for _, r in fr] for fr in ins]
    dep = [[torch.from_numpy(d).pin_memory() for d, _ in fr] for fr in ins]
    torch.cuda.synchronize()
    for f in range(F):                                   # no synchronise inside the loop
        ctx.ggt_frame_host(vol, tgt, views, rgb[f], dep[f], vi, state, staging, outs[f][0], outs[f][1], refine_params=prm)
    torch.cuda.synchronize()
    refs = [gp.frame(f)[0] for f in range(F)]
    refs = [(r["depth"].cpu(), r["conf"].cpu()) for r in refs]
    for f in range(F):
        assert torch.equal(outs[f][0], refs[f][0]) and torch.equal(outs[f][1], refs[f][1]), "frame %d" % f
    # the same stream of frames with the result copies on the context's own stream (GGT_FRAME_RESULTS_ASYNC): the caller's
    # stream is synchronised only after ggt_frame_host_results_wait; two host result buffers alternate
    ctx2 = binding.Context()
    vol2 = ctx2.ggt_volume_bind(tgt.width, tgt.height, wl.z_bins)
    state2 = np.zeros(n_slots, np.uint32)
    two = [(torch.empty(n, dtype=torch.float32).pin_memory(), torch.empty(n, dtype=torch.float32).pin_memory()) for _ in range(2)]
    got = []
    for f in range(F):
        ctx2.ggt_frame_host(vol2, tgt, views, rgb[f], dep[f], vi, state2, staging, two[f & 1][0], two[f & 1][1],
                            flags=binding.GGT_OVERWRITE | binding.GGT_FRAME_RESULTS_ASYNC, refine_params=prm)
        if f % 2 == 1:                                   # read both buffers back every second frame
            ctx2.ggt_frame_host_results_wait()
            torch.cuda.current_stream().synchronize()
            got += [(two[0][0].clone(), two[0][1].clone()), (two[1][0].clone(), two[1][1].clone())]
    for f in range(F):
        assert torch.equal(got[f][0], refs[f][0]) and torch.equal(got[f][1], refs[f][1]), "async frame %d" % f
    # duplicate history slots in one call are rejected, and a failed call leaves the slot state untouched
    before = state2.copy()
    with pytest.raises(binding.GgtError):
        ctx2.ggt_frame_host(vol2, tgt, views, rgb[0], dep[0], [vi[0]] * len(vi), state2, staging, two[0][0], two[0][1], refine_params=prm)
    assert np.array_equal(before, state2)


def test_refine_batch_equals_per_view_and_oracle():
    """ggt_refine_depth_batch (all views of a frame in two launches) = the per-view call = the oracle, including a view
    without history (first-frame rule) in the same batch."""
    import torch
    from paper_2505_18932_b200 import binding
    H, W, V = 136, 200, 5
    rng = np.random.default_rng(42)
    ctx = binding.Context()
    cur, prev, dep, st0 = [], [], [], []
    for k in range(V):
        p = rng.integers(0, 256, (H, W, 3), dtype=np.uint8)
        c = np.clip(p.astype(np.int16) + rng.integers(-1, 2, p.shape), 0, 255).astype(np.uint8)
        c[20 + 10 * k:60 + 10 * k, 30:90] = np.clip(c[20 + 10 * k:60 + 10 * k, 30:90].astype(np.int16) + 40 + 20 * k, 0, 255).astype(np.uint8)
        cur.append(c); prev.append(p if k != 2 else None)                 # view 2 has no history
        d = rng.uniform(0.5, 5, (H, W)).astype(np.float32); d[rng.uniform(size=(H, W)) < 0.05] = 0
        s = rng.uniform(0.5, 5, (H, W)).astype(np.float32); s[rng.uniform(size=(H, W)) < 0.05] = 0
        dep.append(d); st0.append(s)
    theta = 8.0 / 255.0
    g = lambda a: None if a is None else torch.from_numpy(a).cuda()
    states = [g(s.copy()) for s in st0]
    masks = [torch.empty((H, W), dtype=torch.float32, device="cuda") for _ in range(V)]
    ctx.ggt_refine_depth_batch([g(c) for c in cur], [g(p) for p in prev], [g(d) for d in dep], states, mask_out=masks, theta=theta)
    torch.cuda.synchronize()
    for k in range(V):
        if prev[k] is None:
            o_out, o_M = dep[k], np.ones((H, W), np.float32)
        else:
            o_out, o_M, _, _ = oracle.refine(cur[k], prev[k], dep[k], st0[k], theta=theta)
        assert np.array_equal(states[k].cpu().numpy().view(np.uint32), o_out.view(np.uint32)), k
        assert np.array_equal(masks[k].cpu().numpy().view(np.uint32), o_M.view(np.uint32)), k


def test_integrate_batch_equals_per_target_calls():
    """ggt_integrate_batch (8 targets of a C5-shaped frame, weight maps computed once) leaves every volume exactly as
    per-target ggt_integrate calls do, over two accumulated frames."""
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C5", scale=0.125)
    ctx_a, ctx_b = binding.Context(), binding.Context()
    targets = wl.targets(0)
    vis = [wl.views_for(t) for t in targets]
    ids = sorted(set(v for vi in vis for v in vi))
    pos = {v: i for i, v in enumerate(ids)}
    rig_views = [wl.rig[v] for v in ids]
    mk = lambda c: [c.ggt_volume_bind(t.width, t.height, wl.z_bins, weight_cap=wl.weight_cap) for t in targets]
    va, vb = mk(ctx_a), mk(ctx_b)
    for v in va + vb:
        v.ggt_volume_reset()
    for f in range(2):
        dep = {v: torch.from_numpy(wl.view_inputs(f, v)[0]).cuda() for v in ids}
        ctx_a.ggt_integrate_batch(va, targets, rig_views, [dep[v] for v in ids], [[pos[v] for v in vi] for vi in vis],
                                  binding.GGT_ACCUMULATE)
        for t, vi, vol in zip(targets, vis, vb):
            ctx_b.ggt_integrate(vol, t, [wl.rig[v] for v in vi], [dep[v] for v in vi], binding.GGT_ACCUMULATE)
    torch.cuda.synchronize()
    for a, b in zip(va, vb):
        Ta, Wa = a.ggt_volume_export()
        Tb, Wb = b.ggt_volume_export()
        assert torch.equal(Ta, Tb) and torch.equal(Wa, Wb)
    assert float((Wa > 0).float().mean()) > 0.1
    # the fused batch gives the same volumes plus what ggt_extract_depth gives on each of them
    ctx_c = binding.Context()
    vc = mk(ctx_c)
    for v in vc:
        v.ggt_volume_reset()
    n = targets[0].width * targets[0].height
    outs = [[torch.empty(n, device="cuda") for _ in targets] for _ in range(2)]
    bins = [torch.empty(n, dtype=torch.int32, device="cuda") for _ in targets]
    for f in range(2):
        dep = {v: torch.from_numpy(wl.view_inputs(f, v)[0]).cuda() for v in ids}
        ctx_c.ggt_integrate_extract_batch(vc, targets, rig_views, [dep[v] for v in ids], [[pos[v] for v in vi] for vi in vis],
                                          binding.GGT_ACCUMULATE, depth=outs[0], conf=outs[1], bins=bins)
    torch.cuda.synchronize()
    for t, (c, b) in enumerate(zip(vc, vb)):
        Tc, Wc = c.ggt_volume_export()
        Tb, Wb = b.ggt_volume_export()
        assert torch.equal(Tc, Tb) and torch.equal(Wc, Wb)
        d, cf, bn = torch.empty(n, device="cuda"), torch.empty(n, device="cuda"), torch.empty(n, dtype=torch.int32, device="cuda")
        ctx_b.ggt_extract_depth(b, d, cf, bn)
        assert torch.equal(d, outs[0][t]) and torch.equal(cf, outs[1][t]) and torch.equal(bn, bins[t])
    with pytest.raises(binding.GgtError):
        ctx_a.ggt_integrate_batch(va, targets, rig_views, [dep[v] for v in ids], [[99] * len(vis[0])] * len(targets))
