"""The hot path under CUDA-graph capture: a frame (refine each view, integrate into a persistent volume, extract) is
captured once and replayed with new input contents; every replay must match the eager calls and the oracle bit for bit.

Capture needs calls that neither allocate nor synchronise: the {depth, omega} workspace is reserved up front
(ggt_set_workspace), the refine step runs through ggt_refine_depth_static (scratch in the library's fixed device array),
and stage profiling stays off.  Launch-bound frames gain the most (a 64 x 48 frame: 0.056 -> 0.012 ms on a B200).
"""
import numpy as np
import pytest

import helpers
import oracle
from paper_2505_18932_b200 import synth

pytestmark = pytest.mark.gpu


def _inputs(W, H, V, frames, seed):
    wl = synth.workload("C2", scale=0.2)
    rig = synth.grid_rig(W, H)
    tgt = synth.camera_from_pose((0.04, -0.03, 0.01), synth.rot_yaw_pitch(0.02, 0.01), 0.8 * W, 0.8 * W, W / 2, H / 2, W, H)
    views = [rig[i] for i in synth.nearest_views(tgt, rig, V)]
    rng = np.random.default_rng(seed)
    base = [rng.integers(0, 256, (H, W, 3), dtype=np.uint8) for _ in range(V)]
    data = []
    for f in range(frames):
        fr = []
        for k, c in enumerate(views):
            d = synth.noisy_depth(synth.raycast(c, wl.scene)[0], seed + f, k, 0.01, 0.03)
            rgb = np.clip(base[k].astype(np.int16) + rng.integers(-1, 2, base[k].shape), 0, 255).astype(np.uint8)
            x, y = rng.integers(0, W - 40), rng.integers(0, H - 40)
            rgb[y:y + 30, x:x + 36] = np.clip(rgb[y:y + 30, x:x + 36].astype(np.int16) + 60, 0, 255).astype(np.uint8)
            fr.append((d, rgb))
        data.append(fr)
    return tgt, views, data


@pytest.mark.parametrize("dtype_name", ["f32", "f16"])
def test_captured_frame_replays_bit_exact(dtype_name):
    import torch
    from paper_2505_18932_b200 import binding
    W, H, V, D, frames = 200, 136, 4, 48, 4
    tgt, views, data = _inputs(W, H, V, frames, 4242)
    z = synth.bins_inverse(0.5, 5, D)
    tau = oracle.tau_table(z, 2.0)
    dt = binding.GGT_F16 if dtype_name == "f16" else binding.GGT_F32
    n = W * H

    def make():
        ctx = binding.Context()
        ctx.ggt_set_workspace(V, W, H)
        vol = ctx.ggt_volume_bind(W, H, z, dtype=dt, weight_cap=0.5)
        vol.ggt_volume_reset()
        buf = dict(rgb_cur=[torch.empty((H, W, 3), dtype=torch.uint8, device="cuda") for _ in range(V)],
                   rgb_prev=[torch.empty((H, W, 3), dtype=torch.uint8, device="cuda") for _ in range(V)],
                   depth=[torch.empty((H, W), dtype=torch.float32, device="cuda") for _ in range(V)],
                   state=[torch.from_numpy(data[0][k][0]).cuda() for k in range(V)],
                   out=torch.empty(n, dtype=torch.float32, device="cuda"), conf=torch.empty(n, dtype=torch.float32, device="cuda"),
                   bins=torch.empty(n, dtype=torch.int32, device="cuda"))
        return ctx, vol, buf

    def load(buf, f):                      # new contents into the buffers the graph was captured on
        for k in range(V):
            buf["rgb_cur"][k].copy_(torch.from_numpy(data[f][k][1]))
            buf["rgb_prev"][k].copy_(torch.from_numpy(data[f - 1][k][1]))
            buf["depth"][k].copy_(torch.from_numpy(data[f][k][0]))

    def frame(ctx, vol, buf):
        for k in range(V):
            ctx.ggt_refine_depth_static(buf["rgb_cur"][k], buf["rgb_prev"][k], buf["depth"][k], buf["state"][k], **helpers.REFINE)
        ctx.ggt_integrate(vol, tgt, views, buf["state"], binding.GGT_ACCUMULATE)
        ctx.ggt_extract_depth(vol, buf["out"], buf["conf"], buf["bins"])

    # eager run and the oracle, frame by frame
    ctx_e, vol_e, buf_e = make()
    o_state = [data[0][k][0].copy() for k in range(V)]
    T = Wt = None
    eager = []
    for f in range(1, frames):
        load(buf_e, f)
        frame(ctx_e, vol_e, buf_e)
        torch.cuda.synchronize()
        for k in range(V):
            o_state[k] = oracle.refine(data[f][k][1], data[f - 1][k][1], data[f][k][0], o_state[k], **helpers.REFINE)[0]
        maps = [oracle.weight_map(d) for d in o_state]
        T, Wt = oracle.integrate(tgt, z, tau, views, maps, T=T, Wt=Wt, accumulate=True, cap=0.5, half_storage=dtype_name == "f16")
        od, oc, ob = oracle.extract(z, T, Wt)
        st = helpers.compare_frame(dict(rays=None, T=T, W=Wt, depth=od, conf=oc, bins=ob),
                                   dict(vol=vol_e, depth=buf_e["out"], conf=buf_e["conf"], bins=buf_e["bins"]), z, tau)
        helpers.assert_parity(st)
        eager.append((buf_e["out"].clone(), buf_e["conf"].clone(), buf_e["bins"].clone(), [s.clone() for s in buf_e["state"]]))
    assert float(Wt.max()) == 0.5                      # the cap binds by the last frame: the replays are stateful

    # captured once (on frame 1's contents, executed once as the warm-up the capture needs), replayed per frame
    ctx_g, vol_g, buf_g = make()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        load(buf_g, 1)
        frame(ctx_g, vol_g, buf_g)                     # warm-up (also looks up the static scratch address)
        vol_g.ggt_volume_reset()
        for k in range(V):
            buf_g["state"][k].copy_(torch.from_numpy(data[0][k][0]))
        s.synchronize()
        launches = ctx_g.launch_count
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            frame(ctx_g, vol_g, buf_g)
        assert ctx_g.launch_count - launches == 2 * V + 3      # refine 2 per view, weight maps, integrate, extract
    torch.cuda.synchronize()
    # capture executes nothing: the volume is still empty
    Tg, Wg = vol_g.ggt_volume_export()
    torch.cuda.synchronize()
    assert not bool(Tg.any()) and not bool(Wg.any())
    for f in range(1, frames):
        load(buf_g, f)
        g.replay()
        torch.cuda.synchronize()
        e_out, e_conf, e_bins, e_state = eager[f - 1]
        assert torch.equal(buf_g["out"].view(torch.int32), e_out.view(torch.int32)), "depth differs at frame %d" % f
        assert torch.equal(buf_g["conf"].view(torch.int32), e_conf.view(torch.int32)), "conf differs at frame %d" % f
        assert torch.equal(buf_g["bins"], e_bins)
        for k in range(V):
            assert torch.equal(buf_g["state"][k].view(torch.int32), e_state[k].view(torch.int32))
    Te, We = vol_e.ggt_volume_export()
    Tg, Wg = vol_g.ggt_volume_export()
    torch.cuda.synchronize()
    assert torch.equal(Te.view(torch.int32), Tg.view(torch.int32)) and torch.equal(We.view(torch.int32), Wg.view(torch.int32))
