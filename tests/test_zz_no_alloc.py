"""ggt_refine_depth_static (the allocation-free variant of ggt_refine_depth) against ggt_refine_depth, through the C ABI.

The variant keeps Eq. 1's quarter-resolution scratch in a fixed device array of the library instead of the context's
cudaMalloc-ed buffer; the kernels and their arithmetic are the same, so mask, pooled differences and refined depth are
compared bit for bit (the bar every refine test of this repository uses).  The array is shared by all calls and keeps the
last call's contents, so the calls below run back to back, a large frame first and a smaller one after it: a cell read
before it is written would show.  This file sorts last on purpose (pytest -x).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MAX_CELLS = 262144            # GGT_REFINE_STATIC_MAX_CELLS (include/ggt.h)


def _frame(rng, W, H, stride, prev=None):
    if prev is None:
        prev = rng.integers(0, 256, (H, W, stride), dtype=np.uint8)
    cur = np.clip(prev.astype(np.int16) + rng.integers(-1, 2, prev.shape), 0, 255).astype(np.uint8)
    for _ in range(10):
        x, y = rng.integers(0, W), rng.integers(0, H)
        w, h, amp = rng.integers(2, 40), rng.integers(2, 40), rng.integers(2, 120)
        cur[y:y + h, x:x + w] = np.clip(cur[y:y + h, x:x + w].astype(np.int16) + amp, 0, 255).astype(np.uint8)
    d = rng.uniform(0.5, 5, (H, W)).astype(np.float32)
    d[rng.uniform(size=(H, W)) < 0.05] = 0
    return prev, cur, d


def _both(ctx, fn_name, cur, prev, d, state, theta):
    import torch
    H, W = d.shape
    st = state.clone()
    M = torch.empty((H, W), dtype=torch.float32, device="cuda")
    pq = torch.zeros(((H + 3) // 4, (W + 3) // 4), dtype=torch.uint16, device="cuda")
    g = lambda a: None if a is None else torch.from_numpy(a).cuda()
    getattr(ctx, fn_name)(g(cur), g(prev), g(d), st, mask_out=M, pooled_out=pq, theta=theta)
    torch.cuda.synchronize()
    return st, M, pq


def _same(a, b):
    return np.array_equal(a.cpu().numpy().view(np.uint32 if a.dtype.itemsize == 4 else np.uint16),
                          b.cpu().numpy().view(np.uint32 if b.dtype.itemsize == 4 else np.uint16))


def test_static_refine_matches_allocating_path_on_consecutive_calls():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    rng = np.random.default_rng(20250518)
    # two frames of a 1920 x 1080 video (the second call takes the first call's state), then a small ragged view that
    # reuses the front of the array the large calls filled, then a 4-byte pixel stride
    cases = [(1920, 1080, 3), (1920, 1080, 3), (203, 131, 3), (132, 70, 4)]
    state_a = state_b = None
    prev_img = None
    for i, (W, H, stride) in enumerate(cases):
        chained = i == 1
        prev, cur, d = _frame(rng, W, H, stride, prev=prev_img if chained else None)
        if not chained:
            s0 = rng.uniform(0.5, 5, (H, W)).astype(np.float32)
            s0[rng.uniform(size=(H, W)) < 0.05] = 0
            state_a = torch.from_numpy(s0).cuda()
            state_b = state_a.clone()
        theta = 8.0 / 255.0 if i % 2 else 0.0
        launches = ctx.launch_count
        state_a, Ma, pa = _both(ctx, "ggt_refine_depth_static", cur, prev, d, state_a, theta)
        assert ctx.launch_count - launches == 2
        state_b, Mb, pb = _both(ctx, "ggt_refine_depth", cur, prev, d, state_b, theta)
        assert _same(pa, pb), "pooled block differences differ (case %d)" % i
        assert _same(Ma, Mb), "mask differs (case %d)" % i
        assert _same(state_a, state_b), "refined depth differs (case %d)" % i
        assert bool((Ma == 1).any()) and bool((Ma < 1).any())
        prev_img = cur
    # first-frame rule through the new entry point (no scratch involved)
    H, W = 131, 203
    d = torch.from_numpy(rng.uniform(0.5, 5, (H, W)).astype(np.float32)).cuda()
    st = torch.zeros((H, W), dtype=torch.float32, device="cuda")
    M = torch.zeros((H, W), dtype=torch.float32, device="cuda")
    ctx.ggt_refine_depth_static(None, None, d, st, mask_out=M)
    torch.cuda.synchronize()
    assert torch.equal(st, d) and bool((M == 1).all())
    ctx.close()


def test_static_refine_rejects_sizes_beyond_the_fixed_scratch():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    W, H = 2052, 2048                                   # 513 x 512 cells > 262144
    assert ((W + 3) // 4) * ((H + 3) // 4) > MAX_CELLS
    rgb = torch.zeros((H, W, 3), dtype=torch.uint8, device="cuda")
    d = torch.ones((H, W), dtype=torch.float32, device="cuda")
    st = torch.full((H, W), 2.0, dtype=torch.float32, device="cuda")
    launches = ctx.launch_count
    with pytest.raises(binding.GgtError, match="fixed scratch holds 262144"):
        ctx.ggt_refine_depth_static(rgb, rgb, d, st)
    torch.cuda.synchronize()
    assert ctx.launch_count == launches and bool((st == 2.0).all())      # nothing launched, state untouched
    # the largest size that fits runs, and matches the allocating path
    W = 2048
    rng = np.random.default_rng(7)
    prev, cur, dd = _frame(rng, W, H, 3)
    s0 = torch.from_numpy(rng.uniform(0.5, 5, (H, W)).astype(np.float32)).cuda()
    a = _both(ctx, "ggt_refine_depth_static", cur, prev, dd, s0, 0.0)
    b = _both(ctx, "ggt_refine_depth", cur, prev, dd, s0, 0.0)
    assert all(_same(x, y) for x, y in zip(a, b))
    ctx.close()
