"""N > 1 host logic on CPU: world_size-2 gloo processes exercise the frame partition and the
max-over-ranks / sum-of-units reduction bench.py uses (the data path itself has no collective)."""
import os
import socket
import subprocess
import sys
import textwrap

from paper_2505_18932_b200 import sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_is_disjoint_and_equal_sized():
    for world in (1, 2, 4, 8):
        seen = []
        for r in range(world):
            fr = sharding.frames_for_rank(r, world, 3)
            assert len(fr) == 3
            seen += fr
        assert len(set(seen)) == len(seen)
        t = [sharding.assign_targets(8, r, world) for r in range(world)]
        assert sorted(sum(t, [])) == list(range(8))
        assert max(map(len, t)) - min(map(len, t)) <= 0 if 8 % world == 0 else 1


def test_reduce_timing_single_process():
    out = sharding.reduce_timing(12.5, 100.0)
    assert out == {"ms": 12.5, "units": 100.0, "world": 1}


def test_reduce_timing_gloo_world2(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent("""
        import json, os, sys
        sys.path.insert(0, %r)
        import torch.distributed as dist
        from paper_2505_18932_b200 import sharding
        rank, local, world = sharding.env_rank()
        dist.init_process_group("gloo", rank=rank, world_size=world)
        frames = sharding.frames_for_rank(rank, world, 3)
        out = sharding.reduce_timing(10.0 + 5.0 * rank, 1000.0 * (rank + 1))
        dist.barrier()
        print(json.dumps({"rank": rank, "frames": frames, **out}))
        dist.destroy_process_group()
    """ % ROOT))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    import json
    outs = [json.loads(p.communicate(timeout=120)[0].strip().splitlines()[-1]) for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for o in outs:
        assert o["ms"] == 15.0 and o["units"] == 3000.0 and o["world"] == 2
    assert outs[0]["frames"] == [0, 1, 2] and outs[1]["frames"] == [10, 11, 12]
