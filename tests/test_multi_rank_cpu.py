"""N > 1 plumbing on CPU (gloo, world size 2): frame sharding, max-over-ranks timing, and the rule that only
rank 0 of `bench.py --impl reference` prints a line.  No GPU, no compute calls into the CUDA library."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_frame_shards_partition_the_batch():
    from paper_1503_03492_b200.replicas import frame_shard
    for batch in (0, 1, 5, 64, 67):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                s, n = frame_shard(batch, r, world)
                seen += list(range(s, s + n))
            assert seen == list(range(batch))
            sizes = [frame_shard(batch, r, world)[1] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        frame_shard(4, 2, 2)


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import numpy as np
from paper_1503_03492_b200.replicas import frame_shard, max_over_ranks, shard_workload, whole_job_value
dist.init_process_group("gloo")
r, w = dist.get_rank(), dist.get_world_size()
t = max_over_ranks(1.0 + r, dist)                 # rank 1 is the slow one
s, n = frame_shard(7, r, w)
# the code path bench.py uses: a stack shards by frame, a single image is replicated
stack = np.arange(7 * 2 * 3, dtype=np.float32).reshape(7, 2, 3)
part, first, total, scaling = shard_workload(stack, r, w)
np.save(os.path.join({out!r}, "part%d.npy" % r), part)
one, _, total1, scaling1 = shard_workload(stack[0], r, w)
assert scaling == "strong" and total == 7 and first == s and part.shape[0] == n
assert scaling1 == "weak" and total1 == w and one.shape == (2, 3)
dist.barrier()
open(os.path.join({out!r}, "rank%d.txt" % r), "w").write(" ".join(map(str, (r, w, t, s, n, whole_job_value(10.0, w, t)))))
dist.destroy_process_group()
"""


def test_gloo_world_size_2_max_over_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, out=str(tmp_path)))
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
         "127.0.0.1", "--master-port", "29531", str(script)],
        capture_output=True, text=True, timeout=240, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    rows = sorted(open(tmp_path / f).read().split() for f in os.listdir(tmp_path) if f.startswith("rank"))
    assert len(rows) == 2
    for r, row in enumerate(rows):
        assert int(row[0]) == r and int(row[1]) == 2
        assert float(row[2]) == 2.0                   # the max over ranks, on every rank
        assert float(row[5]) == 10.0                  # 2 ranks * 10 units / 2 s
    assert [(int(r[3]), int(r[4])) for r in rows] == [(0, 4), (4, 3)]
    # the two ranks' shards, concatenated, are the whole stack
    import numpy as np
    parts = [np.load(tmp_path / f"part{r}.npy") for r in range(2)]
    assert np.array_equal(np.concatenate(parts), np.arange(7 * 2 * 3, dtype=np.float32).reshape(7, 2, 3))


def test_reference_arm_prints_on_rank_0_only():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
         "127.0.0.1", "--master-port", "29532", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
         "--steps", "1", "--warmup", "0", "--config", "0", "--ref-sweeps", "2"],
        capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
