"""World-size-2 tests on CPU (gloo) of the multi-process host logic: batch sharding without a collective,
max-over-ranks timing, and the reference arm under a multi-rank launch (rank 0 alone prints)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["SP2_ROOT"])
import numpy as np, torch, torch.distributed as dist
from paper_2101_06385_b200 import api
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
B = 1027
a, b = api.shard_range(B, rank, world)
own = torch.zeros(B, dtype=torch.int64); own[a:b] = 1
dist.all_reduce(own)                       # test-side check only: every item owned exactly once
t = bench._max_over_ranks(1.0 + rank, world)
bench._barrier(world)
with open(os.path.join(os.environ["SP2_OUT"], f"rank{rank}.json"), "w") as f:
    json.dump({"rank": rank, "range": [a, b], "cover_ok": bool((own == 1).all()), "tmax": t}, f)
dist.destroy_process_group()
'''


def _torchrun(args, env_extra=None, timeout=300):
    env = dict(os.environ, SP2_ROOT=ROOT, OMP_NUM_THREADS="2")
    env.update(env_extra or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000)] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_shard_range_partitions():
    from paper_2101_06385_b200 import api

    for n in (0, 1, 7, 1024, 1027):
        for world in (1, 2, 3, 8):
            spans = [api.shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        api.shard_range(4, 2, 2)


def test_two_ranks_gloo_sharding_and_max_reduce(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    r = _torchrun([str(w)], {"SP2_OUT": str(tmp_path)})
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads((tmp_path / f"rank{k}.json").read_text()) for k in range(2)]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    assert all(l["cover_ok"] for l in lines)
    assert all(l["tmax"] == 2.0 for l in lines)          # max over ranks of (1, 2)
    spans = sorted(tuple(l["range"]) for l in lines)
    assert spans == [(0, 514), (514, 1027)]


def test_reference_arm_under_two_ranks_prints_once():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--size", "256"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    L = lines[0]
    assert L["impl"] == "reference" and L["cpu_baseline"]["kind"] == "oracle" and L["value"] > 0
    assert L["e2e"]["h2d_bytes_per_step"] == 0 and L["e2e"]["value"] == L["value"]
