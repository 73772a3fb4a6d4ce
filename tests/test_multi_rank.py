"""N > 1 path of bench.py on CPU (gloo, world_size 2): "replicas only" -- the only cross-rank step is
the max-over-ranks reduction of the per-rank device time; the reference arm prints on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
per_rank_ms = [10.0, 12.5][rank]                        # rank 1 is the slow replica
ms = bench.max_over_ranks(per_rank_ms, world)
val = bench.aggregate_value(world, 1000.0, ms * 1e-3)
print(json.dumps({{"rank": rank, "ms": ms, "value": val}}), flush=True)
dist.barrier()
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(code_or_args, world=2, script=None):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        cmd = [sys.executable, "-c", code_or_args] if script is None else [sys.executable, str(script), *code_or_args]
        procs.append(subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, cwd=str(ROOT)))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=600)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_max_over_ranks_and_aggregate_value_gloo_world2():
    outs = _spawn(WORKER.format(root=str(ROOT)))
    rows = [json.loads(o.strip().splitlines()[-1]) for o in outs]
    for r in rows:
        assert r["ms"] == 12.5                                   # every rank sees the slowest replica's time
        assert r["value"] == pytest.approx(2 * 1000.0 / 12.5e-3)  # whole-job aggregate: both replicas / max time


def test_single_rank_helpers_need_no_process_group():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.max_over_ranks(3.0, 1) == 3.0
    assert bench.aggregate_value(1, 10.0, 2.0) == 5.0


def test_reference_arm_prints_on_rank0_only():
    outs = _spawn(["--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "tiny",
                   "--oracle-samples", "4000"], script=ROOT / "bench.py")
    lines0 = [l for l in outs[0].splitlines() if l.strip().startswith("{")]
    lines1 = [l for l in outs[1].splitlines() if l.strip().startswith("{")]
    assert len(lines0) == 1 and not lines1
    d = json.loads(lines0[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
