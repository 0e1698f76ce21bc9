"""World-size-2 `gloo` tests (CPU) of the N > 1 path of bench.py.

The hot path does not shard across GPUs ("replicas only"): every rank migrates one replica of the
workload and the only `torch.distributed` traffic is the barrier and the max-over-ranks of the device time.  These tests
cover exactly that host logic: the MAX reduction, the whole-job value, and the reference arm's "rank 0 alone works"."""
from __future__ import annotations
import json
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, local_rank, world = bench.dist_env()
dist.init_process_group("gloo", init_method="env://", rank=rank, world_size=world)
my_ms = [3.0, 7.5][rank]                      # rank 1 is the slow one
dist.barrier()
ms = bench.max_over_ranks(my_ms, world)
val = bench.job_value(world, 1_000_000_000, ms)
# a second reduction with the roles swapped (the max must not depend on which rank is slow)
ms2 = bench.max_over_ranks([9.25, 1.0][rank], world)
dist.barrier()
print(json.dumps(dict(rank=rank, local_rank=local_rank, world=world, ms=ms, ms2=ms2, value=val)), flush=True)
dist.destroy_process_group()
"""


def _spawn(code, world=2, extra_env=None, args=()):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, "-c", code, *args], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = []
    for p in procs:
        try:
            o, e = p.communicate(timeout=300)
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            raise
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_max_over_ranks_and_job_value_gloo_world2():
    outs = _spawn(_WORKER.format(root=ROOT))
    recs = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda r: r["rank"])
    assert [r["rank"] for r in recs] == [0, 1] and all(r["world"] == 2 for r in recs)
    for r in recs:                               # every rank sees the slowest rank's time
        assert r["ms"] == 7.5 and r["ms2"] == 9.25
        # two replicas' bytes over the slowest time: 2 * 1e9 B / 7.5 ms
        assert abs(r["value"] - 2 * 1e9 / 7.5e-3 / 1e9) < 1e-9


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(4.25, 1) == 4.25
    assert bench.job_value(1, 2_000_000_000, 2.0) == pytest.approx(1000.0)


_REF_WORKER = r"""
import sys
sys.path.insert(0, {root!r})
sys.argv = ["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "c1",
            "--ref-elems", "20000"]
import bench
bench.main()
"""


def test_reference_arm_runs_on_rank0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the one JSON line, rank 1 exits 0 silently."""
    outs = _spawn(_REF_WORKER.format(root=ROOT))
    lines0 = [l for l in outs[0].splitlines() if l.startswith("{")]
    assert len(lines0) == 1
    rec = json.loads(lines0[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["value"] > 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["e2e"]["h2d_bytes_per_step"] == 0
    assert rec["config"]["workload"] == "c1"
    assert outs[1].strip() == ""
