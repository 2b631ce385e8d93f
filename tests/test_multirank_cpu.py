"""The N > 1 path of bench.py on CPU (gloo, world_size 2).  The path does not shard across GPUs in this build
(replicas only), so what there is to cover is the host logic: per-rank seeds, the
max-over-ranks time, the whole-job value, and that under torchrun only rank 0 prints the reference arm's line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # rank 1 is the slow one
assert ms == 15.0, ms
val = bench.whole_job_value(world, 3, 1000.0, ms)
assert abs(val - 2 * 3 * 1000.0 / 15e-3) < 1e-6, val
seeds = [None, None]
dist.all_gather_object(seeds, bench.replica_seed(42, rank, world))
assert seeds == [42, 1042], seeds
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("ok%d\n" % rank); sys.stdout.flush()
"""


def _free_port() -> int:
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_replica_seeds_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.count("ok") == 2, r.stdout


def test_reference_arm_under_torchrun_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--N", "4096"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_single_rank_helpers():
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.replica_seed(7, 0, 1) == 7
    assert bench.whole_job_value(1, 2, 10.0, 1.0) == pytest.approx(2e4)
