"""World-size-2 host logic on CPU (gloo): the replica bench's max-over-ranks reduction, and the reference arm
under torchrun (rank 0 alone runs the oracle and prints the JSON line; the other rank exits 0 without work).
The path itself does not shard ("replicas only"), so there is no collective to test."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    vals = [1.0 + rank, 5.0 - 2.0 * rank]               # rank 0: (1, 5); rank 1: (2, 3)
    out = bench.max_over_ranks(dist, vals, torch.device("cpu"))
    seeds = bench.replica_seed(202, rank)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, out, seeds))


def test_max_over_ranks_and_replica_seeds_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [2.0, 5.0] and res[1][1] == [2.0, 5.0]    # every rank holds the max of each entry
    assert res[0][2] != res[1][2]                                  # replicas run different seeded boxes


@pytest.mark.timeout(600)
def test_reference_arm_under_torchrun_two_ranks():
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus",
           "2", "--steps", "1", "--warmup", "0", "--ref-budget-s", "4"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=580, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout                               # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
