"""The N > 1 path of bench.py is "replicas only": no collective on the
data path, timing = max over ranks, value = work of all replicas / that time.  Covered here
with world_size 2 on CPU over gloo."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local_ms = 2.0 + rank                      # rank 1 is the slow replica
    ms = bench.max_over_ranks(local_ms, world)
    plan = bench.replica_plan(world, rank, n_conversations=1)
    job = bench.whole_job(ms, world, per_replica_kv_bytes=3.0e9, per_replica_flops=6.0e12)
    dist.barrier()
    q.put((rank, ms, plan, job))
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, plan, job in got:
        assert ms == pytest.approx(3.0)                            # max over ranks, on every rank
        assert plan == {"replica": rank, "replicas": 2, "conversations": 2, "collective_on_data_path": None}
        assert job["kv_gbs"] == pytest.approx(2 * 3.0e9 / 3.0 / 1e6)
        assert job["attn_tflops"] == pytest.approx(2 * 6.0e12 / 3.0 / 1e9)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(1.25, 1) == 1.25
    assert bench.whole_job(2.0, 1, 4.0e9, 2.0e12) == {"kv_gbs": 2000.0, "attn_tflops": 1000.0}
