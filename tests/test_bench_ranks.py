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


def test_summary_is_flat_small_and_last():
    """The driver's record keeps scalars and the tail of stdout: `summary` must be flat numbers,
    under 2 KB, built from whatever parts of the line exist (absent parts leave no key)."""
    import json
    import bench
    pk = {"hbm_gbs": 6500.0, "bf16_tflops": 1600.0, "bf16_tflops_sustained": 1400.0}
    line = {"value": 1.7, "config": {"mode": "staged"}, "other_mode": {"mode": "fused", "value": 1.1},
            "roofline": {"attention_alone": {"frac": 0.31}},
            "isolated": {"gather": {"frac_of_measured_hbm": 0.78}}, "kernels": {"gather": {"frac_of_measured_hbm": 0.5}},
            "e2e": {"value": 4.6}, "cpu_baseline": {"value": 25000.0}, "parity": {"max_abs": 1e-4, "rel_l2": 2e-3},
            "sweep": {"lwm_50k": {"staged": {"ms_per_turn": 9.0, "kernels": {"gather": {"frac_of_measured_hbm": 0.6}}},
                                  "fused": {"ms_per_turn": 8.2, "kernels": {"attention": {"frac_of_bf16_burst": 0.57}}},
                                  "sorted_table": {"fused": {"ms_per_turn": 8.1}}},
                      "multiturn": {"fused": {"ms_per_turn": 20.0}, "turn_9": {"fused": {"ms_per_turn": 23.0}}},
                      "gqa_128k_host": {"staged": {"ms_per_turn": 343.0}, "pcie": {"gather_pool_read_GBs": 50.2,
                                        "pinned_memcpy_h2d_GBs": 55.6, "frac_of_memcpy_rate": 0.9}}},
            "decode": {"lwm_5k": {"fused": {"ms_per_step": 0.88, "frac_of_measured_hbm": 0.39}}},
            "overlap_f4": {"lwm_5k": {"filler": {"exposed_load_pct_of_turn": 3.5, "single_buffer_ms": 4.2}}},
            "host_enqueue_us_per_turn": {"staged": 400.0, "fused": 150.0}}
    s = bench.build_summary(line, pk, turn_flops=7.0e11, hbm_floor_ms=1.2)
    assert all(isinstance(v, float) for v in s.values())
    assert len(json.dumps(s)) < 2048
    assert s["staged_ms"] == 1.7 and s["fused_ms"] == 1.1
    assert s["fused_frac"] == pytest.approx(7.0e11 / 1.1 / 1e9 / 1600.0, abs=1e-4)
    assert s["step_frac_of_hbm_floor"] == pytest.approx(1.2 / 1.7, abs=1e-4)
    assert s["lwm_50k_fused_frac"] == 0.57 and s["multiturn_last_fused_ms"] == 23.0
    assert s["host_pool_frac_pcie"] == 0.9 and s["decode_5k_fused_frac_hbm"] == 0.39
    assert s["f4_exposed_pct_5k"] == 3.5 and s["host_enqueue_us_staged"] == 400.0
    assert "gqa_128k_fused_ms" not in s and "decode_50k_fused_ms" not in s       # parts that did not run
    # a fused headline swaps the two
    line["config"]["mode"] = "fused"
    s = bench.build_summary(line, pk, 7.0e11, 1.2)
    assert s["fused_ms"] == 1.7 and s["staged_ms"] == 1.1
