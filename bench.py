#!/usr/bin/env python
"""bench.py -- per-turn layer-streamed prefill on one B200 (BASELINE.json metric).

A "step" is one whole turn of the hot path (all SURVEY.md 8(a) rows) over one batch of
synthetic input: for each of the L layers, paged gather of the history KV pool -> LSC on the
copy stream, scatter of the turn's new K/V into pool blocks, causal attention of the new
tokens over history + themselves, split-KV combine; two streams, double-buffered LSC.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload lwm_5k] [--mode staged|fused]
    python bench.py --impl reference ...     # the CPU oracle, as it stands, on the host cores

Prints ONE JSON line (rank 0).  The headline is BASELINE.json configs[1] (`lwm_5k`); the other
full-size configs are measured in the same run under `sweep` (fewer steps each).
section 7 for what every key means.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "per-turn layer-streamed prefill ms (256 new tok) & paged-KV GB/s vs HBM peak"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
SWEEP = ("lwm_50k", "gqa_128k", "gqa_128k_host", "multiturn")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="lwm_5k")
    ap.add_argument("--mode", default="staged", choices=["staged", "fused"])
    ap.add_argument("--engine", default="auto", choices=["auto", "mma", "tcgen05"])
    ap.add_argument("--copy", default="auto", choices=["auto", "ldg", "bulk"])
    ap.add_argument("--n-new", type=int, default=None,
                    help="new tokens per conversation instead of the config's (1 = a decode step); for profiling runs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--pool", default="config", choices=["config", "peer"],
                    help="peer (needs --gpus 2): the pool lives on rank 1's GPU, rank 0 reads it over NVLink (f2)")
    ap.add_argument("--peer-same-gpu", action="store_true",
                    help="with --pool peer: both ranks on cuda:0, gloo control plane (exercises the IPC path on a 1-GPU box)")
    ap.add_argument("--no-sweep", action="store_true", help="only the headline workload")
    ap.add_argument("--sweep", default=",".join(SWEEP), help="comma-separated workloads measured beside the headline")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        p["_source"] = "measured"
        return p
    p = dict(FALLBACK_PEAKS)
    p["_source"] = "fallback"
    return p


# ------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "25", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------- workload
def flops_per_layer(shape, hist, n):
    """4*Hq*D*n*(T_h + (n+1)/2): QK^T and PV, 2 flop per MAC, causal triangle counted once."""
    return 4.0 * shape.Hq * shape.D * n * (hist + (n + 1) / 2.0)


def config_dict(name: str, shape, mode: str, replicas: int) -> dict:
    """`config` of the JSON line; identical in the product arm and the reference arm."""
    kv_turn_bytes = float(sum(shape.hist)) * shape.tok_bytes * shape.L
    return {"workload": workload_string(name, shape), "mode": mode, "replicas": replicas,
            "l2": f"inputs larger than L2: each turn streams {kv_turn_bytes/1e9:.2f} GB of pool KV"}


def workload_string(name: str, shape, n_new=None) -> str:
    """Names the workload; the same string in the product arm and the reference arm."""
    hist = list(shape.hist)
    return (f"{name}: {shape.L} layers, {shape.Hq}q/{shape.Hkv}kv heads, D {shape.D}, block {shape.B}, "
            f"history {hist} tokens in a shuffled {shape.n_blocks}-block "
            f"{'pinned-host' if shape.pool_kind == 'host' else 'HBM'} pool, {n_new or shape.n_new} new tokens")


class Workload:
    """Synthetic conversations of one BASELINE.json config, resident in HBM."""

    def __init__(self, name: str, device, engine="auto", copy="auto", keep_host_layers=1, n_new=None, peer_pool_ptr=None,
                 sorted_table=False):
        import torch
        from paper_2606_16135_b200 import binding as sc
        from paper_2606_16135_b200 import inputs as I
        from paper_2606_16135_b200.runtime import Session

        self.torch, self.sc, self.I = torch, sc, I
        shape = I.configs()[name]
        self.shape, self.name = shape, name
        B = shape.B
        self.n_seq = len(shape.hist)
        self.hist = list(shape.hist)
        self.n_new = [n_new or shape.n_new] * self.n_seq
        self.cu = np.concatenate([[0], np.cumsum(self.n_new)]).astype(np.int32)
        blocks = [-(-(h + n * shape.turns) // B) for h, n in zip(self.hist, self.n_new)]   # room for every turn
        self.max_blocks = max(blocks)
        pool_kind = sc.SC_POOL_HOST_PINNED if shape.pool_kind == "host" else sc.SC_POOL_HBM
        if peer_pool_ptr is not None:          # f2: the region is another GPU's memory, mapped by the caller
            pool_kind = sc.SC_POOL_PEER
        self.sess = Session(shape.L, shape.Hq, shape.Hkv, shape.D, B, shape.n_blocks, sum(blocks),
                            int(self.cu[-1]), max_seqs=self.n_seq, pool_kind=pool_kind,
                            alloc_seed=0 if sorted_table else I.BASE_SEED + shape.config_id, device=device,
                            pool_ptr=peer_pool_ptr)          # alloc_seed 0: ids in order (the locality best case)
        eng = {"auto": sc.SC_ENGINE_AUTO, "mma": sc.SC_ENGINE_MMA_SYNC, "tcgen05": sc.SC_ENGINE_TCGEN05}[engine]
        cpy = {"auto": sc.SC_COPY_AUTO, "ldg": sc.SC_COPY_LDG, "bulk": sc.SC_COPY_BULK}[copy]
        self.sess.pool.set_engine(eng, cpy)
        # tables: the library's allocator hands out a seeded shuffle of the pool ("shuffled pool")
        self.tables = np.full((self.n_seq, self.max_blocks), -1, dtype=np.int32)
        self.n_table = []
        for s in range(self.n_seq):
            nt = self.sess.pool.append_blocks(self.tables[s], 0, 0, self.hist[s])
            nt = self.sess.pool.append_blocks(self.tables[s], nt, self.hist[s], self.n_new[s])
            self.n_table.append(nt)
        self.tables_dev = self.sess.table_dev(self.tables)
        # history: one layer at a time, generated on the device from its seed, stored via the ABI
        self.host_hist = {}
        dev = self.sess.device
        for l in range(shape.L):
            for s in range(self.n_seq):
                k = I.normal_bf16_device((self.hist[s], shape.Hkv, shape.D), I.seed_for(shape.config_id, l, "k", conv=s), dev)
                v = I.normal_bf16_device((self.hist[s], shape.Hkv, shape.D), I.seed_for(shape.config_id, l, "v", conv=s), dev)
                self.sess.store_prefix(l, k, v, 0, self.tables_dev[s])
                if l < keep_host_layers and s == 0:
                    self.host_hist[(l, s)] = (k.view(torch.int16).cpu().numpy().view(np.uint16),
                                              v.view(torch.int16).cpu().numpy().view(np.uint16))
            torch.cuda.synchronize()
        tot = int(self.cu[-1])
        self.q = I.normal_bf16_device((shape.L, tot, shape.Hq, shape.D), I.seed_for(shape.config_id, 0, "q"), dev)
        self.k = I.normal_bf16_device((shape.L, tot, shape.Hkv, shape.D), I.seed_for(shape.config_id, 0, "k_new"), dev)
        self.v = I.normal_bf16_device((shape.L, tot, shape.Hkv, shape.D), I.seed_for(shape.config_id, 0, "v_new"), dev)
        self.out = torch.zeros_like(self.q)
        torch.cuda.synchronize()

    def turn(self, mode, io="device", bufs=None):
        sc, s = self.sc, self.sess
        q, k, v, out = bufs if bufs is not None else (self.q, self.k, self.v, self.out)
        s.pool.prefill_turn(q.data_ptr(), k.data_ptr(), v.data_ptr(), out.data_ptr(),
                            sc.SC_MEM_HOST_PINNED if io == "host" else sc.SC_MEM_DEVICE,
                            self.tables_dev.data_ptr(), self.max_blocks, self.hist, self.cu, mode,
                            s.copy_stream.cuda_stream, s.compute_stream.cuda_stream)

    def new_inputs(self, turn: int):
        """Seeded q / k_new / v_new of all layers for turn `turn` (device)."""
        I, shape, dev = self.I, self.shape, self.sess.device
        tot = int(self.cu[-1])
        self.q = I.normal_bf16_device((shape.L, tot, shape.Hq, shape.D), I.seed_for(shape.config_id, 0, "q", turn=turn), dev)
        self.k = I.normal_bf16_device((shape.L, tot, shape.Hkv, shape.D), I.seed_for(shape.config_id, 0, "k_new", turn=turn), dev)
        self.v = I.normal_bf16_device((shape.L, tot, shape.Hkv, shape.D), I.seed_for(shape.config_id, 0, "v_new", turn=turn), dev)

    def advance(self, turn: int):
        """After a turn: its new tokens are history now (they were scattered into the pool);
        grow every table for the next turn's new tokens and draw that turn's inputs."""
        for s in range(self.n_seq):
            self.hist[s] += self.n_new[s]
        blocks = [-(-(h + n) // self.shape.B) for h, n in zip(self.hist, self.n_new)]
        if max(blocks) > self.tables.shape[1]:
            grown = np.full((self.n_seq, max(blocks) + 64), -1, dtype=np.int32)
            grown[:, :self.tables.shape[1]] = self.tables
            self.tables = grown
        self.max_blocks = self.tables.shape[1]
        for s in range(self.n_seq):
            self.n_table[s] = self.sess.pool.append_blocks(self.tables[s], self.n_table[s], self.hist[s], self.n_new[s])
        self.tables_dev = self.sess.table_dev(self.tables)
        self.new_inputs(turn)
        self.torch.cuda.synchronize()

    # algorithmic work of one layer
    def layer_flops(self):
        return sum(flops_per_layer(self.shape, h, n) for h, n in zip(self.hist, self.n_new))

    def layer_gather_bytes(self):
        cell = self.sess.pool.info().cell_bytes
        return 2.0 * sum(-(-h // self.shape.B) for h in self.hist) * cell      # read + write

    def layer_hist_kv_bytes(self):
        return float(sum(self.hist)) * self.shape.tok_bytes

    def layer_scatter_bytes(self, staged):
        return float(self.cu[-1]) * self.shape.tok_bytes * (3.0 if staged else 2.0)


# ------------------------------------------------------------------ CPU baseline
class HostSample:
    """Host (numpy) inputs of layer 0, conversation 0 of a workload for the oracle: history K/V,
    the turn's q / k_new / v_new as bf16 bits, and a block table.  Built either from a resident
    product workload (same bytes: the parity spot check) or, for the reference arm, from the
    seeded host generators alone -- nothing of the product library, no GPU."""

    def __init__(self, shape, kh, vh, q, kn, vn, table, hist_all, n_new_all):
        self.shape, self.kh, self.vh, self.q, self.kn, self.vn, self.table = shape, kh, vh, q, kn, vn, table
        self.hist_all, self.n_new_all = list(hist_all), list(n_new_all)

    @classmethod
    def from_workload(cls, w: "Workload"):
        torch = w.torch
        n = w.n_new[0]
        kh, vh = w.host_hist[(0, 0)]
        bits = lambda t: t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)   # noqa: E731
        return cls(w.shape, kh, vh, bits(w.q[0, :n]), bits(w.k[0, :n]), bits(w.v[0, :n]),
                   w.tables[0][:w.n_table[0]].copy(), w.hist, w.n_new)

    @classmethod
    def from_seeds(cls, name: str):
        from paper_2606_16135_b200 import inputs as I            # seeded generators only: no method arithmetic
        shape = I.configs()[name]
        T_h, n = shape.hist[0], shape.n_new
        cid = shape.config_id
        kh = I.normal_bf16((T_h, shape.Hkv, shape.D), I.seed_for(cid, 0, "k"))
        vh = I.normal_bf16((T_h, shape.Hkv, shape.D), I.seed_for(cid, 0, "v"))
        q = I.normal_bf16((n, shape.Hq, shape.D), I.seed_for(cid, 0, "q"))
        kn = I.normal_bf16((n, shape.Hkv, shape.D), I.seed_for(cid, 0, "k_new"))
        vn = I.normal_bf16((n, shape.Hkv, shape.D), I.seed_for(cid, 0, "v_new"))
        table = I.block_table(cid, shape.n_blocks, -(-(T_h + n) // shape.B))
        return cls(shape, kh, vh, q, kn, vn, table, shape.hist, [n] * len(shape.hist))


def set_omp_threads(n: int) -> bool:
    """Thread count of the oracle's OpenMP runtime (the oracle itself is not touched)."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def oracle_sample(hs: HostSample, step_budget_s=1.2, total_budget_s=12.0, max_steps=None, rows=None):
    """Times the CPU oracle, as it stands, on a bounded sample of the workload: layer 0 of
    conversation 0 -- the whole layer's paged gather + scatter and the attention of `rows`
    middle new-token rows x all heads over the full history (ALL rows when they fit the step
    budget, as at lwm_5k), repeated.  Returns (ms per turn extrapolated to L layers x n rows x
    all conversations, info, (a, b, out))."""
    from oracle import sc_oracle as O
    shape = hs.shape
    n, T_h = len(hs.q), len(hs.kh)
    tab = hs.table
    if rows is None:      # ~2e10 flop/s is what the fp32 oracle reaches on 16 cores; never tuned, only sized
        rows = int(max(8, min(n, step_budget_s * 2.0e10 / (4.0 * shape.Hq * shape.D * (T_h + n / 2.0)))))
    rows = max(1, min(rows, n))
    a = max(0, n // 2 - rows // 2)
    b = min(n, a + rows)
    # the oracle's own pool, one layer deep, same block ids
    opool = O.Pool(1, shape.Hkv, shape.D, shape.B, shape.n_blocks)
    opool.store(0, 0, hs.kh, 0, tab)
    opool.store(0, 1, hs.vh, 0, tab)
    t_move, t_attn, steps, out = [], [], 0, None
    t_start = time.perf_counter()
    while True:
        t0 = time.perf_counter()
        lk = opool.gather(0, 0, tab, T_h)
        lv = opool.gather(0, 1, tab, T_h)
        opool.store(0, 0, hs.kn, T_h, tab)
        opool.store(0, 1, hs.vn, T_h, tab)
        t1 = time.perf_counter()
        K = np.concatenate([lk, hs.kn[:b]])
        V = np.concatenate([lv, hs.vn[:b]])
        out = O.attention(hs.q[a:b], K, V, T_h + a)
        t2 = time.perf_counter()
        t_move.append(t1 - t0)
        t_attn.append(t2 - t1)
        steps += 1
        if (max_steps and steps >= max_steps) or (not max_steps and time.perf_counter() - t_start > total_budget_s):
            break
    # rows [a, b) sit in the middle of the turn: their mean causal length is that of the whole turn
    scale_rows = n / float(b - a)
    work_ratio = (sum(flops_per_layer(shape, h, m) for h, m in zip(hs.hist_all, hs.n_new_all)) /
                  flops_per_layer(shape, T_h, n))
    move_ratio = sum(hs.hist_all) / float(max(T_h, 1))
    per_layer_s = np.mean(t_move) * move_ratio + np.mean(t_attn) * scale_rows * work_ratio
    full = (b - a) == n
    info = {"cores": O.openmp_threads(), "kind": "oracle",
            "sample": (f"layer 0, conversation 0: full-layer paged gather+scatter ({np.mean(t_move)*1e3:.0f} ms) + "
                       f"attention of {'ALL ' if full else ''}new-token rows [{a},{b}) x {shape.Hq} heads over {T_h}+{n} keys "
                       f"({np.mean(t_attn)*1e3:.0f} ms), {steps} repeats; extrapolated "
                       + ("" if full else f"x{scale_rows:.1f} rows ") + f"x{shape.L} layers"
                       + (f" x{work_ratio:.2f} conversations" if len(hs.hist_all) > 1 else "")),
            "step_s": [float(x + y) for x, y in zip(t_move, t_attn)]}
    return per_layer_s * shape.L * 1e3, info, (a, b, out)


def single_thread_figure(hs: HostSample) -> dict:
    """The same oracle on ONE host thread (BASELINE.md promises it), on 1/16 of the rows."""
    from oracle import sc_oracle as O
    n_threads = O.openmp_threads()
    if not set_omp_threads(1):
        return {"unavailable": "libgomp not found"}
    try:
        ms, info, _ = oracle_sample(hs, max_steps=1, rows=max(4, len(hs.q) // 16))
    finally:
        set_omp_threads(n_threads)
    return {"value": round(ms, 1), "unit": "ms", "cores": 1, "sample": info["sample"]}


# ------------------------------------------------------------------ N > 1: replicas only
def replica_plan(world: int, rank: int, n_conversations: int = 1) -> dict:
    """The path has no exchange step: N GPUs run N independent replicas of
    the workload, each with its own pool and conversations.  Pure bookkeeping, no collective."""
    return {"replica": rank, "replicas": world, "conversations": n_conversations * world,
            "collective_on_data_path": None}


def max_over_ranks(ms: float, world: int, device="cpu") -> float:
    """Timing of a multi-rank run is the MAX over ranks (the job is done when the slowest
    replica is).  Works on any backend (nccl on GPUs, gloo in the CPU tests)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job(ms_per_step: float, world: int, per_replica_kv_bytes: float, per_replica_flops: float) -> dict:
    """Aggregate throughput of all replicas over the max-over-ranks step time."""
    return {"kv_gbs": world * per_replica_kv_bytes / ms_per_step / 1e6,
            "attn_tflops": world * per_replica_flops / ms_per_step / 1e9}


# ------------------------------------------------------------------------- ours
def _avg(rec):
    return rec[0] / rec[1] if rec[1] else None


def kernel_table(w: "Workload", prof: dict, p_steps: int, staged: bool, pk: dict) -> dict:
    """Per-kernel device time (events around every launch, inside the pipeline) against the
    algorithmic work of DESIGN.md section 6 and the measured peaks."""
    work = {"gather": ("hbm", w.layer_gather_bytes()), "attention": ("tensor", w.layer_flops()),
            "scatter": ("hbm", w.layer_scatter_bytes(staged)), "combine": ("hbm", None)}
    link = "pcie" if w.shape.pool_kind == "host" else "hbm"
    kernels = {}
    tot = sum(rec[0] for rec in prof.values())
    for name, rec in prof.items():
        a = _avg(rec)
        if a is None:
            continue
        bound, amount = work[name]
        k = {"avg_ms": round(a, 5), "launches_per_turn": rec[1] // p_steps, "share": round(rec[0] / tot, 4) if tot else None,
             "bound": link if name == "gather" else bound}
        if amount:
            if bound == "hbm":
                k["achieved_GBs"] = round(amount / a / 1e6, 1)
                if name == "gather" and link == "pcie":
                    k["pool_read_GBs"] = round(amount / 2 / a / 1e6, 2)          # what crosses the link: the reads
                else:
                    k["frac_of_measured_hbm"] = round(amount / a / 1e6 / pk["hbm_gbs"], 4)
            else:
                k["achieved_TFLOPs"] = round(amount / a / 1e9, 1)
                k["frac_of_bf16_burst"] = round(amount / a / 1e9 / pk["bf16_tflops"], 4)
                k["frac_of_bf16_sustained"] = round(amount / a / 1e9 / pk["bf16_tflops_sustained"], 4)
        kernels[name] = k
    return kernels


def pinned_copy_rates(torch, device, mb=1024) -> tuple:
    """GB/s of a plain pinned cudaMemcpy host -> device and device -> host, measured in this run: the
    link rate the host-pool gather (reads: H2D direction) is held against."""
    h = torch.empty(mb << 20, dtype=torch.uint8).pin_memory()
    d = torch.empty(mb << 20, dtype=torch.uint8, device=device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rates = []
    for dst, src in ((d, h), (h, d)):
        dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()
        best = 0.0
        for _ in range(3):
            e0.record()
            dst.copy_(src, non_blocking=True)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, (mb << 20) / e0.elapsed_time(e1) / 1e6)
        rates.append(best)
    return rates[0], rates[1]


def peer_pool(args, world: int, rank: int, local: int):
    """with `--gpus 2 --pool peer` the pool region is allocated on rank 1's GPU
    (cudaMalloc, exported through CUDA IPC: paper_2606_16135_b200/peer.py) and opened on rank 0 (one
    process per GPU); rank 0 then runs the workload with pool_kind = SC_POOL_PEER, i.e. every pool read
    and write crosses NVLink, and rank 1 only lends the memory.  With --peer-same-gpu both ranks use
    cuda:0 over a gloo control plane: the same handle / offset / mapping code runs, the link does not.
    Returns (pointer valid on this rank's device or None, keep-alive object).
    The NVLink rate is UNMEASURED by the builder: it needs two GPUs."""
    import torch.distributed as dist
    from paper_2606_16135_b200 import binding as sc
    from paper_2606_16135_b200 import inputs as I
    from paper_2606_16135_b200 import peer
    shape = I.configs()[args.workload]
    blocks = sum(-(-(h + shape.n_new * shape.turns) // shape.B) for h in shape.hist)
    cfg = sc.make_config(shape.L, shape.Hq, shape.Hkv, shape.D, shape.B, shape.n_blocks, blocks, shape.n_new)
    pool_bytes, _ = sc.sc_pool_bytes_required(cfg)
    keep, payload = None, [None]
    if rank == 1:
        keep = peer.LentRegion(pool_bytes, device=local)
        keep.fill(0)
        payload = [keep.ticket()]
    dist.broadcast_object_list(payload, src=1)
    ptr = None
    if rank == 0:
        keep = peer.OpenedRegion(payload[0], need_bytes=pool_bytes, device=local)
        ptr = keep.ptr
    return ptr, keep


class Filler:
    """The work a model does between two attentions -- o-proj, FFN (gate, up, down) of layer l and the
    QKV projection of layer l+1 for the turn's new tokens, Llama-2-7B sizes, random weights -- as ONE
    CUDA graph of cuBLAS GEMMs.  It is NOT on the method's path (the GEMMs are
    outside); the f4 harness only needs something of the right length on the compute stream for the
    single-buffer load to hide behind."""

    def __init__(self, torch, device, stream, n_tokens, hidden, ffn=11008):
        self.torch, self.stream = torch, stream
        bf = torch.bfloat16
        self.x = torch.randn(n_tokens, hidden, device=device, dtype=bf)
        self.wo = torch.randn(hidden, hidden, device=device, dtype=bf) * 0.01
        self.w13 = torch.randn(hidden, 2 * ffn, device=device, dtype=bf) * 0.01
        self.w2 = torch.randn(ffn, hidden, device=device, dtype=bf) * 0.01
        self.wqkv = torch.randn(hidden, 3 * hidden, device=device, dtype=bf) * 0.01
        self.ffn = ffn
        self.flops = 2.0 * n_tokens * hidden * (hidden + 2 * ffn + ffn + 3 * hidden)
        torch.cuda.synchronize()
        with torch.cuda.stream(stream):
            self._body()                                  # warm cuBLAS up outside the capture
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, stream=stream):
            self._body()
        torch.cuda.synchronize()

    def _body(self):
        t = self.torch
        h = t.matmul(self.x, self.wo)
        g = t.matmul(h, self.w13)
        a = g[:, :self.ffn] * g[:, self.ffn:]
        y = t.matmul(a, self.w2)
        self.y = t.matmul(y, self.wqkv)

    def __call__(self, layer=None, stream_handle=None):
        with self.torch.cuda.stream(self.stream):
            self.graph.replay()


def measure_overlap(w: "Workload", timed_fn, steps: int) -> dict:
    """the paper's single-buffer schedule (sc_prefill_turn_ex, lsc_buffers = 1).
    Exposed load time per layer = (turn with loads) - (the same compute with no loads), measured once
    with nothing between the attentions (nothing to hide behind) and once with the Filler GEMMs
    enqueued after every attention by the hook."""
    torch, sc = w.torch, w.sc
    pool, sess, shape = w.sess.pool, w.sess, w.shape
    L = shape.L
    fill = Filler(torch, sess.device, sess.compute_stream, int(w.cu[-1]), shape.Hq * shape.D)
    # the same GEMMs over a 4096-token batch (many conversations prefilled together): compute-bound,
    # where the turn's own tokens make them stream their weights, i.e. HBM-bound like the load itself
    fill_big = Filler(torch, sess.device, sess.compute_stream, 4096, shape.Hq * shape.D)
    xs = sess.compute_stream.cuda_stream

    def turn_ex(nbuf, hook):
        pool.prefill_turn_ex(w.q.data_ptr(), w.k.data_ptr(), w.v.data_ptr(), w.out.data_ptr(), sc.SC_MEM_DEVICE,
                             w.tables_dev.data_ptr(), w.max_blocks, w.hist, w.cu, sc.SC_ATTN_STAGED,
                             sess.copy_stream.cuda_stream, xs, lsc_buffers=nbuf, after_attention=hook)

    def compute_only(hook):
        # the same scatter + attention per layer reading LSC[0] as it stands (no load): timing reference
        for l in range(L):
            pool.prefill_layer_batched(l, w.q[l].data_ptr(), w.k[l].data_ptr(), w.v[l].data_ptr(),
                                       w.tables_dev.data_ptr(), w.max_blocks, w.hist, w.cu, 0,
                                       sc.SC_ATTN_STAGED, w.out[l].data_ptr(), xs)
            if hook:
                hook(l, xs)

    res = {}
    for tag, hook in (("no_filler", None), ("filler", fill), ("filler_4096_tokens", fill_big)):
        t = {}
        for name, fn in (("single_buffer", lambda: turn_ex(1, hook)), ("double_buffer", lambda: turn_ex(2, hook)),
                         ("compute_only", lambda: compute_only(hook))):
            for _ in range(2):
                fn()
            t[name] = timed_fn(fn, steps) / steps
        res[tag] = {"single_buffer_ms": round(t["single_buffer"], 3), "double_buffer_ms": round(t["double_buffer"], 3),
                    "compute_only_ms": round(t["compute_only"], 3),
                    "exposed_load_ms_per_layer": round(max(0.0, t["single_buffer"] - t["compute_only"]) / L, 4),
                    "exposed_load_pct_of_turn": round(100.0 * max(0.0, t["single_buffer"] - t["compute_only"]) / t["single_buffer"], 2)}
    res["filler"]["filler_gflop_per_layer"] = round(fill.flops / 1e9, 1)
    res["filler_4096_tokens"]["filler_gflop_per_layer"] = round(fill_big.flops / 1e9, 1)
    res["schedule"] = "lsc_buffers=1: load(l+1) waits attention(l)+store(l), then runs beside the hook's GEMMs (PAPER.md:192)"
    return res


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_16135_b200 import build as sc_build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if rank == 0:
        sc_build.build()
    same_gpu = args.pool == "peer" and args.peer_same_gpu
    if same_gpu:
        local = 0
    if world > 1:
        if same_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        dist.barrier()
    device = torch.device(f"cuda:{local}")
    torch.cuda.set_device(device)
    from paper_2606_16135_b200 import binding as sc
    pk = peaks()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(w, mode, n_steps, io="device", bufs=None):
        xs = w.sess.compute_stream
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(xs)
        for _ in range(n_steps):
            w.turn(mode, io, bufs)
        ev1.record(xs)
        barrier()
        return max_over_ranks(ev0.elapsed_time(ev1), world, device)

    def timed_fn(fn, n_steps, stream=None):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(stream)
        for _ in range(n_steps):
            fn()
        ev1.record(stream)
        barrier()
        return ev0.elapsed_time(ev1)

    def profile(w, mode, p_steps):
        pool = w.sess.pool
        pool.profile_enable(True)
        for _ in range(p_steps):
            w.turn(mode)
        torch.cuda.synchronize()
        prof = pool.profile_collect()
        pool.profile_enable(False)
        return prof

    STAGED, FUSED = sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED
    peer_ptr, peer_keep = None, None
    if args.pool == "peer":
        if world != 2:
            raise SystemExit("--pool peer needs exactly two ranks (torchrun --nproc-per-node 2 ... --gpus 2)")
        peer_ptr, peer_keep = peer_pool(args, world, rank, local)
        if rank == 1:                          # lends its memory and waits for rank 0
            dist.barrier()
            peer_keep.free()                   # rank 0 has closed its mapping by now
            dist.destroy_process_group()
            return
        world = 1                              # one conversation, one compute GPU: no max-over-ranks below
    w = Workload(args.workload, device, args.engine, args.copy, peer_pool_ptr=peer_ptr, n_new=args.n_new)
    shape, pool, xs = w.shape, w.sess.pool, w.sess.compute_stream
    mode = STAGED if args.mode == "staged" else FUSED

    # warm-up, then the timed region (inputs resident in HBM)
    for _ in range(max(args.warmup, 3)):
        w.turn(mode)
    barrier()
    clk = ClockSampler(local) if rank == 0 else None
    l0 = pool.launch_count()
    total_ms = timed(w, mode, args.steps)
    launches = pool.launch_count() - l0
    clocks = clk.stop() if clk else None
    ms_per_step = total_ms / args.steps
    # the same turns one by one (an event after every turn, no host synchronisation in between): median and min
    n_each = max(3, min(args.steps, 20))
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(n_each + 1)]
    barrier()
    evs[0].record(xs)
    for i in range(n_each):
        w.turn(mode)
        evs[i + 1].record(xs)
    barrier()
    each = [evs[i].elapsed_time(evs[i + 1]) for i in range(n_each)]
    per_turn = {"median_ms": round(float(np.median(each)), 4), "min_ms": round(float(np.min(each)), 4), "turns": n_each}

    # the other variant of the path beside it (same workload, same timing protocol, fewer steps):
    # fused = attention reads pool blocks through the block table, no gather into the LSC
    other_mode = FUSED if mode == STAGED else STAGED
    for _ in range(3):
        w.turn(other_mode)
    o_steps = max(3, min(args.steps, 50))
    other_ms = timed(w, other_mode, o_steps) / o_steps

    # host side of a turn: wall time of the sc_prefill_turn CALL (argument checks, ~2 launches and ~4 event
    # operations per layer) while the GPU is held up by a sleep kernel, i.e. pure enqueue cost; a turn is
    # GPU-bound only if this is below its device time
    host_enqueue = {}
    for m, mname in ((STAGED, "staged"), (FUSED, "fused")):
        torch.cuda.synchronize()
        with torch.cuda.stream(xs):
            torch.cuda._sleep(int(6e7))                     # ~30 ms at 1.9 GHz: the queue does not drain meanwhile
        t0 = time.perf_counter()
        for _ in range(3):
            w.turn(m)
        host_enqueue[mname] = round((time.perf_counter() - t0) / 3 * 1e6, 1)
        torch.cuda.synchronize()

    # the same turn captured once into a CUDA graph and replayed (one launch per turn instead of ~64 launches
    # and ~130 event operations); same kernels, same ordering (tests/test_gpu_pipeline.py checks the bits)
    graph_replay = {}
    for m, mname in ((STAGED, "staged"), (FUSED, "fused")):
        try:
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr, stream=xs):
                w.turn(m)
            g_steps = max(3, min(args.steps, 50))
            with torch.cuda.stream(xs):                      # a replay goes to torch's current stream
                for _ in range(3):
                    gr.replay()
                graph_replay[mname] = round(timed_fn(gr.replay, g_steps, xs) / g_steps, 4)
            del gr
        except Exception as e:                               # noqa: BLE001 -- reported, the headline does not depend on it
            graph_replay[mname] = None
            graph_replay[mname + "_error"] = f"{type(e).__name__}: {e}"[:160]
    torch.cuda.synchronize()

    # end to end through the C ABI with HOST buffers (pinned): H2D of q/k/v and D2H of out inside
    e2e = None
    if not args.no_e2e:
        hq, hk, hv = (t.cpu().pin_memory() for t in (w.q, w.k, w.v))
        hout = torch.zeros(w.q.shape, dtype=torch.bfloat16).pin_memory()
        bufs = (hq, hk, hv, hout)
        for _ in range(3):
            w.turn(mode, "host", bufs)
        e_steps = max(3, min(args.steps, 20))
        e_ms = timed(w, mode, e_steps, "host", bufs) / e_steps
        h2d = sum(int(t.numel()) * 2 for t in (hq, hk, hv))
        d2h = int(hout.numel()) * 2
        e2e = {"value": round(e_ms, 4), "unit": "ms", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "pcie_gbs": round((h2d + d2h) / e_ms / 1e6, 2)}

    # per-kernel device times: events around every launch, on its own stream, inside the pipeline
    p_steps = 5
    prof = profile(w, mode, p_steps)
    # and each kernel alone (no concurrent stream): gather over all layers, fused attention
    iso = {}
    st = xs.cuda_stream
    pool.profile_enable(True)
    for _ in range(3):
        for l in range(shape.L):
            pool.load_layer_batched(l, w.tables_dev.data_ptr(), w.max_blocks, w.hist, w.cu, l & 1, st)
    torch.cuda.synchronize()
    iso["gather"] = pool.profile_collect()["gather"]
    pool.profile_enable(True)
    for _ in range(3):
        for l in range(shape.L):
            pool.prefill_layer_batched(l, w.q[l].data_ptr(), w.k[l].data_ptr(), w.v[l].data_ptr(),
                                       w.tables_dev.data_ptr(), w.max_blocks, w.hist, w.cu, 0,
                                       FUSED, w.out[l].data_ptr(), st)
    torch.cuda.synchronize()
    c = pool.profile_collect()
    iso["attention_fused"], iso["scatter"], iso["combine"] = c["attention"], c["scatter"], c["combine"]
    pool.profile_enable(False)

    staged = mode == STAGED
    kernels = kernel_table(w, prof, p_steps, staged, pk)
    work = {"gather": ("hbm", w.layer_gather_bytes()), "attention": ("tensor", w.layer_flops()),
            "scatter": ("hbm", w.layer_scatter_bytes(staged))}
    dom = max((n for n in prof if n in work and prof[n][1]), key=lambda n: prof[n][0])
    d_avg = _avg(prof[dom])
    bound, amount = work[dom]
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.txt")
    if os.path.exists(tpath):
        with open(tpath) as f:
            tj = json.load(f)
        traffic = tj.get(f"{args.workload}:{args.mode}:{dom}")
        traffic_src = (tj.get("_source", "") + " | " + tj.get("_commit", "")) if traffic is not None else None
    if bound == "hbm":
        roof = {"kernel": dom, "bound": "hbm", "achieved": round(amount / d_avg / 1e6, 1), "peak": pk["hbm_gbs"],
                "unit": "GB/s", "peak_source": pk["_source"] + " copy bandwidth"}
    else:
        # burst peak: the timed region is milliseconds long at the maximum SM clock (see `clocks`), not the
        # seconds-long power-capped regime the sustained figure describes; the sustained fraction is beside it
        roof = {"kernel": dom, "bound": "tensor", "achieved": round(amount / d_avg / 1e9, 1),
                "peak": pk["bf16_tflops"], "unit": "TFLOP/s",
                "peak_source": pk["_source"] + " cuBLAS bf16, burst",
                "frac_of_sustained_peak": round(amount / d_avg / 1e9 / pk["bf16_tflops_sustained"], 4)}
    roof["frac"] = round(roof["achieved"] / roof["peak"], 4)
    roof["traffic"] = traffic
    roof["traffic_source"] = traffic_src       # a committed ncu capture of an earlier run of this command, not this run
    roof["avg_launch_ms"] = round(d_avg, 5)
    roof["timed"] = "inside the two-stream pipeline" if staged else "fused turn, one stream"
    af = _avg(iso["attention_fused"])
    if af:
        roof["attention_alone"] = {"avg_launch_ms": round(af, 5), "achieved": round(w.layer_flops() / af / 1e9, 1),
                                   "frac": round(w.layer_flops() / af / 1e9 / pk["bf16_tflops"], 4)}

    # the oracle beside it (rank 0, bounded sample) and a parity spot check on that sample
    cpu, parity = None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        hs = HostSample.from_workload(w)
        cpu_ms, info, (a, b, ref) = oracle_sample(hs)
        got = w.I.bf16_bits_to_f32(w.out[0, a:b].view(torch.int16).cpu().numpy().view(np.uint16)).astype(np.float64)
        parity = {"layer": 0, "rows": [a, b], "max_abs": float(np.abs(got - ref).max()),
                  "rel_l2": float(np.linalg.norm(got - ref) / np.linalg.norm(ref)), "tol": [1e-2, 5e-3]}
        info.pop("step_s")
        cpu = {"value": round(cpu_ms, 1), "unit": "ms", **info, "single_thread": single_thread_figure(hs)}

    kv_turn_bytes = w.layer_hist_kv_bytes() * shape.L
    job = whole_job(ms_per_step, world, kv_turn_bytes, w.layer_flops() * shape.L)
    fused_turn_flops = w.layer_flops() * shape.L
    # what a staged turn must move through HBM at least: the gather's read + write and the attention's read
    hbm_floor_ms = (w.layer_gather_bytes() + w.layer_hist_kv_bytes()) * shape.L / (pk["hbm_gbs"] * 1e6)
    line = {
        "metric": METRIC, "value": round(ms_per_step, 4), "unit": "ms", "n_gpus": (1 if same_gpu else 2) if peer_ptr else world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": round(ms_per_step, 4), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": config_dict(args.workload, shape, args.mode, world),
        "pool": (("region lent by a second PROCESS on the same GPU (CUDA IPC, SC_POOL_PEER): exercises the mapping, not a link"
                  if same_gpu else "peer GPU over NVLink (CUDA IPC, SC_POOL_PEER); link rate ~900 GB/s per direction")
                 if peer_ptr else shape.pool_kind),
        "kv_gbs": round(job["kv_gbs"], 1),
        "attn_tflops": round(job["attn_tflops"], 1),
        "other_mode": {"mode": "fused" if other_mode == FUSED else "staged", "value": round(other_ms, 4),
                       "unit": "ms", "steps": o_steps},
        "per_turn": per_turn, "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roof, "kernels": kernels,
        "isolated": {k: {"avg_ms": round(_avg(v), 5)} for k, v in iso.items() if _avg(v) is not None},
        "cpu_baseline": cpu, "parity": parity,
        "host_enqueue_us_per_turn": host_enqueue, "graph_replay_ms": graph_replay,
    }
    if args.n_new:
        line["config"]["workload"] = workload_string(args.workload, shape, n_new=args.n_new)
    g = _avg(iso["gather"])
    if g:
        line["isolated"]["gather"]["GBs"] = round(w.layer_gather_bytes() / g / 1e6, 1)
        line["isolated"]["gather"]["frac_of_measured_hbm"] = round(w.layer_gather_bytes() / g / 1e6 / pk["hbm_gbs"], 4)
    if af:
        line["isolated"]["attention_fused"]["TFLOPs"] = round(w.layer_flops() / af / 1e9, 1)
        line["isolated"]["attention_fused"]["kv_read_GBs"] = round(w.layer_hist_kv_bytes() / af / 1e6, 1)
    sweep_on = rank == 0 and world == 1 and not args.no_sweep and args.workload == "lwm_5k" and not peer_ptr
    if sweep_on:
        line["overlap_f4"] = {args.workload: measure_overlap(w, lambda fn, n: timed_fn(fn, n, xs), 10)}
    w.sess.close()
    del w
    torch.cuda.empty_cache()

    # ---- the other full-size configs of BASELINE.json, same protocol, fewer steps (rank 0 of a 1-GPU run) ----
    if sweep_on:
        line["sweep"] = run_sweep(args, device, timed, profile, pk, local, timed_fn, line["overlap_f4"])
        line["decode"] = run_decode(args, device, timed, profile, pk)
    if rank == 0:
        # the driver's record keeps the scalars inside `roofline` and the last ~4 KB of stdout: every figure
        # DESIGN.md section 9 quotes goes, flat, into both places (`summary` is the LAST key of the line)
        summary = build_summary(line, pk, fused_turn_flops, hbm_floor_ms)
        line["roofline"].update(summary)
        line["summary"] = summary
        print(json.dumps(line))
    if peer_ptr:
        peer_keep.close()                      # the session over it was closed above
        dist.barrier()                         # releases rank 1
        dist.destroy_process_group()
    elif world > 1:
        dist.destroy_process_group()


def build_summary(line: dict, pk: dict, turn_flops: float, hbm_floor_ms: float) -> dict:
    """Flat scalars (no nesting, < 2 KB) of everything the line measures beside the headline; keys absent
    where a part did not run.  Fractions: `_frac` of the burst bf16 peak, `_frac_hbm` of the measured
    copy bandwidth, `_frac_pcie` of a pinned cudaMemcpy measured in the same run."""
    out = {}

    def put(key, val, nd=4):
        if val is not None:
            out[key] = round(float(val), nd)

    def dig(d, *path):
        for k in path:
            if not isinstance(d, dict) or k not in d:
                return None
            d = d[k]
        return d

    mode = line["config"].get("mode") if isinstance(line.get("config"), dict) else None
    staged_ms = line["value"] if mode == "staged" else dig(line, "other_mode", "value")
    fused_ms = line["value"] if mode == "fused" else dig(line, "other_mode", "value")
    put("staged_ms", staged_ms)
    put("fused_ms", fused_ms)
    if fused_ms:
        put("fused_frac", turn_flops / fused_ms / 1e9 / pk["bf16_tflops"])
    if staged_ms:
        put("step_frac_of_hbm_floor", hbm_floor_ms / staged_ms)
    put("attention_alone_frac", dig(line, "roofline", "attention_alone", "frac"))
    put("gather_alone_frac_hbm", dig(line, "isolated", "gather", "frac_of_measured_hbm"))
    put("gather_in_pipeline_frac_hbm", dig(line, "kernels", "gather", "frac_of_measured_hbm"))
    put("e2e_ms", dig(line, "e2e", "value"))
    put("cpu_oracle_ms", dig(line, "cpu_baseline", "value"), 1)
    put("parity_max_abs", dig(line, "parity", "max_abs"), 6)
    put("parity_rel_l2", dig(line, "parity", "rel_l2"), 6)
    sw = line.get("sweep") or {}
    for name, short in (("lwm_50k", "lwm_50k"), ("gqa_128k", "gqa_128k"), ("multiturn", "multiturn_t0")):
        for m in ("staged", "fused"):
            put(f"{short}_{m}_ms", dig(sw, name, m, "ms_per_turn"), 3)
        put(f"{short}_fused_frac", dig(sw, name, "fused", "kernels", "attention", "frac_of_bf16_burst"))
        put(f"{short}_gather_in_pipeline_frac_hbm", dig(sw, name, "staged", "kernels", "gather", "frac_of_measured_hbm"))
    last = [k for k in (sw.get("multiturn") or {}) if k.startswith("turn_")]
    if last:
        put("multiturn_last_fused_ms", dig(sw, "multiturn", last[0], "fused", "ms_per_turn"), 3)
        put("multiturn_last_staged_ms", dig(sw, "multiturn", last[0], "staged", "ms_per_turn"), 3)
    put("lwm_50k_sorted_fused_ms", dig(sw, "lwm_50k", "sorted_table", "fused", "ms_per_turn"), 3)
    put("host_pool_staged_ms", dig(sw, "gqa_128k_host", "staged", "ms_per_turn"), 3)
    put("host_pool_fused_ms", dig(sw, "gqa_128k_host", "fused", "ms_per_turn"), 3)
    put("host_pool_pcie_gbs", dig(sw, "gqa_128k_host", "pcie", "gather_pool_read_GBs"), 2)
    put("host_pool_memcpy_gbs", dig(sw, "gqa_128k_host", "pcie", "pinned_memcpy_h2d_GBs"), 2)
    put("host_pool_frac_pcie", dig(sw, "gqa_128k_host", "pcie", "frac_of_memcpy_rate"))
    dc = line.get("decode") or {}
    for name, short in (("lwm_5k", "decode_5k"), ("lwm_50k", "decode_50k"), ("gqa_128k", "decode_gqa_128k")):
        for m in ("staged", "fused"):
            put(f"{short}_{m}_ms", dig(dc, name, m, "ms_per_step"))
            put(f"{short}_{m}_frac_hbm", dig(dc, name, m, "frac_of_measured_hbm"))
    put("decode_5k_forced_decode_engine_ms", dig(dc, "lwm_5k", "fused_decode_engine_forced", "ms_per_step"))
    put("decode_5k_forced_decode_engine_frac_hbm", dig(dc, "lwm_5k", "fused_decode_engine_forced", "frac_of_measured_hbm"))
    ov = line.get("overlap_f4") or {}
    for name, short in (("lwm_5k", "5k"), ("lwm_50k", "50k"), ("gqa_128k_host", "host")):
        put(f"f4_exposed_pct_{short}", dig(ov, name, "filler", "exposed_load_pct_of_turn"), 2)
        put(f"f4_single_buffer_ms_{short}", dig(ov, name, "filler", "single_buffer_ms"), 3)
    he = line.get("host_enqueue_us_per_turn") or {}
    put("host_enqueue_us_staged", he.get("staged"), 1)
    put("host_enqueue_us_fused", he.get("fused"), 1)
    gr = line.get("graph_replay_ms") or {}
    put("graph_replay_staged_ms", gr.get("staged"))
    put("graph_replay_fused_ms", gr.get("fused"))
    return out


def run_decode(args, device, timed, profile, pk) -> dict:
    """n = 1 (one decode step of one conversation) over the same pools: the path degenerates to a paged
    read of the whole history per layer, so the roofline is HBM (history KV bytes / attention time)."""
    import torch
    from paper_2606_16135_b200 import binding as sc
    out = {}
    for name in ("lwm_5k", "lwm_50k", "gqa_128k"):
        w = Workload(name, device, args.engine, args.copy, keep_host_layers=0, n_new=1)
        e = {"workload": workload_string(name, w.shape, n_new=1)}
        for m, mname in ((sc.SC_ATTN_STAGED, "staged"), (sc.SC_ATTN_FUSED, "fused")):
            for _ in range(3):
                w.turn(m)
            steps = 20
            ms = timed(w, m, steps) / steps
            prof = profile(w, m, 2)
            att = _avg(prof["attention"])
            e[mname] = {"ms_per_step": round(ms, 4), "kv_gbs": round(w.layer_hist_kv_bytes() * w.shape.L / ms / 1e6, 1),
                        "attention_avg_ms": round(att, 5) if att else None,
                        "attention_kv_read_GBs": round(w.layer_hist_kv_bytes() / att / 1e6, 1) if att else None,
                        "frac_of_measured_hbm": round(w.layer_hist_kv_bytes() / att / 1e6 / pk["hbm_gbs"], 4) if att else None}
        if name == "lwm_5k":
            # the evidence behind AUTO's choice at short histories: the decode engine FORCED on the same input
            # (a faster attention launch, but scatter + merge as separate launches; sc_ops.cu keeps the tcgen05
            # kernel below 128 MiB of K/V per layer)
            w.sess.pool.set_engine(sc.SC_ENGINE_DECODE, sc.SC_COPY_AUTO)
            for _ in range(3):
                w.turn(sc.SC_ATTN_FUSED)
            ms = timed(w, sc.SC_ATTN_FUSED, 20) / 20
            att = _avg(profile(w, sc.SC_ATTN_FUSED, 2)["attention"])
            e["fused_decode_engine_forced"] = {
                "ms_per_step": round(ms, 4), "attention_avg_ms": round(att, 5) if att else None,
                "frac_of_measured_hbm": round(w.layer_hist_kv_bytes() / att / 1e6 / pk["hbm_gbs"], 4) if att else None}
        out[name] = e
        w.sess.close()
        del w
        torch.cuda.empty_cache()
    return out


def run_sweep(args, device, timed, profile, pk, local, timed_fn, overlap) -> dict:
    """lwm_50k, gqa_128k (HBM and pinned-host pool), multiturn (turns 0 and 9): ms per turn in both
    modes, per-kernel averages against the measured peaks, clocks sampled during each timed region."""
    import torch
    from paper_2606_16135_b200 import binding as sc
    STAGED, FUSED = sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED
    out = {}
    h2d_rate = d2h_rate = None
    for name in [x for x in args.sweep.split(",") if x]:
        t_begin = time.perf_counter()
        try:
            w = Workload(name, device, args.engine, args.copy, keep_host_layers=0)
        except Exception as e:                    # e.g. not enough pinned host memory on this box
            out[name] = {"unavailable": f"{type(e).__name__}: {e}"[:200]}
            continue
        shape = w.shape
        host = shape.pool_kind == "host"
        steps = 3 if host else (5 if name != "lwm_50k" else 10)
        entry = {"workload": workload_string(name, shape), "steps": steps, "warmup": 3}

        def measure(dst):
            for m, mname in ((STAGED, "staged"), (FUSED, "fused")):
                for _ in range(3):
                    w.turn(m)
                clk = ClockSampler(local)
                ms = timed(w, m, steps) / steps
                c = clk.stop()
                prof = profile(w, m, 2)
                dst[mname] = {"ms_per_turn": round(ms, 3),
                              "kv_gbs": round(w.layer_hist_kv_bytes() * shape.L / ms / 1e6, 1),
                              "attn_tflops": round(w.layer_flops() * shape.L / ms / 1e9, 1),
                              "kernels": kernel_table(w, prof, 2, m == STAGED, pk),
                              "clocks": {k: c[k] for k in ("sm_mhz", "sm_max_mhz", "reasons")}}

        measure(entry)
        if host:
            if h2d_rate is None:
                h2d_rate, d2h_rate = pinned_copy_rates(torch, device)
            g = entry["staged"]["kernels"].get("gather", {})
            entry["pcie"] = {"pinned_memcpy_h2d_GBs": round(h2d_rate, 2), "pinned_memcpy_d2h_GBs": round(d2h_rate, 2),
                             "gather_pool_read_GBs": g.get("pool_read_GBs"),
                             "frac_of_memcpy_rate": round(g["pool_read_GBs"] / h2d_rate, 4) if g.get("pool_read_GBs") else None}
        if name in ("lwm_50k", "gqa_128k_host"):   # f4 over a long HBM history and over the host pool
            overlap[name] = measure_overlap(w, lambda fn, n: timed_fn(fn, n, w.sess.compute_stream), 2 if host else 4)
        if shape.turns > 1:                         # config 5: ten successive turns; turn 0 above, now the last one
            entry["turn"] = 0
            for t in range(1, shape.turns):
                w.turn(FUSED)                       # the turn's new KV becomes history (scattered into the pool)
                w.advance(t)
            last = {"turn": shape.turns - 1, "history": list(w.hist)}
            measure(last)
            entry[f"turn_{shape.turns - 1}"] = last
        entry["wall_s"] = round(time.perf_counter() - t_begin, 1)
        out[name] = entry
        w.sess.close()
        del w
        torch.cuda.empty_cache()
        if name == "lwm_50k":
            # the same workload with block ids in ORDER (the locality best case for the paged reads)
            w = Workload(name, device, args.engine, args.copy, keep_host_layers=0, sorted_table=True)
            srt = {}
            for m, mname in ((STAGED, "staged"), (FUSED, "fused")):
                for _ in range(3):
                    w.turn(m)
                srt[mname] = {"ms_per_turn": round(timed(w, m, 5) / 5, 3)}
            entry["sorted_table"] = srt
            w.sess.close()
            del w
            torch.cuda.empty_cache()
    return out


# -------------------------------------------------------------------- reference
def run_reference(args):
    """The CPU oracle, as it stands, on the host cores: same config, metric and unit.  Touches
    nothing of the product library and no GPU: inputs come from the seeded host generators
    (paper_2606_16135_b200/inputs.py holds no method arithmetic), the table from inputs.block_table.
    Each step is a bounded sample of the workload (see oracle_sample) sized so that
    --steps K --warmup W ends within a few minutes; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_16135_b200 import inputs as I
    shape = I.configs()[args.workload]
    hs = HostSample.from_seeds(args.workload)
    n_steps = max(args.steps, 1)
    step_budget = min(1.2, 150.0 / (n_steps + max(args.warmup, 1)))
    oracle_sample(hs, step_budget_s=step_budget, max_steps=max(args.warmup, 1))
    ms, info, _ = oracle_sample(hs, step_budget_s=step_budget, max_steps=n_steps)
    step_s = info.pop("step_s")
    cpu = {"value": round(ms, 1), "unit": "ms", **info, "single_thread": single_thread_figure(hs)}
    line = {
        "impl": "reference", "metric": METRIC, "value": round(ms, 1), "unit": "ms", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(float(np.mean(step_s)) * 1e3, 2),
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(args.workload, shape, args.mode, 1),
        "cpu_baseline": cpu,
        "e2e": {"value": round(ms, 1), "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
