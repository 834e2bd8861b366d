"""f2 end to end between TWO PROCESSES: the worker
process allocates the pool region on its GPU and exports it through CUDA IPC, the master process
opens it and runs a turn with pool_kind = SC_POOL_PEER -- the code path of
`bench.py --gpus 2 --pool peer` (paper_2606_16135_b200/peer.py), which needs two GPUs to say
anything about NVLink but only two processes to be exercised.  On the one-GPU test box both
processes use cuda:0 and talk over gloo; the bytes still travel through the IPC mapping, so the
handle, offset and alignment logic is what runs in a real two-GPU launch.

Checked: in the master, staged and fused attention against the oracle and the written tokens read
back through the mapping; in the WORKER, after the master is done, the raw bytes of its own
allocation at the offsets sc_cell_offset gives against the oracle's pool -- i.e. the master's
writes really landed in the lender's memory, where the layout says."""
import os
import socket
import sys
import traceback

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

pytestmark = pytest.mark.gpu

SHAPE = dict(L=2, Hq=8, Hkv=2, D=128, B=16, NB=48, T_h=333, n=70)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _inputs(l):
    from paper_2606_16135_b200 import inputs as I
    s = SHAPE
    return I.make_qkv(s["n"], s["T_h"], s["Hq"], s["Hkv"], s["D"], 5150 + l)


def _oracle_pool_and_refs(table):
    from oracle import sc_oracle as O
    s = SHAPE
    opool = O.Pool(s["L"], s["Hkv"], s["D"], s["B"], s["NB"])
    refs = []
    for l in range(s["L"]):
        q, kh, vh, kn, vn = _inputs(l)
        opool.store(l, 0, kh, 0, table)
        opool.store(l, 1, vh, 0, table)
        refs.append(O.prefill_layer(opool, l, q, kn, vn, table, s["T_h"]))     # also stores kn, vn
    return opool, refs


def _worker(rank, port, q):
    try:
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE="2")
        import torch
        import torch.distributed as dist
        from oracle import sc_oracle as O
        from paper_2606_16135_b200 import binding as sc
        from paper_2606_16135_b200 import inputs as I
        from paper_2606_16135_b200 import peer
        from paper_2606_16135_b200.runtime import Session, bits_to_torch, torch_to_bits
        dist.init_process_group("gloo", rank=rank, world_size=2)
        torch.cuda.set_device(0)
        s = SHAPE
        cfg = sc.make_config(s["L"], s["Hq"], s["Hkv"], s["D"], s["B"], s["NB"], 32, s["n"], pool_kind=sc.SC_POOL_PEER)
        pool_bytes, _ = sc.sc_pool_bytes_required(cfg)
        table = I.block_table(3, s["NB"], O.blocks_for(s["T_h"] + s["n"], s["B"]))
        payload = [None]
        lent = None
        if rank == 1:                      # the worker: lends memory, computes nothing
            lent = peer.LentRegion(pool_bytes, device=0)
            lent.fill(0xFF)                # never cleared: NaN bit patterns everywhere
            payload = [lent.ticket()]
        dist.broadcast_object_list(payload, src=1)
        report = {"rank": rank}
        if rank == 0:                      # the master: opens the region and runs the turn over it
            opened = peer.OpenedRegion(payload[0], need_bytes=pool_bytes, device=0)
            sess = Session(s["L"], s["Hq"], s["Hkv"], s["D"], s["B"], s["NB"], 32, s["n"],
                           pool_kind=sc.SC_POOL_PEER, pool_ptr=opened.ptr, zero_fill=False)
            tdev = sess.table_dev(table)
            opool, refs = _oracle_pool_and_refs(table)
            st = torch.cuda.current_stream().cuda_stream
            errs = []
            for l in range(s["L"]):
                qb, kh, vh, kn, vn = _inputs(l)
                sess.store_prefix(l, bits_to_torch(kh, sess.device), bits_to_torch(vh, sess.device), 0, tdev)
                dq, dk, dv = (bits_to_torch(x, sess.device) for x in (qb, kn, vn))
                for mode in (sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED):
                    out = torch.zeros((s["n"], s["Hq"], s["D"]), dtype=torch.bfloat16, device=sess.device)
                    if mode == sc.SC_ATTN_STAGED:
                        sess.pool.load_layer(l, tdev.data_ptr(), len(table), s["T_h"], l & 1, st)
                    sess.pool.prefill_layer(l, dq.data_ptr(), dk.data_ptr(), dv.data_ptr(), tdev.data_ptr(), len(table),
                                            s["T_h"], s["n"], l & 1, mode, out.data_ptr(), st)
                    torch.cuda.synchronize()
                    got = I.bf16_bits_to_f32(torch_to_bits(out)).astype(np.float64)
                    ref = refs[l].astype(np.float64)
                    errs.append((l, mode, float(np.abs(got - ref).max()),
                                 float(np.linalg.norm(got - ref) / np.linalg.norm(ref)), bool(np.isnan(got).any())))
                k, v = sess.read_tokens(l, 0, tdev, 0, s["T_h"] + s["n"])
                report[f"tokens_{l}"] = bool(np.array_equal(torch_to_bits(k), opool.gather(l, 0, table, s["T_h"] + s["n"])) and
                                             np.array_equal(torch_to_bits(v), opool.gather(l, 1, table, s["T_h"] + s["n"])))
            report["errs"] = errs
            sess.close()
            opened.close()
        dist.barrier()                     # the master is done and has closed its mapping
        if rank == 1:
            raw = lent.to_host().view(np.uint16)
            opool, _ = _oracle_pool_and_refs(table)
            geom = sc.Pool(cfg)            # host-only pool object: offsets only
            rng = np.random.default_rng(7)
            T = s["T_h"] + s["n"]
            bad = 0
            for _ in range(3000):
                l, kv = int(rng.integers(s["L"])), int(rng.integers(2))
                t, h, d = int(rng.integers(T)), int(rng.integers(s["Hkv"])), int(rng.integers(s["D"]))
                off = geom.cell_offset(int(table[t // s["B"]]), l, kv, h, t % s["B"], d)
                want = opool.gather(l, kv, table[t // s["B"]:t // s["B"] + 1], s["B"])[t % s["B"], h, d]
                bad += int(raw[off // 2] != want)
            report["bad_bytes"] = bad
            # a block the conversation never used still holds what the worker put there
            unused = sorted(set(range(s["NB"])) - set(int(x) for x in table))[0]
            off = geom.cell_offset(unused, 0, 0, 0, 0, 0)
            report["unused_untouched"] = bool(raw[off // 2] == 0xFFFF)
            geom.destroy()
            lent.free()
        dist.destroy_process_group()
        q.put(report)
    except Exception:                      # noqa: BLE001 -- reported to the parent, which fails the test
        q.put({"rank": rank, "error": traceback.format_exc()})


def test_pool_lent_by_another_process_through_cuda_ipc():
    import torch.multiprocessing as mp
    from paper_2606_16135_b200 import build as sc_build
    from gpu_util import MAX_ABS_TOL, REL_L2_TOL
    sc_build.build()
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    reports = {}
    for _ in range(2):
        r = q.get(timeout=300)
        reports[r["rank"]] = r
    for p in procs:
        p.join(timeout=60)
    for r in reports.values():
        assert "error" not in r, r["error"]
    for p in procs:
        assert p.exitcode == 0
    master, worker = reports[0], reports[1]
    assert len(master["errs"]) == 2 * SHAPE["L"]
    for l, mode, max_abs, rel, has_nan in master["errs"]:
        assert not has_nan and max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, (l, mode, max_abs, rel, has_nan)
    assert all(master[f"tokens_{l}"] for l in range(SHAPE["L"]))
    assert worker["bad_bytes"] == 0 and worker["unused_untouched"]
