"""GPU parity of the ragged batch (a9), the multi-turn loop (O6) and the layer-streaming
pipeline (a8), all through the C ABI against the CPU oracle."""
import numpy as np
import pytest
import torch

from oracle import sc_oracle as O
from paper_2606_16135_b200 import binding as sc
from paper_2606_16135_b200 import build as sc_build
from paper_2606_16135_b200 import inputs as I
from paper_2606_16135_b200.runtime import Session, bits_to_torch, torch_to_bits

from gpu_util import assert_close

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="session", autouse=True)
def _built():
    sc_build.build()


class Conversations:
    """n_seq conversations sharing one pool; tables come from the library's allocator and are
    mirrored, id for id, in the oracle's pool."""

    def __init__(self, L, Hq, Hkv, D, hist, NB, max_new, seed, pool_kind=sc.SC_POOL_HBM, lsc_blocks=None):
        self.L, self.Hq, self.Hkv, self.D, self.B = L, Hq, Hkv, D, 16
        self.n_seq = len(hist)
        self.hist = list(hist)
        self.max_blocks = max(O.blocks_for(h, 16) for h in hist) + 64
        if lsc_blocks is None:
            lsc_blocks = sum(O.blocks_for(h, 16) for h in hist) + 64 * self.n_seq
        self.sess = Session(L, Hq, Hkv, D, 16, NB, lsc_blocks, max_new, max_seqs=self.n_seq,
                            pool_kind=pool_kind, alloc_seed=seed)
        self.opool = O.Pool(L, Hkv, D, 16, NB)
        self.tables = np.full((self.n_seq, self.max_blocks), -1, dtype=np.int32)
        self.n_table = [0] * self.n_seq
        self.logical = [[[None, None] for _ in range(L)] for _ in range(self.n_seq)]
        dev = self.sess.device
        for s, h in enumerate(hist):
            self.n_table[s] = self.sess.pool.append_blocks(self.tables[s], 0, 0, h)
        self.tables_dev = self.sess.table_dev(self.tables)
        for s, h in enumerate(hist):
            for l in range(L):
                kh = I.normal_bf16((h, Hkv, D), seed + 1000 * s + 10 * l)
                vh = I.normal_bf16((h, Hkv, D), seed + 1000 * s + 10 * l + 5)
                self.logical[s][l] = [kh, vh]
                if h:
                    self.sess.store_prefix(l, bits_to_torch(kh, dev), bits_to_torch(vh, dev), 0,
                                           self.tables_dev[s])
                    self.opool.store(l, 0, kh, 0, self.tables[s][:self.n_table[s]])
                    self.opool.store(l, 1, vh, 0, self.tables[s][:self.n_table[s]])
        torch.cuda.synchronize()

    def begin_turn(self, n_new):
        for s in range(self.n_seq):
            self.n_table[s] = self.sess.pool.append_blocks(self.tables[s], self.n_table[s], self.hist[s], n_new[s])
        self.tables_dev.copy_(torch.from_numpy(self.tables))
        all_ids = np.concatenate([self.tables[s][:self.n_table[s]] for s in range(self.n_seq)])
        assert len(set(all_ids.tolist())) == len(all_ids)            # tables stay pairwise disjoint
        self.cu = np.concatenate([[0], np.cumsum(n_new)]).astype(np.int32)

    def make_inputs(self, n_new, seed, variant="normal"):
        """q/k/v for every layer, packed over the batch: bits [L][sum n][H][D]."""
        qs, ks, vs = [], [], []
        for l in range(self.L):
            ql, kl, vl = [], [], []
            for s in range(self.n_seq):
                q, _, _, kn, vn = I.make_qkv(n_new[s], 0, self.Hq, self.Hkv, self.D, seed + 97 * l + 13 * s, variant)
                ql.append(q); kl.append(kn); vl.append(vn)
            qs.append(np.concatenate(ql)); ks.append(np.concatenate(kl)); vs.append(np.concatenate(vl))
        return np.stack(qs), np.stack(ks), np.stack(vs)

    def oracle_turn(self, q_all, k_all, v_all):
        outs = []
        for l in range(self.L):
            rows = []
            for s in range(self.n_seq):
                a, b = self.cu[s], self.cu[s + 1]
                tab = self.tables[s][:self.n_table[s]]
                rows.append(O.prefill_layer(self.opool, l, q_all[l][a:b], k_all[l][a:b], v_all[l][a:b], tab, self.hist[s]))
                self.logical[s][l][0] = np.concatenate([self.logical[s][l][0], k_all[l][a:b]])
                self.logical[s][l][1] = np.concatenate([self.logical[s][l][1], v_all[l][a:b]])
            outs.append(np.concatenate(rows))
        return np.stack(outs)

    def end_turn(self, n_new):
        for s in range(self.n_seq):
            self.hist[s] += int(n_new[s])

    def check_pool_equals_logical(self):
        for s in range(self.n_seq):
            for l in range(self.L):
                k, v = self.sess.read_tokens(l, 0, self.tables_dev[s], 0, self.hist[s])
                assert np.array_equal(torch_to_bits(k), self.logical[s][l][0])
                assert np.array_equal(torch_to_bits(v), self.logical[s][l][1])


@pytest.mark.parametrize("mode", [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED])
def test_ragged_batch_multi_turn(mode):
    """Config 5 in miniature: ragged histories (remainders mod 16: 5, 12, 0, 1), ragged n_new,
    3 turns; every turn's new KV is scattered back and read by the next turn (I2, O6)."""
    cv = Conversations(L=2, Hq=4, Hkv=2, D=64, hist=[37, 300, 16, 1025], NB=220, max_new=200, seed=5)
    p, dev = cv.sess.pool, cv.sess.device
    st = torch.cuda.current_stream().cuda_stream
    for turn in range(3):
        n_new = [20 + turn, 33, 16, 64 - turn]
        cv.begin_turn(n_new)
        q_all, k_all, v_all = cv.make_inputs(n_new, 900 + turn)
        ref = cv.oracle_turn(q_all, k_all, v_all)
        for l in range(cv.L):
            dq, dk, dv = (bits_to_torch(x[l], dev) for x in (q_all, k_all, v_all))
            out = torch.zeros_like(dq)
            if mode == sc.SC_ATTN_STAGED:
                p.load_layer_batched(l, cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, l & 1, st)
            p.prefill_layer_batched(l, dq.data_ptr(), dk.data_ptr(), dv.data_ptr(), cv.tables_dev.data_ptr(),
                                    cv.max_blocks, cv.hist, cv.cu, l & 1, mode, out.data_ptr(), st)
            torch.cuda.synchronize()
            assert_close(torch_to_bits(out), ref[l], f"turn {turn} layer {l}")
        cv.end_turn(n_new)
        cv.check_pool_equals_logical()
    cv.sess.close()


@pytest.mark.parametrize("io_kind", [sc.SC_MEM_DEVICE, sc.SC_MEM_HOST_PINNED])
@pytest.mark.parametrize("mode", [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED])
def test_prefill_turn_pipeline(mode, io_kind):
    """a8: the two-stream, double-buffered pipeline over L layers, several turns issued back
    to back with no host synchronisation in between (PAPER.md:192 ordering rule)."""
    cv = Conversations(L=5, Hq=8, Hkv=2, D=128, hist=[700, 45], NB=200, max_new=160, seed=9)
    p, dev = cv.sess.pool, cv.sess.device
    refs, outs, keep = [], [], []
    for turn in range(3):
        n_new = [96, 40 + turn]
        cv.begin_turn(n_new)
        q_all, k_all, v_all = cv.make_inputs(n_new, 300 + turn, "peaked" if turn == 1 else "normal")
        refs.append(cv.oracle_turn(q_all, k_all, v_all))
        if io_kind == sc.SC_MEM_HOST_PINNED:
            tq, tk, tv = (bits_to_torch(x).pin_memory() for x in (q_all, k_all, v_all))
            out = torch.zeros(tq.shape, dtype=torch.bfloat16).pin_memory()
        else:
            tq, tk, tv = (bits_to_torch(x, dev) for x in (q_all, k_all, v_all))
            out = torch.zeros_like(tq)
            torch.cuda.synchronize()
        keep.append((tq, tk, tv))
        cv.sess.compute_stream.wait_stream(torch.cuda.current_stream())   # table upload, inputs
        p.prefill_turn(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out.data_ptr(), io_kind,
                       cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, mode,
                       cv.sess.copy_stream.cuda_stream, cv.sess.compute_stream.cuda_stream)
        outs.append(out)
        cv.end_turn(n_new)
        # tables_dev is rewritten by the next begin_turn on the current stream: order it
        torch.cuda.current_stream().wait_stream(cv.sess.compute_stream)
    torch.cuda.synchronize()
    for turn in range(3):
        for l in range(cv.L):
            assert_close(torch_to_bits(outs[turn][l]), refs[turn][l], f"turn {turn} layer {l}")
    cv.check_pool_equals_logical()
    cv.sess.close()


def test_host_pinned_pool_matches_oracle():
    """Config 4's second variant in miniature: the pool lives in pinned host memory (the PCIe
    reload path); gather, scatter and fused attention read and write it directly."""
    cv = Conversations(L=2, Hq=8, Hkv=2, D=128, hist=[333], NB=40, max_new=64, seed=21,
                       pool_kind=sc.SC_POOL_HOST_PINNED)
    p, dev = cv.sess.pool, cv.sess.device
    st = torch.cuda.current_stream().cuda_stream
    for turn, mode in enumerate([sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED]):
        n_new = [50]
        cv.begin_turn(n_new)
        q_all, k_all, v_all = cv.make_inputs(n_new, 40 + turn)
        ref = cv.oracle_turn(q_all, k_all, v_all)
        for l in range(cv.L):
            dq, dk, dv = (bits_to_torch(x[l], dev) for x in (q_all, k_all, v_all))
            out = torch.zeros_like(dq)
            if mode == sc.SC_ATTN_STAGED:
                p.load_layer_batched(l, cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, 0, st)
            p.prefill_layer_batched(l, dq.data_ptr(), dk.data_ptr(), dv.data_ptr(), cv.tables_dev.data_ptr(),
                                    cv.max_blocks, cv.hist, cv.cu, 0, mode, out.data_ptr(), st)
            torch.cuda.synchronize()
            assert_close(torch_to_bits(out), ref[l], f"host pool turn {turn} layer {l}")
        cv.end_turn(n_new)
        cv.check_pool_equals_logical()
    # the host copy itself holds the bytes (the CPU can see what the GPU scattered)
    raw = cv.sess.pool_mem.numpy().view(np.uint16)
    t, h, d = 370, 1, 77
    off = p.cell_offset(int(cv.tables[0][t // 16]), 1, 0, h, t % 16, d)
    assert raw[off // 2] == cv.logical[0][1][0][t, h, d]
    cv.sess.close()


@pytest.mark.parametrize("slow", ["copy", "compute"])
def test_pipeline_ordering_survives_a_slow_stream(slow):
    """PAPER.md:192 ordering rule (reading S8): attention(l) must wait for load(l), load(l+1) for
    attention(l-1).  One of the two streams is held up by a long busy kernel right before the
    turns are enqueued; if an event were missing, the other stream would run ahead and read an
    LSC buffer that is not loaded yet (or overwrite one that is still being read)."""
    cv = Conversations(L=6, Hq=4, Hkv=4, D=128, hist=[1500, 300], NB=260, max_new=200, seed=17)
    p, dev = cv.sess.pool, cv.sess.device
    refs, outs, keep = [], [], []
    for turn in range(2):
        n_new = [100, 37]
        cv.begin_turn(n_new)
        q_all, k_all, v_all = cv.make_inputs(n_new, 700 + turn)
        refs.append(cv.oracle_turn(q_all, k_all, v_all))
        tq, tk, tv = (bits_to_torch(x, dev) for x in (q_all, k_all, v_all))
        out = torch.zeros_like(tq)
        torch.cuda.synchronize()
        keep.append((tq, tk, tv))
        stream = cv.sess.copy_stream if slow == "copy" else cv.sess.compute_stream
        with torch.cuda.stream(stream):
            torch.cuda._sleep(int(2e8))                    # ~0.1 s of busy waiting on that stream
        p.prefill_turn(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out.data_ptr(), sc.SC_MEM_DEVICE,
                       cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, sc.SC_ATTN_STAGED,
                       cv.sess.copy_stream.cuda_stream, cv.sess.compute_stream.cuda_stream)
        outs.append(out)
        cv.end_turn(n_new)
        torch.cuda.current_stream().wait_stream(cv.sess.compute_stream)
        torch.cuda.current_stream().wait_stream(cv.sess.copy_stream)
    torch.cuda.synchronize()
    for turn in range(2):
        for l in range(cv.L):
            assert_close(torch_to_bits(outs[turn][l]), refs[turn][l], f"slow {slow}: turn {turn} layer {l}")
    cv.check_pool_equals_logical()
    cv.sess.close()


@pytest.mark.parametrize("slow", [None, "copy", "compute"])
@pytest.mark.parametrize("mode", [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED])
def test_single_buffer_paper_ordering(mode, slow):
    """f4 (Fig. 10 at :404): ONE LSC buffer, load(l+1) waits for attention(l) and the
    store of layer l, and hides behind what the model does next -- here a hook that puts a GEMM on
    the compute stream after every attention.  Same oracle, same answer bit for bit as the
    two-buffer schedule, also with one stream held up right before the turn."""
    cv = Conversations(L=6, Hq=4, Hkv=4, D=128, hist=[1500, 300], NB=260, max_new=200, seed=23)
    p, dev = cv.sess.pool, cv.sess.device
    n_new = [100, 37]
    cv.begin_turn(n_new)
    q_all, k_all, v_all = cv.make_inputs(n_new, 811)
    ref = cv.oracle_turn(q_all, k_all, v_all)
    tq, tk, tv = (bits_to_torch(x, dev) for x in (q_all, k_all, v_all))
    out2, out1 = torch.zeros_like(tq), torch.zeros_like(tq)
    wa = torch.randn(512, 512, device=dev)
    seen = []

    def hook(layer, stream_handle):
        assert stream_handle == cv.sess.compute_stream.cuda_stream
        seen.append(layer)
        with torch.cuda.stream(cv.sess.compute_stream):
            torch.matmul(wa, wa)                          # the "FFN" the load hides behind

    torch.cuda.synchronize()
    args = (sc.SC_MEM_DEVICE, cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, mode,
            cv.sess.copy_stream.cuda_stream, cv.sess.compute_stream.cuda_stream)
    p.prefill_turn(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out2.data_ptr(), *args)
    torch.cuda.synchronize()
    if slow:
        with torch.cuda.stream(cv.sess.copy_stream if slow == "copy" else cv.sess.compute_stream):
            torch.cuda._sleep(int(2e8))
    p.prefill_turn_ex(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out1.data_ptr(), *args,
                      lsc_buffers=1, after_attention=hook)
    torch.cuda.synchronize()
    assert seen == list(range(cv.L))
    assert torch.equal(out1.view(torch.int16), out2.view(torch.int16))
    for l in range(cv.L):
        assert_close(torch_to_bits(out1[l]), ref[l], f"single buffer, mode {mode}, slow {slow}: layer {l}")
    cv.end_turn(n_new)
    cv.check_pool_equals_logical()
    with pytest.raises(sc.SwiftCacheError):
        p.prefill_turn_ex(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out1.data_ptr(), *args, lsc_buffers=3)
    cv.sess.close()


def test_an_exception_in_the_layer_hook_reaches_the_caller():
    """A failing assertion inside after_attention must fail the call that ran it, not vanish on
    stderr: the binding keeps the hook's first exception, stops calling the hook, lets the library
    finish enqueuing the turn and re-raises.  The turn itself is still complete and correct."""
    cv = Conversations(L=4, Hq=4, Hkv=4, D=128, hist=[700], NB=80, max_new=64, seed=29)
    p, dev = cv.sess.pool, cv.sess.device
    n_new = [50]
    cv.begin_turn(n_new)
    q_all, k_all, v_all = cv.make_inputs(n_new, 912)
    ref = cv.oracle_turn(q_all, k_all, v_all)
    tq, tk, tv = (bits_to_torch(x, dev) for x in (q_all, k_all, v_all))
    out = torch.zeros_like(tq)
    seen = []

    def hook(layer, stream_handle):
        seen.append(layer)
        assert layer != 1, "layer 1 went wrong"

    torch.cuda.synchronize()
    with pytest.raises(AssertionError, match="layer 1 went wrong"):
        p.prefill_turn_ex(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out.data_ptr(), sc.SC_MEM_DEVICE,
                          cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, sc.SC_ATTN_STAGED,
                          cv.sess.copy_stream.cuda_stream, cv.sess.compute_stream.cuda_stream,
                          lsc_buffers=1, after_attention=hook)
    torch.cuda.synchronize()
    assert seen == [0, 1]                                   # not called again after it failed
    for l in range(cv.L):
        assert_close(torch_to_bits(out[l]), ref[l], f"turn with a failing hook: layer {l}")
    cv.end_turn(n_new)
    cv.check_pool_equals_logical()
    cv.sess.close()


@pytest.mark.parametrize("mode", [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED])
def test_a_turn_is_capturable_into_a_cuda_graph(mode):
    """a turn is 32 layers x 2-3 launches plus ~4 event operations per layer
    from the host; captured once into a CUDA graph it is replayed with ONE launch.  sc_prefill_turn is
    capturable as it stands once the first (warm-up) turn has set the kernel attributes: it allocates
    nothing, and the copy stream forks from and joins the compute stream through the pool's events, which
    is exactly the ordering of PAPER.md:192.  Checked: a replay gives the eager turn's bits, and a replay
    after the inputs were overwritten in place gives the eager bits and the oracle's values for those."""
    import copy
    cv = Conversations(L=5, Hq=4, Hkv=4, D=128, hist=[900, 260], NB=200, max_new=256, seed=41)
    p, dev = cv.sess.pool, cv.sess.device
    n_new = [200, 56]
    cv.begin_turn(n_new)
    saved = copy.deepcopy(cv.logical)
    a = cv.make_inputs(n_new, 1201)
    b = cv.make_inputs(n_new, 1202, variant="peaked")
    tq, tk, tv = (bits_to_torch(x, dev) for x in a)
    out = torch.zeros_like(tq)
    args = (tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out.data_ptr(), sc.SC_MEM_DEVICE, cv.tables_dev.data_ptr(),
            cv.max_blocks, cv.hist, cv.cu, mode, cv.sess.copy_stream.cuda_stream, cv.sess.compute_stream.cuda_stream)
    p.prefill_turn(*args)                                   # eager, inputs A (also the warm-up)
    torch.cuda.synchronize()
    eager_a = out.clone()
    ref_a = cv.oracle_turn(*a)
    for l in range(cv.L):
        assert_close(torch_to_bits(eager_a[l]), ref_a[l], f"eager turn, mode {mode}, layer {l}")

    graph = torch.cuda.CUDAGraph()
    launches_before = p.launch_count()
    with torch.cuda.graph(graph, stream=cv.sess.compute_stream):
        p.prefill_turn(*args)
    captured_launches = p.launch_count() - launches_before
    assert captured_launches >= cv.L                        # the whole turn went into the graph
    out.zero_()
    torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int16), eager_a.view(torch.int16))

    for dst, src in zip((tq, tk, tv), b):                   # new inputs, same addresses
        dst.copy_(bits_to_torch(src, dev))
    out.zero_()
    torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    graph_b = out.clone()
    p.prefill_turn(*args)
    torch.cuda.synchronize()
    assert torch.equal(graph_b.view(torch.int16), out.view(torch.int16))
    cv.logical = saved                                      # the turn was redone with inputs B over the same slots
    ref_b = cv.oracle_turn(*b)
    for l in range(cv.L):
        assert_close(torch_to_bits(graph_b[l]), ref_b[l], f"graph replay, mode {mode}, layer {l}")
    cv.end_turn(n_new)
    cv.check_pool_equals_logical()
    del graph
    cv.sess.close()


def test_block_major_resize_on_the_device():
    """f1: growing the pool appends blocks and releasing the tail frees them;
    no existing block moves -- the conversation's KV reads back bit-exactly through the same
    table before and after, and the appended blocks are usable at once."""
    L, Hkv, D, B = 3, 2, 128, 16
    cfg = sc.make_config(L, 4, Hkv, D, B, 8, 0, 64)
    pool_bytes8, _ = sc.sc_pool_bytes_required(cfg)
    region = torch.full((pool_bytes8 // 8 * 12 + 1024,), 0x5A, dtype=torch.uint8, device="cuda")   # room for 12 blocks, dirty
    off = (-region.data_ptr()) % 1024
    base = region.data_ptr() + off
    p = sc.Pool(cfg, base, pool_bytes8, 0, 0)
    table = p.alloc_blocks(6)
    tdev = torch.from_numpy(table.copy()).cuda()
    T = 6 * B - 5
    ks = [bits_to_torch(I.normal_bf16((T, Hkv, D), 300 + l), "cuda") for l in range(L)]
    vs = [bits_to_torch(I.normal_bf16((T, Hkv, D), 400 + l), "cuda") for l in range(L)]
    for l in range(L):
        p.store_prefix(l, ks[l].data_ptr(), vs[l].data_ptr(), 0, T, tdev.data_ptr(), 6)

    def read(l, tab, n_tab, start, n):
        k = torch.empty((n, Hkv, D), dtype=torch.bfloat16, device="cuda")
        v = torch.empty_like(k)
        p.read_tokens(l, 0, tab.data_ptr(), n_tab, 0, start, n, k.data_ptr(), v.data_ptr())
        torch.cuda.synchronize()
        return k, v

    p.resize(12, pool_bytes8 // 8 * 12)                        # grow: O(1), nothing moves
    torch.cuda.synchronize()
    for l in range(L):
        k, v = read(l, tdev, 6, 0, T)
        assert torch.equal(k.view(torch.int16), ks[l].view(torch.int16)) and torch.equal(v.view(torch.int16), vs[l].view(torch.int16))
    raw = region[off:off + pool_bytes8 // 8 * 12]
    assert int(raw[pool_bytes8:].max()) == 0                   # the appended tail was zero-filled
    # the conversation grows into the appended blocks
    more = p.alloc_blocks(4)
    assert sorted(more.tolist()) == [6, 7, 8, 9]               # old free ids first, then the new ones
    table2 = np.concatenate([table, more]).astype(np.int32)
    t2 = torch.from_numpy(table2).cuda()
    kn = bits_to_torch(I.normal_bf16((4 * B, Hkv, D), 500), "cuda")
    vn = bits_to_torch(I.normal_bf16((4 * B, Hkv, D), 501), "cuda")
    p.store_prefix(1, kn.data_ptr(), vn.data_ptr(), T, 4 * B, t2.data_ptr(), 10)
    k, v = read(1, t2, 10, 0, T + 4 * B)
    assert torch.equal(k.view(torch.int16), torch.cat([ks[1], kn]).view(torch.int16))
    assert torch.equal(v.view(torch.int16), torch.cat([vs[1], vn]).view(torch.int16))
    # release the tail: refused while block 9 is in use, fine once the tail is free
    with pytest.raises(sc.SwiftCacheError):
        p.resize(9)
    p.free_blocks(more[more >= 8])
    p.resize(8)                                                # blocks 6 and 7 stay allocated
    for l in range(L):
        k, v = read(l, tdev, 6, 0, T)
        assert torch.equal(k.view(torch.int16), ks[l].view(torch.int16))
    p.destroy()


def test_elastic_exchange_between_master_and_worker_pools():
    """f1, both sides of the exchange ("whenever the master scales by MEU_m blocks the
    i-th worker must simultaneously scale by MEU_i").  One borrowed region is the memory budget of a
    worker GPU; an LWM-1M-Text-shaped master pool (32 layers x 32 kv heads: 8 MiB per block) and a
    Qwen3-14B-shaped worker pool (40 layers x 8 kv heads: 2.5 MiB per block) are carved from it.
    sc_scale_up's answer drives sc_pool_resize on BOTH: the worker gains d_worker blocks, the
    master gives up d_master; the two byte counts are equal to the byte (MEU_m * BE_m = MEU_i * BE_i,
    Eq. 8-9), so the budget is conserved, and neither pool moves a block: both conversations read
    back bit-exactly through their old tables, the worker's new blocks are usable at once."""
    mcfg = sc.make_config(32, 32, 32, 128, 16, 15, 0, 64)
    wcfg = sc.make_config(40, 32, 8, 128, 16, 16, 0, 64)
    meu_m, meu_w = sc.sc_elastic_units(mcfg, wcfg)
    assert (meu_m, meu_w) == (5, 16)
    m_bytes, _ = sc.sc_pool_bytes_required(mcfg)
    w_bytes, _ = sc.sc_pool_bytes_required(wcfg)
    bbm, bbw = m_bytes // 15, w_bytes // 16
    assert meu_m * bbm == meu_w * bbw == 40 << 20                  # one elastic unit: the same 40 MiB on both sides
    # the worker's share starts where the master's 15 blocks end and has room for the unit it may gain
    region = torch.empty(m_bytes + w_bytes + meu_w * bbw + 1024, dtype=torch.uint8, device="cuda")
    base = region.data_ptr() + (-region.data_ptr()) % 1024
    master = sc.Pool(mcfg, base, m_bytes, 0, 0)
    worker = sc.Pool(wcfg, base + m_bytes, w_bytes, 0, 0)
    budget = master.info().pool_bytes + worker.info().pool_bytes

    def fill(pool, cfg_, n_blocks, seed):
        ids = pool.alloc_blocks(n_blocks)
        tdev = torch.from_numpy(ids.copy()).cuda()
        T = n_blocks * 16 - 3
        data = {}
        for l in (0, cfg_.n_layers - 1):
            k = bits_to_torch(I.normal_bf16((T, cfg_.n_kv_heads, 128), seed + l), "cuda")
            v = bits_to_torch(I.normal_bf16((T, cfg_.n_kv_heads, 128), seed + 50 + l), "cuda")
            pool.store_prefix(l, k.data_ptr(), v.data_ptr(), 0, T, tdev.data_ptr(), len(ids))
            data[l] = (k, v)
        torch.cuda.synchronize()
        return ids, tdev, T, data

    def check(pool, cfg_, tdev, T, data):
        for l, (k, v) in data.items():
            ko, vo = torch.empty_like(k), torch.empty_like(v)
            pool.read_tokens(l, 0, tdev.data_ptr(), tdev.numel(), 0, 0, T, ko.data_ptr(), vo.data_ptr())
            torch.cuda.synchronize()
            assert torch.equal(ko.view(torch.int16), k.view(torch.int16))
            assert torch.equal(vo.view(torch.int16), v.view(torch.int16))

    m_ids, m_t, m_T, m_data = fill(master, mcfg, 8, 700)           # ids 0..7: the master's tail stays free
    w_ids, w_t, w_T, w_data = fill(worker, wcfg, 16, 900)          # the worker is full
    # a 400-token request arrives at the worker: it holds 16 blocks, needs 25
    d_w, d_m = sc.sc_scale_up(16, 16, meu_w, meu_m, 400)
    assert (d_w, d_m) == (16, 5) and d_w * bbw == d_m * bbm
    master.resize(15 - d_m)                                        # releases blocks 10..14 (free), moves nothing
    worker.resize(16 + d_w, w_bytes + d_w * bbw)                   # appends blocks 16..31
    assert master.info().pool_bytes + worker.info().pool_bytes == budget
    assert m_bytes - master.info().pool_bytes == worker.info().pool_bytes - w_bytes == d_m * bbm
    check(master, mcfg, m_t, m_T, m_data)
    check(worker, wcfg, w_t, w_T, w_data)
    new_ids, n_t, n_T, n_data = fill(worker, wcfg, d_w, 1100)      # the new blocks hold a second conversation
    assert sorted(new_ids.tolist()) == list(range(16, 32))
    check(worker, wcfg, n_t, n_T, n_data)
    check(worker, wcfg, w_t, w_T, w_data)
    with pytest.raises(sc.SwiftCacheError):
        master.cell_offset(10, 0, 0, 0, 0, 0)                      # gone from the master
    # and back: the request is gone, nothing longer than 250 tokens was seen lately
    worker.free_blocks(new_ids)
    b_w, b_m = sc.sc_scale_down(32, 16, meu_w, meu_m, 250)
    assert (b_w, b_m) == (16, 5)
    worker.resize(32 - b_w)
    master.resize(10 + b_m, m_bytes)
    assert master.info().pool_bytes + worker.info().pool_bytes == budget
    check(master, mcfg, m_t, m_T, m_data)
    check(worker, wcfg, w_t, w_T, w_data)
    master.destroy()
    worker.destroy()
