"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle on the
same seeded inputs.  KV movement and block-table indexing bit-exact; bf16 attention
within max-abs 1e-2 and relative-L2 5e-3 of the fp32 oracle (BASELINE.json)."""
import numpy as np
import pytest
import torch

from oracle import sc_oracle as O
from paper_2606_16135_b200 import binding as sc
from paper_2606_16135_b200 import build as sc_build
from paper_2606_16135_b200 import inputs as I
from paper_2606_16135_b200.runtime import Session, bits_to_torch, torch_to_bits

from gpu_util import Case, assert_close, errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="session", autouse=True)
def _built():
    sc_build.build()
    assert sc.lib() is not None


MODES = [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED]


# ------------------------------------------------------------------ KV movement
def test_store_prefix_places_every_element_where_the_accessor_says():
    """a3 + the logical accessor: raw pool bytes at sc_cell_offset == the oracle's pool."""
    c = Case(L=2, Hq=4, Hkv=4, D=64, T_h=509, n=0, NB=64, seed=3)
    raw = c.sess.pool_mem.cpu().numpy().view(np.uint16)
    rng = np.random.default_rng(0)
    for l in range(2):
        for kv in range(2):
            want = c.opool.gather(l, kv, c.table, 509)
            for _ in range(400):
                t, h, d = int(rng.integers(509)), int(rng.integers(4)), int(rng.integers(64))
                off = c.sess.pool.cell_offset(int(c.table[t // 16]), l, kv, h, t % 16, d)
                assert raw[off // 2] == want[t, h, d]
    # blocks outside the table were never touched (pool zero-filled at create)
    other = np.setdiff1d(np.arange(64), c.table)
    bb = c.sess.pool.info().block_bytes
    for b in other[:8]:
        assert not raw[b * bb // 2:(b + 1) * bb // 2].any()
    c.close()


@pytest.mark.parametrize("D,Hkv,T", [(64, 4, 509), (128, 2, 300), (128, 8, 16), (64, 1, 1)])
def test_I1_store_then_read_is_bit_exact(D, Hkv, T):
    c = Case(L=2, Hq=8, Hkv=Hkv, D=D, T_h=T, n=0, NB=40, seed=5)
    for l in range(2):
        k, v = c.sess.read_tokens(l, 0, c.table_dev, 0, T)
        assert np.array_equal(torch_to_bits(k), c.data[l][1]) and np.array_equal(torch_to_bits(v), c.data[l][2])
        assert np.array_equal(torch_to_bits(k), c.opool.gather(l, 0, c.table, T))
        k2, v2 = c.sess.read_tokens(l, 0, c.table_dev, T // 2, T - T // 2)      # mid-block start
        assert np.array_equal(torch_to_bits(v2), c.data[l][2][T // 2:])
    c.close()


@pytest.mark.parametrize("engine", [sc.SC_COPY_LDG, sc.SC_COPY_BULK])
@pytest.mark.parametrize("D,Hkv,T", [(64, 4, 512), (128, 32, 200), (128, 8, 333), (64, 1, 17)])
def test_I1_load_layer_gathers_history_bit_exact(engine, D, Hkv, T):
    """a4: LSC[buf] holds the logically contiguous history after the paged gather."""
    c = Case(L=2, Hq=32, Hkv=Hkv, D=D, T_h=T, n=0, NB=48, seed=7)
    c.sess.pool.set_engine(sc.SC_ENGINE_AUTO, engine)
    st = torch.cuda.current_stream().cuda_stream
    for l, buf in ((0, 0), (1, 1), (0, 1)):
        c.sess.pool.load_layer(l, c.table_dev.data_ptr(), len(c.table), T, buf, st)
        k, v = c.sess.read_tokens(l, 1 + buf, None, 0, T)
        assert np.array_equal(torch_to_bits(k), c.data[l][1]) and np.array_equal(torch_to_bits(v), c.data[l][2])
    # whole-cell equality: LSC block j == pool cell (table[j], layer) byte for byte
    info = c.sess.pool.info()
    c.sess.pool.load_layer(1, c.table_dev.data_ptr(), len(c.table), T, 0, st)
    torch.cuda.synchronize()
    pool_raw, lsc_raw = c.sess.pool_mem.cpu().numpy(), c.sess.lsc_mem.cpu().numpy()
    for j in range(O.blocks_for(T, 16)):
        src = int(c.table[j]) * info.block_bytes + 1 * info.cell_bytes
        assert np.array_equal(lsc_raw[j * info.cell_bytes:(j + 1) * info.cell_bytes],
                              pool_raw[src:src + info.cell_bytes])
    c.close()


# ------------------------------------------------------------------ attention
@pytest.mark.parametrize("mode", MODES)
def test_tiny_config_matches_oracle(mode):
    """BASELINE.json config 1: 2 layers, 4 heads, D 64, 512 history in a 64-block pool, 32 new."""
    c = Case(L=2, Hq=4, Hkv=4, D=64, T_h=512, n=32, NB=64, seed=16135)
    for l in range(2):
        got = c.run_layer(l, mode, buf=l & 1)
        assert_close(got, c.oracle_layer(l), f"layer {l}")
        # I2: the turn's K/V were scattered back: pool now holds [history ; new] bit-exactly
        k, v = c.sess.read_tokens(l, 0, c.table_dev, 0, 544)
        assert np.array_equal(torch_to_bits(k), c.opool.gather(l, 0, c.table, 544))
        assert np.array_equal(torch_to_bits(v), np.concatenate([c.data[l][2], c.data[l][4]]))
        if mode == sc.SC_ATTN_STAGED:
            k, v = c.sess.read_tokens(l, 1 + (l & 1), None, 0, 544)
            assert np.array_equal(torch_to_bits(k), np.concatenate([c.data[l][1], c.data[l][3]]))
    c.close()


@pytest.mark.parametrize("T_h", [0, 1, 15, 16, 17, 509])
@pytest.mark.parametrize("n", [1, 31, 32, 33, 256])
def test_edge_lengths(T_h, n):
    mode = MODES[(T_h + n) % 2]
    c = Case(L=1, Hq=4, Hkv=4, D=64, T_h=T_h, n=n, NB=64, seed=1000 + T_h * 7 + n)
    assert_close(c.run_layer(0, mode), c.oracle_layer(0), f"T_h={T_h} n={n}")
    k, v = c.sess.read_tokens(0, 0, c.table_dev, 0, T_h + n)
    assert np.array_equal(torch_to_bits(k), c.opool.gather(0, 0, c.table, T_h + n))
    c.close()


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("variant", ["normal", "peaked", "adversarial"])
@pytest.mark.parametrize("Hq,Hkv,D", [(8, 2, 128), (4, 4, 128), (8, 8, 64), (4, 1, 64)])
def test_shapes_and_score_distributions(mode, variant, Hq, Hkv, D):
    """GQA 4:1, MHA, D 64/128; peaked and adversarial scores force the running-max rescale."""
    c = Case(L=1, Hq=Hq, Hkv=Hkv, D=D, T_h=700, n=70, NB=64, seed=77, variant=variant)
    assert_close(c.run_layer(0, mode), c.oracle_layer(0), f"{variant} {Hq}/{Hkv}/{D}")
    c.close()


@pytest.mark.parametrize("split_tiles", [1, 2, 3, 5, 1000])
def test_split_kv_and_combine(split_tiles):
    """a7: any partition of the keys gives the same answer within tolerance, including
    partitions whose last split is fully masked for the first rows."""
    c = Case(L=1, Hq=4, Hkv=2, D=128, T_h=777, n=200, NB=80, seed=91, variant="peaked",
             split_tiles=split_tiles)
    ref = c.oracle_layer(0)
    assert_close(c.run_layer(0, sc.SC_ATTN_FUSED), ref, f"split_tiles={split_tiles}")
    c.close()


def test_I5_block_permutation_gives_bit_identical_output():
    """I5 on the GPU: work partitioning depends on logical positions only."""
    outs = []
    for perm_id, ident in ((1, False), (2, False), (1, True)):
        c = Case(L=1, Hq=8, Hkv=2, D=128, T_h=1000, n=100, NB=96, seed=55, perm_id=perm_id, identity=ident)
        outs.append((c.run_layer(0, sc.SC_ATTN_FUSED), c.run_layer(0, sc.SC_ATTN_STAGED)))
        c.close()
    for fused, staged in outs[1:]:
        assert np.array_equal(fused, outs[0][0]) and np.array_equal(staged, outs[0][1])
    assert np.array_equal(outs[0][0], outs[0][1])          # same kernel, identity table over the LSC


def test_softmax_invariants_on_gpu():
    """I4 through the CUDA path: V == 1 gives exactly 1.0; q == 0 gives the running mean of V."""
    c = Case(L=1, Hq=4, Hkv=2, D=64, T_h=300, n=40, NB=32, seed=66)
    q, kh, vh, kn, vn = c.data[0]
    ones = np.full_like(vh, 0x3F80)
    c.sess.store_prefix(0, bits_to_torch(kh, c.sess.device), bits_to_torch(ones, c.sess.device), 0, c.table_dev)
    c.data[0] = (q, kh, ones, kn, np.full_like(vn, 0x3F80))
    got = I.bf16_bits_to_f32(c.run_layer(0, sc.SC_ATTN_FUSED))
    assert np.abs(got - 1).max() <= 2 ** -8
    c.close()
    c = Case(L=1, Hq=4, Hkv=2, D=64, T_h=45, n=9, NB=8, seed=67)
    q, kh, vh, kn, vn = c.data[0]
    c.data[0] = (np.zeros_like(q), kh, vh, kn, vn)
    got = I.bf16_bits_to_f32(c.run_layer(0, sc.SC_ATTN_STAGED))
    V = I.bf16_bits_to_f32(np.concatenate([vh, vn])).astype(np.float64)
    for i in range(9):
        want = V[:45 + i + 1].mean(axis=0)
        for h in range(4):
            assert np.abs(got[i, h] - want[h // 2]).max() < 4e-3
    c.close()


# ------------------------------------------------------------------ errors
def test_argument_errors_launch_nothing():
    c = Case(L=1, Hq=4, Hkv=4, D=64, T_h=64, n=16, NB=16, seed=1)
    p, t = c.sess.pool, c.table_dev
    before = p.launch_count()
    x = torch.zeros(16 * 4 * 64, dtype=torch.bfloat16, device=c.sess.device).data_ptr()
    bad = [
        (sc.SC_ERR_INVALID_ARG, lambda: p.prefill_layer(1, x, x, x, t.data_ptr(), len(c.table), 64, 16, 0, 1, x)),
        (sc.SC_ERR_CAPACITY, lambda: p.prefill_layer(0, x, x, x, t.data_ptr(), 4, 64, 16, 0, 1, x)),
        (sc.SC_ERR_CAPACITY, lambda: p.prefill_layer(0, x, x, x, t.data_ptr(), len(c.table), 64, 17, 0, 1, x)),
        (sc.SC_ERR_INVALID_ARG, lambda: p.prefill_layer(0, 0, x, x, t.data_ptr(), len(c.table), 64, 16, 0, 1, x)),
        (sc.SC_ERR_INVALID_ARG, lambda: p.prefill_layer(0, x, x, x, t.data_ptr(), len(c.table), 64, 16, 2, 0, x)),
        (sc.SC_ERR_CAPACITY, lambda: p.load_layer(0, t.data_ptr(), 2, 64, 0)),
        (sc.SC_ERR_CAPACITY, lambda: p.store_prefix(0, x, x, 0, 16 * 6, t.data_ptr(), len(c.table))),
    ]
    for status, call in bad:
        with pytest.raises(sc.SwiftCacheError) as e:
            call()
        assert e.value.status == status, str(e.value)
    assert p.launch_count() == before
    c.close()


# ------------------------------------------------------------------ f3: regular cache + LSC
@pytest.mark.parametrize("resident", [1, 7, 10_000])
def test_resident_leading_blocks_are_read_in_place(resident):
    """the first N_RC blocks of a conversation stay resident; only the rest is
    gathered into the LSC.  Same answer as streaming everything (bit for bit: same kernel, same
    partitioning), and the LSC cells of the resident blocks are never written."""
    T_h, n = 333, 70                                             # 20 complete history blocks + 13 tokens
    base = Case(L=2, Hq=8, Hkv=2, D=128, T_h=T_h, n=n, NB=64, seed=88)
    want = [base.run_layer(l, sc.SC_ATTN_STAGED, buf=l & 1) for l in range(2)]
    refs = [base.oracle_layer(l) for l in range(2)]
    base.close()
    c = Case(L=2, Hq=8, Hkv=2, D=128, T_h=T_h, n=n, NB=64, seed=88)
    c.sess.pool.set_resident_blocks(resident)
    rc = min(resident, T_h // 16)
    info = c.sess.pool.info()
    for l in range(2):
        got = c.run_layer(l, sc.SC_ATTN_STAGED, buf=l & 1)
        assert np.array_equal(got, want[l])
        assert_close(got, refs[l], f"resident {resident} layer {l}")
        lsc = c.sess.lsc_mem.cpu().numpy()
        buf0 = (l & 1) * info.lsc_buffer_bytes
        assert not lsc[buf0:buf0 + rc * info.cell_bytes].any()                   # resident blocks: not gathered
        assert lsc[buf0 + rc * info.cell_bytes:buf0 + (rc + 1) * info.cell_bytes].any()   # the next one was
        k, v = c.sess.read_tokens(l, 0, c.table_dev, 0, T_h + n)                 # I2 still holds
        assert np.array_equal(torch_to_bits(k), np.concatenate([c.data[l][1], c.data[l][3]]))
        assert np.array_equal(torch_to_bits(v), np.concatenate([c.data[l][2], c.data[l][4]]))
    before = c.sess.pool.launch_count()
    with pytest.raises(sc.SwiftCacheError) as e:                                 # mma.sync engine: not supported
        c.sess.pool.set_engine(sc.SC_ENGINE_MMA_SYNC, sc.SC_COPY_AUTO)
        c.run_layer(0, sc.SC_ATTN_STAGED, load=False)
    assert e.value.status == sc.SC_ERR_UNSUPPORTED
    assert c.sess.pool.launch_count() == before                                  # refused before anything was launched
    c.close()


# ------------------------------------------------------------------ memory that was never cleared
@pytest.mark.parametrize("engine", [sc.SC_ENGINE_TCGEN05, sc.SC_ENGINE_MMA_SYNC])
@pytest.mark.parametrize("T_h,n,split_tiles", [(333, 70, 0), (1000, 255, 2), (2049, 257, 8), (5, 3, 0)])
def test_pool_and_lsc_prefilled_with_nan(engine, T_h, n, split_tiles):
    """sc_pool_create(zero_fill = 0) over memory full of bf16 NaNs (0x7FC0 is not expressible as one
    byte, 0xFF 0xFF = a NaN with every bit set): slots the conversation never wrote -- the tail of the
    last block, unused blocks, stale LSC cells -- are masked in S, but P = 0 times a NaN V would still
    poison the row.  The scatter zero-fills the rest of the last block, so the output must be finite
    and within tolerance in both modes, with one CTA per pair, clusters and plain split-KV."""
    for mode in (sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED):
        c = Case(L=1, Hq=4, Hkv=2, D=128, T_h=T_h, n=n, NB=200, seed=991 + T_h, engine=engine,
                 split_tiles=split_tiles, zero_fill=False, fill_byte=0xFF)
        got = c.run_layer(0, mode)
        assert not np.isnan(I.bf16_bits_to_f32(got)).any(), f"NaN in the output, mode {mode}"
        assert_close(got, c.oracle_layer(0), f"nan-filled pool, engine {engine} mode {mode} T_h {T_h} n {n}")
        k, v = c.sess.read_tokens(0, 0, c.table_dev, 0, T_h + n)                 # I2: the written tokens, bit-exact
        assert np.array_equal(torch_to_bits(k), np.concatenate([c.data[0][1], c.data[0][3]]))
        assert np.array_equal(torch_to_bits(v), np.concatenate([c.data[0][2], c.data[0][4]]))
        c.close()


@pytest.mark.parametrize("Hq,T_h,n,split_tiles,what", [
    (4, 333, 70, 0, "one CTA per pair"),
    (4, 100, 256, 0, "one CTA per pair, full query pair"),
    (4, 1000, 255, 2, "forced cluster of 5"),
    (4, 2049, 130, 3, "forced cluster of 6, second query tile nearly empty"),
    (32, 5117, 250, 0, "lwm_5k layer shape, the split the heuristic picks"),
])
def test_folded_scatter_pads_over_nan_memory(Hq, T_h, n, split_tiles, what):
    """The headline path: Hq == Hkv and n <= 256, where the tcgen05 kernel stores the new K/V ITSELF
    (one CTA per pair, or the CTAs of a cluster sharing the rows) and must also zero the rest of the
    last block -- over a pool and an LSC full of NaN bits, with T_h + n not a multiple of 16.  The
    launch count proves the scatter kernel did not run; the output must be finite and match the
    oracle; the written tokens are bit-exact and the tail of the last block reads back as zeros,
    in the pool and (staged) in the LSC."""
    assert (T_h + n) % 16 != 0
    tail = 16 - (T_h + n) % 16
    for mode in (sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED):
        c = Case(L=1, Hq=Hq, Hkv=Hq, D=128, T_h=T_h, n=n, NB=400, seed=7300 + T_h, engine=sc.SC_ENGINE_TCGEN05,
                 split_tiles=split_tiles, zero_fill=False, fill_byte=0xFF)
        before = c.sess.pool.launch_count()
        got = c.run_layer(0, mode)
        launches = c.sess.pool.launch_count() - before
        assert launches == (2 if mode == sc.SC_ATTN_STAGED else 1), (what, mode, launches)   # (gather +) attention only
        assert not np.isnan(I.bf16_bits_to_f32(got)).any(), f"NaN in the output: {what}, mode {mode}"
        assert_close(got, c.oracle_layer(0), f"folded scatter over NaN memory: {what}, mode {mode}")
        srcs = [0] + ([1] if mode == sc.SC_ATTN_STAGED else [])      # the pool; LSC buffer 0 too when staged
        for src in srcs:
            k, v = c.sess.read_tokens(0, src, c.table_dev, 0, T_h + n + tail)
            k, v = torch_to_bits(k), torch_to_bits(v)
            assert np.array_equal(k[:T_h + n], np.concatenate([c.data[0][1], c.data[0][3]])), (what, mode, src)
            assert np.array_equal(v[:T_h + n], np.concatenate([c.data[0][2], c.data[0][4]])), (what, mode, src)
            assert not k[T_h + n:].any() and not v[T_h + n:].any(), f"tail of the last block not zeroed: {what} src {src}"
        c.close()


# ------------------------------------------------------------------ f2: a pool behind a peer pointer
def test_peer_pool_kind_routes_like_hbm():
    """the donor pool is another GPU's memory,
    mapped by the caller and handed over as pool_base with pool_kind = SC_POOL_PEER.  One GPU is
    all a test can have, so the "peer" region here is a second local allocation the session does
    not own; what is checked is that every call takes the pointer as it is: store, gather,
    scatter, staged and fused attention against the oracle, and the raw bytes of the region."""
    L, Hq, Hkv, D, B, NB, T_h, n = 2, 8, 2, 128, 16, 48, 333, 70
    cfg = sc.make_config(L, Hq, Hkv, D, B, NB, 32, n, pool_kind=sc.SC_POOL_PEER)
    pool_bytes, _ = sc.sc_pool_bytes_required(cfg)
    region = torch.full((pool_bytes + 1024,), 0xFF, dtype=torch.uint8, device="cuda")    # never cleared: NaN bits
    ptr = region.data_ptr() + (-region.data_ptr()) % 1024
    sess = Session(L, Hq, Hkv, D, B, NB, 32, n, pool_kind=sc.SC_POOL_PEER, pool_ptr=ptr, zero_fill=False)
    table = I.block_table(3, NB, O.blocks_for(T_h + n, B))
    tdev = sess.table_dev(table)
    opool = O.Pool(L, Hkv, D, B, NB)
    st = torch.cuda.current_stream().cuda_stream
    for l in range(L):
        q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 4242 + l)
        sess.store_prefix(l, bits_to_torch(kh, sess.device), bits_to_torch(vh, sess.device), 0, tdev)
        opool.store(l, 0, kh, 0, table)
        opool.store(l, 1, vh, 0, table)
        ref = O.prefill_layer(opool, l, q, kn, vn, table, T_h)
        dq, dk, dv = (bits_to_torch(x, sess.device) for x in (q, kn, vn))
        for mode in (sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED):
            out = torch.zeros((n, Hq, D), dtype=torch.bfloat16, device=sess.device)
            if mode == sc.SC_ATTN_STAGED:
                sess.pool.load_layer(l, tdev.data_ptr(), len(table), T_h, l & 1, st)
            sess.pool.prefill_layer(l, dq.data_ptr(), dk.data_ptr(), dv.data_ptr(), tdev.data_ptr(), len(table),
                                    T_h, n, l & 1, mode, out.data_ptr(), st)
            torch.cuda.synchronize()
            assert_close(torch_to_bits(out), ref, f"peer pool, layer {l} mode {mode}")
        k, v = sess.read_tokens(l, 0, tdev, 0, T_h + n)
        assert np.array_equal(torch_to_bits(k), opool.gather(l, 0, table, T_h + n))
        assert np.array_equal(torch_to_bits(v), opool.gather(l, 1, table, T_h + n))
    # the bytes are in the caller's region, where sc_cell_offset says
    raw = region.cpu().numpy()[ptr - region.data_ptr():].view(np.uint16)
    t, h, d = 350, 1, 77
    off = sess.pool.cell_offset(int(table[t // 16]), 1, 0, h, t % 16, d)
    assert raw[off // 2] == opool.gather(1, 0, table, T_h + n)[t, h, d]
    sess.close()
