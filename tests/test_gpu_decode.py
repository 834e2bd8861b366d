"""GPU parity of the decode engine (sc_attn_decode.cu: a few new tokens per conversation, one CTA per
(split, KV head, conversation), 16 padded rows = new tokens x query heads of the group) against the
CPU oracle through the C ABI -- SURVEY.md 8(f) row f4 "decode (n = 1) over the pool".  Shapes put the
causal boundary at every position of a 16-token block and a 64-token tile, use one to sixteen rows,
grouped-query heads (the group's heads share one pass over K/V), forced and automatic splits (in-CTA
merge of the four warps, then sc_combine_kernel), both modes, uncleared memory, and a ragged batch."""
import numpy as np
import pytest
import torch

from paper_2606_16135_b200 import binding as sc
from paper_2606_16135_b200 import build as sc_build
from paper_2606_16135_b200 import inputs as I
from paper_2606_16135_b200.runtime import bits_to_torch, torch_to_bits

from gpu_util import Case, assert_close

pytestmark = pytest.mark.gpu
MODES = [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED]


@pytest.fixture(scope="module", autouse=True)
def _built():
    sc_build.build()


@pytest.mark.parametrize("D", [64, 128])
@pytest.mark.parametrize("T_h", [0, 1, 15, 16, 17, 63, 64, 65, 509, 2049])
def test_one_new_token(D, T_h):
    c = Case(L=1, Hq=4, Hkv=4, D=D, T_h=T_h, n=1, NB=160, seed=5000 + T_h, engine=sc.SC_ENGINE_DECODE)
    for mode in MODES:
        assert_close(c.run_layer(0, mode), c.oracle_layer(0), f"decode D={D} T_h={T_h} mode={mode}")
    c.close()


@pytest.mark.parametrize("Hq,Hkv,n", [(8, 2, 1), (8, 2, 4), (8, 2, 3), (4, 4, 16), (4, 4, 7), (4, 2, 8), (8, 1, 2)])
@pytest.mark.parametrize("T_h", [40, 1000])
def test_rows_are_tokens_times_group_heads(Hq, Hkv, n, T_h):
    """Row r of a KV head's CTA is (new token r / G, query head hk*G + r % G): up to 16 rows, every row
    with its own causal limit T_h + token."""
    c = Case(L=1, Hq=Hq, Hkv=Hkv, D=128, T_h=T_h, n=n, NB=80, seed=5100 + T_h + n + Hq, variant="peaked",
             engine=sc.SC_ENGINE_DECODE)
    mode = MODES[(n + T_h // 40) % 2]
    assert_close(c.run_layer(0, mode), c.oracle_layer(0), f"decode Hq={Hq} Hkv={Hkv} n={n} T_h={T_h}")
    c.close()


@pytest.mark.parametrize("variant", ["normal", "peaked", "adversarial"])
@pytest.mark.parametrize("split_tiles", [0, 1, 2, 5, 1000])
def test_splits_and_rescaling(variant, split_tiles):
    """Forced splits of 1..5 tiles of 64 tokens (up to 24 partitions merged by sc_combine_kernel), one
    partition (the CTA writes the output itself), and the automatic one-wave choice."""
    c = Case(L=1, Hq=8, Hkv=2, D=128, T_h=1500, n=2, NB=128, seed=5200, variant=variant,
             split_tiles=split_tiles, engine=sc.SC_ENGINE_DECODE)
    a = c.run_layer(0, sc.SC_ATTN_FUSED)
    assert_close(a, c.oracle_layer(0), f"decode {variant} split={split_tiles}")
    assert np.array_equal(a, c.run_layer(0, sc.SC_ATTN_FUSED))          # deterministic
    c.close()


def test_auto_picks_the_decode_engine_for_long_small_calls_only():
    """AUTO: at most 16 (token, group head) rows per KV head AND at least 128 MiB of K/V to read per layer
    (the measured cross-over: below it the tcgen05 kernel's single launch per layer wins) -> decode engine;
    otherwise the tcgen05 engine.  Told apart by bit-equality with the forced engines.  Forcing the decode
    engine on a call with more rows is refused before anything is launched."""
    kw = dict(L=1, Hq=8, Hkv=8, D=128, NB=2100, seed=5300)
    long_h = 32768                                          # x 8 KV heads x 128 x 4 bytes = 128 MiB
    got = {}
    for name, eng, T_h, n in (("auto_long", sc.SC_ENGINE_AUTO, long_h, 1), ("dec_long", sc.SC_ENGINE_DECODE, long_h, 1),
                              ("auto_short", sc.SC_ENGINE_AUTO, 700, 1), ("tc_short", sc.SC_ENGINE_TCGEN05, 700, 1),
                              ("dec_short", sc.SC_ENGINE_DECODE, 700, 1),
                              ("auto_rows", sc.SC_ENGINE_AUTO, long_h, 17), ("tc_rows", sc.SC_ENGINE_TCGEN05, long_h, 17)):
        c = Case(T_h=T_h, n=n, engine=eng, **kw)
        got[name] = c.run_layer(0, sc.SC_ATTN_FUSED)
        if name in ("dec_long", "dec_short", "tc_rows"):
            assert_close(got[name], c.oracle_layer(0), name)
        c.close()
    assert np.array_equal(got["auto_long"], got["dec_long"])
    assert np.array_equal(got["auto_short"], got["tc_short"]) and not np.array_equal(got["auto_short"], got["dec_short"])
    assert np.array_equal(got["auto_rows"], got["tc_rows"])
    bad = Case(T_h=700, n=17, engine=sc.SC_ENGINE_DECODE, **kw)
    before = bad.sess.pool.launch_count()
    with pytest.raises(sc.SwiftCacheError) as e:
        bad.run_layer(0, sc.SC_ATTN_FUSED)
    assert e.value.status == sc.SC_ERR_UNSUPPORTED and bad.sess.pool.launch_count() == before
    bad.close()


@pytest.mark.parametrize("T_h,n,split_tiles", [(333, 1, 0), (1000, 3, 2), (5, 2, 0)])
def test_decode_over_memory_that_was_never_cleared(T_h, n, split_tiles):
    """Pool and LSC full of NaN bit patterns: the scatter pads the last block, tiles past the end re-read
    the last block masked, so the output is finite and right in both modes; written tokens bit-exact."""
    for mode in MODES:
        c = Case(L=1, Hq=4, Hkv=2, D=128, T_h=T_h, n=n, NB=100, seed=5400 + T_h, engine=sc.SC_ENGINE_DECODE,
                 split_tiles=split_tiles, zero_fill=False, fill_byte=0xFF)
        got = c.run_layer(0, mode)
        assert not np.isnan(I.bf16_bits_to_f32(got)).any()
        assert_close(got, c.oracle_layer(0), f"decode over NaN memory T_h={T_h} n={n} mode={mode}")
        k, v = c.sess.read_tokens(0, 0, c.table_dev, 0, T_h + n)
        assert np.array_equal(torch_to_bits(k), np.concatenate([c.data[0][1], c.data[0][3]]))
        assert np.array_equal(torch_to_bits(v), np.concatenate([c.data[0][2], c.data[0][4]]))
        c.close()


@pytest.mark.parametrize("mode", MODES)
def test_ragged_decode_batch_three_steps(mode):
    """Continuous batching: four conversations of very different lengths each append one
    or two tokens per step, three steps in a row through sc_prefill_turn with the decode engine; every
    step against the oracle, the pool against the logical KV at the end."""
    from test_gpu_pipeline import Conversations
    cv = Conversations(L=3, Hq=4, Hkv=4, D=128, hist=[2000, 17, 640, 0], NB=260, max_new=8, seed=57)
    cv.sess.pool.set_engine(sc.SC_ENGINE_DECODE, sc.SC_COPY_AUTO)
    dev = cv.sess.device
    for step in range(3):
        n_new = [1, 2, 1, 1] if step != 1 else [2, 1, 1, 3]
        cv.begin_turn(n_new)
        q_all, k_all, v_all = cv.make_inputs(n_new, 1300 + step)
        ref = cv.oracle_turn(q_all, k_all, v_all)
        tq, tk, tv = (bits_to_torch(x, dev) for x in (q_all, k_all, v_all))
        out = torch.zeros_like(tq)
        cv.sess.pool.prefill_turn(tq.data_ptr(), tk.data_ptr(), tv.data_ptr(), out.data_ptr(), sc.SC_MEM_DEVICE,
                                  cv.tables_dev.data_ptr(), cv.max_blocks, cv.hist, cv.cu, mode,
                                  cv.sess.copy_stream.cuda_stream, cv.sess.compute_stream.cuda_stream)
        torch.cuda.synchronize()
        for l in range(cv.L):
            assert_close(torch_to_bits(out[l]), ref[l], f"ragged decode step {step} layer {l} mode {mode}")
        cv.end_turn(n_new)
    cv.check_pool_equals_logical()
    cv.sess.close()
