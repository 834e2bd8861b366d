"""GPU parity of BOTH attention engines (mma.sync and tcgen05/TMEM) against the CPU oracle,
through the C ABI, on shapes chosen to stress the tcgen05 engine's tiling: one and two
128-row query tiles, KV tiles of 128 tokens with ragged tails, splits whose last tiles are
masked for the first query tile, GQA, D 64 and 128."""
import numpy as np
import pytest

from paper_2606_16135_b200 import binding as sc
from paper_2606_16135_b200 import build as sc_build

from gpu_util import Case, assert_close

pytestmark = pytest.mark.gpu

ENGINES = [sc.SC_ENGINE_MMA_SYNC, sc.SC_ENGINE_TCGEN05]
MODES = [sc.SC_ATTN_STAGED, sc.SC_ATTN_FUSED]


@pytest.fixture(scope="session", autouse=True)
def _built():
    sc_build.build()


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("D", [64, 128])
@pytest.mark.parametrize("T_h,n", [(0, 128), (0, 256), (300, 256), (1, 129), (127, 1), (128, 128),
                                   (1000, 255), (2049, 257), (640, 300)])
def test_query_tile_pairs_and_kv_tiles(engine, D, T_h, n):
    c = Case(L=1, Hq=2, Hkv=2, D=D, T_h=T_h, n=n, NB=160, seed=4000 + T_h + n, engine=engine)
    mode = MODES[(T_h + n + D) % 2]
    assert_close(c.run_layer(0, mode), c.oracle_layer(0), f"engine={engine} D={D} T_h={T_h} n={n}")
    c.close()


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("variant", ["normal", "peaked", "adversarial"])
@pytest.mark.parametrize("split_tiles", [0, 1, 2, 3, 7])
def test_splits_with_rescaling(engine, variant, split_tiles):
    """Peaked / adversarial scores force the (lazy) rescale of the accumulated O; splits of
    1..7 KV tiles put the causal boundary in every position relative to a split."""
    c = Case(L=1, Hq=4, Hkv=1, D=128, T_h=1500, n=256, NB=128, seed=31, variant=variant,
             split_tiles=split_tiles, engine=engine)
    assert_close(c.run_layer(0, sc.SC_ATTN_FUSED), c.oracle_layer(0), f"{variant} split={split_tiles}")
    c.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_engines_are_deterministic(engine):
    c = Case(L=1, Hq=4, Hkv=2, D=128, T_h=900, n=200, NB=80, seed=8, variant="peaked", engine=engine)
    a = c.run_layer(0, sc.SC_ATTN_FUSED)
    b = c.run_layer(0, sc.SC_ATTN_FUSED)     # the scatter rewrites the same bytes; same result
    assert np.array_equal(a, b)
    c.close()


def test_lwm_layer_shape_tcgen05():
    """One layer of BASELINE.json config 2 (32 heads, D 128, 5120 history, 256 new), default
    split heuristic, in the launch configuration bench.py times; sampled heads vs the oracle."""
    c = Case(L=1, Hq=32, Hkv=32, D=128, T_h=5120, n=256, NB=400, seed=2, engine=sc.SC_ENGINE_TCGEN05)
    got = c.run_layer(0, sc.SC_ATTN_FUSED)
    ref = c.oracle_layer(0)
    assert_close(got, ref, "lwm layer")
    for h in (0, 13, 31):
        assert_close(got[:, h], ref[:, h], f"head {h}")
    c.close()


@pytest.mark.parametrize("Hq,Hkv,n,folded", [(4, 4, 200, True), (4, 4, 300, False), (8, 2, 200, False)])
def test_scatter_is_folded_only_with_one_writer_per_row(Hq, Hkv, n, folded):
    """The tcgen05 kernel stores the turn's new K/V itself only where that leaves ONE writer per row: no
    grouped-query heads (each query head of a group would store the KV head's rows) and one query pair
    per sequence (a later pair would store the earlier pair's rows).  Otherwise the scatter kernel runs
    first -- one more launch.  Either way the pool holds the new tokens bit for bit afterwards."""
    T_h = 700
    c = Case(L=1, Hq=Hq, Hkv=Hkv, D=128, T_h=T_h, n=n, NB=80, seed=6100 + n + Hq, engine=sc.SC_ENGINE_TCGEN05)
    before = c.sess.pool.launch_count()
    got = c.run_layer(0, sc.SC_ATTN_FUSED)
    launches = c.sess.pool.launch_count() - before
    assert_close(got, c.oracle_layer(0), f"Hq={Hq} Hkv={Hkv} n={n}")
    k, v = c.sess.read_tokens(0, 0, c.table_dev, 0, T_h + n)
    from paper_2606_16135_b200.runtime import torch_to_bits
    assert np.array_equal(torch_to_bits(k), np.concatenate([c.data[0][1], c.data[0][3]]))
    assert np.array_equal(torch_to_bits(v), np.concatenate([c.data[0][2], c.data[0][4]]))
    # attention alone when folded; scatter + attention (+ combine when the KV range was split) otherwise
    assert (launches == 1) if folded else (launches >= 2), launches
    c.close()
