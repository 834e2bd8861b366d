"""Host integer logic of SURVEY.md 8(f) rows f3 / f1 behind the C ABI, against the oracle:
LSC / RC sizing (Eq. 1-5), minimum elastic units (Eq. 6-9), Algorithm 1, and the block-major
resize that moves no block.  No GPU needed: pools are created host-only."""
import numpy as np
import pytest

from oracle import sc_oracle as O
from paper_2606_16135_b200 import binding as sc

SHAPES = {"lwm": (32, 32, 128), "qwen3_8b": (36, 8, 128), "qwen3_14b": (40, 8, 128), "qwen3_32b": (64, 8, 128)}


def cfg(L, Hkv, D, B=16, n_blocks=8):
    return sc.make_config(L, max(Hkv, 1), Hkv, D, B, n_blocks, 0, 16)


def test_sizing_worked_example_through_the_abi():
    """PAPER.md:180 with a real M_block: L=10 -> the call only reads L, Hkv, D, B of the config."""
    c = sc.make_config(10, 4, 4, 64, 16, 8, 0, 16)
    m_block = O.block_bytes(16, 4, 64)
    got = sc.sc_lsc_rc_sizing(c, 100 * m_block, [9 * m_block * 10, 8 * m_block * 10 + 123])
    assert (got["n_lsc"], got["n_rc"], got["max_context_blocks"], got["conventional_blocks"]) == (17, 8, 25, 10)


def test_sizing_matches_oracle_on_random_memory_sizes():
    rng = np.random.default_rng(3)
    for name, (L, Hkv, D) in SHAPES.items():
        c = cfg(L, Hkv, D)
        m_block = O.block_bytes(16, Hkv, D)
        for _ in range(50):
            c_master = int(rng.integers(0, 96 << 30))
            workers = [int(x) for x in rng.integers(0, 96 << 30, size=int(rng.integers(0, 4)))]
            assert sc.sc_lsc_rc_sizing(c, c_master, workers) == O.lsc_rc_sizing(c_master, workers, m_block, L), name


def test_elastic_units_match_oracle():
    for m_name, (Lm, Hm, Dm) in SHAPES.items():
        for w_name, (Lw, Hw, Dw) in SHAPES.items():
            for Bw in (16, 32):
                want = O.meu(O.block_elems(Lm, 16, Hm, Dm), O.block_elems(Lw, Bw, Hw, Dw))
                assert sc.sc_elastic_units(cfg(Lm, Hm, Dm), cfg(Lw, Hw, Dw, B=16) if Bw == 16 else
                                           sc.sc_pool_config_t(Lw, Hw, Hw, Dw, Bw, 8, 0, 0, 16, 1, 0)) == want, (m_name, w_name)
    assert sc.sc_elastic_units(cfg(32, 32, 128), cfg(40, 8, 128)) == (5, 16)


def test_algorithm1_matches_oracle():
    rng = np.random.default_rng(5)
    for _ in range(500):
        n_i, b_i = int(rng.integers(0, 5000)), int(rng.choice([8, 16, 32]))
        mi, mm = int(rng.integers(1, 40)), int(rng.integers(1, 40))
        length = int(rng.integers(0, 200000))
        assert sc.sc_scale_up(n_i, b_i, mi, mm, length) == O.scale_up(n_i, b_i, mi, mm, length)
        assert sc.sc_scale_down(n_i, b_i, mi, mm, length) == O.scale_down(n_i, b_i, mi, mm, length)
    with pytest.raises(sc.SwiftCacheError):
        sc.sc_scale_up(1, 0, 1, 1, 1)


def test_block_major_resize_moves_nothing():
    """Growing and shrinking change only the free list: surviving blocks keep their offsets."""
    c = sc.make_config(4, 4, 2, 64, 16, 6, 0, 16)
    p = sc.Pool(c)                                            # host-only
    probe = [(b, l, kv, h, s, d) for b in (0, 3, 5) for l in (0, 3) for kv in (0, 1) for h in (0, 1) for s in (0, 15) for d in (0, 63)]
    before = [p.cell_offset(*x) for x in probe]
    held = p.alloc_blocks(4)                                  # ids 0..3
    p.resize(10)
    assert p.num_free_blocks() == 6 and p.info().pool_bytes == 10 * p.info().block_bytes
    assert [p.cell_offset(*x) for x in probe] == before
    # the old free ids go first, the appended ids last and in ascending order
    assert p.alloc_blocks(6).tolist() == [4, 5, 6, 7, 8, 9]
    assert p.cell_offset(9, 3, 1, 1, 15, 63) == 9 * p.info().block_bytes + before[-1] - 5 * p.info().block_bytes
    # shrinking below a block that is in use is refused and changes nothing
    with pytest.raises(sc.SwiftCacheError) as e:
        p.resize(8)
    assert e.value.status == sc.SC_ERR_BAD_BLOCK_ID and p.info().pool_bytes == 10 * p.info().block_bytes
    p.free_blocks([8, 9, 7])
    p.resize(7)
    assert p.num_free_blocks() == 0 and p.info().pool_bytes == 7 * p.info().block_bytes
    with pytest.raises(sc.SwiftCacheError):
        p.cell_offset(7, 0, 0, 0, 0, 0)                       # gone
    assert [p.cell_offset(*x) for x in probe] == before
    p.free_blocks(held)
    assert sorted(p.alloc_blocks(4).tolist()) == [0, 1, 2, 3]
    p.destroy()


def test_scale_decisions_drive_a_resize_in_whole_units():
    """Worker side of Sec. 3.5: ScaleUp says how many blocks to append, ScaleDown how many of the
    tail to release; both in multiples of the elastic unit."""
    master, worker = cfg(32, 32, 128), cfg(40, 8, 128, n_blocks=32)
    mm, mw = sc.sc_elastic_units(master, worker)
    p = sc.Pool(worker)
    dw, dm = sc.sc_scale_up(32, 16, mw, mm, 1000)             # needs 63 blocks
    assert (dw, dm) == (32, 10)                               # 31 missing -> 2 units of 16
    p.resize(32 + dw)
    assert p.num_free_blocks() == 64
    bw, bm = sc.sc_scale_down(64, 16, mw, mm, 300)            # 19 blocks needed lately
    assert (bw, bm) == (32, 10)                               # 45 spare -> 2 units
    p.resize(64 - bw)
    assert p.num_free_blocks() == 32
    p.destroy()


def test_layer_major_would_move_what_block_major_does_not():
    """PAPER.md:208-216 (Fig. 6): in a layer-major pool [L][n_blocks] the slab of layer l starts at
    l * n_blocks * cell; growing n_blocks -> n_blocks' shifts the slab of every layer l >= 1, i.e.
    (L - 1) * n_blocks cells must be copied -- O(n_layers * n_blocks).  The block-major pool of this
    library moves nothing: the offset of every surviving (block, layer) cell is unchanged."""
    L, nb, nb2 = 32, 384, 400
    c = sc.make_config(L, 32, 32, 128, 16, nb, 0, 16)
    p = sc.Pool(c)                                            # host-only
    cell = p.info().cell_bytes
    probe = [(b, l) for b in (0, 1, nb // 2, nb - 1) for l in (0, 1, L // 2, L - 1)]
    before = [p.cell_offset(b, l, 0, 0, 0, 0) for b, l in probe]
    p.resize(nb2)
    assert [p.cell_offset(b, l, 0, 0, 0, 0) for b, l in probe] == before         # block-major: 0 bytes moved
    layer_major = lambda n, b, l: (l * n + b) * cell                              # noqa: E731
    moved = sum(cell for l in range(L) for b in range(nb) if layer_major(nb, b, l) != layer_major(nb2, b, l))
    assert moved == (L - 1) * nb * cell == 31 * 384 * 256 * 1024                  # 2.9 GiB for 16 more blocks
    p.destroy()
