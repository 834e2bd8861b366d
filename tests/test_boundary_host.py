"""Host-side logic of the C ABI (no GPU needed): the library loads and exports every
symbol the header declares; pool geometry (Eq. 1, block-major); the logical accessor;
the block allocator and sc_append_blocks (checked against the oracle's counts)."""
import os
import re

import numpy as np
import pytest

from oracle import sc_oracle as O
from paper_2606_16135_b200 import binding as sc
from paper_2606_16135_b200 import build as sc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="session", autouse=True)
def _built():
    sc_build.build()


def host_pool(L=2, Hq=4, Hkv=4, D=64, B=16, NB=64, lsc=0, seed=0, max_new=256, max_seqs=8):
    return sc.Pool(sc.make_config(L, Hq, Hkv, D, B, NB, lsc, max_new, max_seqs, alloc_seed=seed))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "swiftcache.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(sc_[a-z0-9_]+)\s*\(", header))
    assert declared == set(sc.SYMBOLS), declared ^ set(sc.SYMBOLS)
    lib = sc.lib()
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in sc.sc_version()


def test_bytes_required_is_eq1_block_major():
    for (L, Hkv, D, NB, lsc) in [(32, 32, 128, 364, 340), (32, 8, 128, 8256, 8210), (2, 4, 64, 64, 40)]:
        cfg = sc.make_config(L, 32 if Hkv != 4 else 4, Hkv, D, 16, NB, lsc, 256)
        pool_b, lsc_b = sc.sc_pool_bytes_required(cfg)
        m_block = O.block_bytes(16, Hkv, D, 2)                  # Eq. 1
        assert pool_b == NB * L * m_block
        assert lsc_b == 2 * lsc * m_block
        assert pool_b == NB * 16 * O.kv_bytes_per_token(L, Hkv, D, 2)   # Table 2 x tokens


@pytest.mark.parametrize("cfg_kw,status", [
    (dict(D=96), sc.SC_ERR_UNSUPPORTED), (dict(B=32), sc.SC_ERR_UNSUPPORTED),
    (dict(Hq=6, Hkv=4), sc.SC_ERR_UNSUPPORTED), (dict(NB=0), sc.SC_ERR_INVALID_ARG),
    (dict(max_seqs=64), sc.SC_ERR_UNSUPPORTED),
])
def test_unsupported_configs_fail_loudly(cfg_kw, status):
    with pytest.raises(sc.SwiftCacheError) as e:
        host_pool(**cfg_kw)
    assert e.value.status == status and len(str(e.value)) > 10


def test_cell_offset_is_a_bijection_with_documented_formula():
    L, Hkv, D, NB = 2, 4, 64, 8
    p = host_pool(L=L, Hkv=Hkv, D=D, NB=NB)
    info = p.info()
    assert info.chunk_bytes == 16 * D * 2 and info.cell_bytes == 2 * Hkv * info.chunk_bytes
    assert info.block_bytes == L * info.cell_bytes
    seen = set()
    for kv in range(2):
        for h in range(Hkv):
            for s in range(16):
                for d in range(D):
                    off = p.cell_offset(3, 1, kv, h, s, d)
                    inner = ((s // 8) * (D // 64) * 1024 + (d // 64) * 1024 + (s % 8) * 128
                             + ((((d % 64) // 8) ^ (s % 8)) * 16) + (d % 8) * 2)
                    assert off == 3 * info.block_bytes + 1 * info.cell_bytes + (kv * Hkv + h) * info.chunk_bytes + inner
                    seen.add(off)
    base = 3 * info.block_bytes + info.cell_bytes
    assert len(seen) == 2 * Hkv * 16 * D and min(seen) == base and max(seen) == base + info.cell_bytes - 2
    # block-major: the next block is one full-layer block further
    assert p.cell_offset(4, 1, 0, 0, 0, 0) - p.cell_offset(3, 1, 0, 0, 0, 0) == info.block_bytes
    assert p.cell_offset(3, 1, 0, 0, 0, 0) - p.cell_offset(3, 0, 0, 0, 0, 0) == info.cell_bytes
    with pytest.raises(sc.SwiftCacheError):
        p.cell_offset(NB, 0, 0, 0, 0, 0)


def test_cell_offset_d128_16_byte_units_stay_whole():
    p = host_pool(L=1, Hq=8, Hkv=2, D=128, NB=2)
    for s in range(16):
        for d0 in range(0, 128, 8):
            offs = [p.cell_offset(1, 0, 1, 1, s, d0 + i) for i in range(8)]
            assert offs[0] % 16 == 0 and offs == list(range(offs[0], offs[0] + 16, 2))


def test_allocator_properties():
    NB = 50
    p = host_pool(NB=NB)
    assert p.num_free_blocks() == NB
    a = p.alloc_blocks(20)
    b = p.alloc_blocks(30)
    ids = np.concatenate([a, b])
    assert sorted(ids.tolist()) == list(range(NB)) and p.num_free_blocks() == 0
    assert a.tolist() == list(range(20))                         # seed 0: ascending
    with pytest.raises(sc.SwiftCacheError) as e:
        p.alloc_blocks(1)
    assert e.value.status == sc.SC_ERR_OUT_OF_BLOCKS
    p.free_blocks(a[:5])
    assert p.num_free_blocks() == 5
    for bad in ([a[0]], [NB], [-1], [int(a[7]), int(a[7])]):     # already free, range, repeated
        with pytest.raises(sc.SwiftCacheError) as e:
            p.free_blocks(bad)
        assert e.value.status == sc.SC_ERR_BAD_BLOCK_ID
    assert p.num_free_blocks() == 5                              # failed frees changed nothing
    p.free_blocks([int(a[7])])
    again = p.alloc_blocks(6)
    assert set(again.tolist()) == set(a[:5].tolist()) | {int(a[7])}
    with pytest.raises(sc.SwiftCacheError) as e:                 # all-or-nothing
        p.alloc_blocks(1)
    assert p.num_free_blocks() == 0


def test_allocator_seeded_shuffle_is_reproducible_permutation():
    a = host_pool(NB=200, seed=7).alloc_blocks(200)
    b = host_pool(NB=200, seed=7).alloc_blocks(200)
    c = host_pool(NB=200, seed=8).alloc_blocks(200)
    assert a.tolist() == b.tolist() and a.tolist() != c.tolist()
    assert sorted(a.tolist()) == list(range(200)) and a.tolist() != list(range(200))


@pytest.mark.parametrize("h,n", [(0, 1), (0, 16), (0, 17), (512, 32), (5120, 256), (4321, 256),
                                 (15, 1), (16, 1), (17, 15), (17, 16), (509, 33), (1, 256)])
def test_append_blocks_matches_oracle_count(h, n):
    p = host_pool(NB=400, seed=3)
    table = np.full(400, -1, dtype=np.int32)
    nt = p.append_blocks(table, 0, 0, h)                         # history blocks
    assert nt == O.blocks_for(h, 16)
    before = table[:nt].copy()
    nt2 = p.append_blocks(table, nt, h, n)
    assert nt2 - nt == O.append_count(h, n, 16) and nt2 == O.blocks_for(h + n, 16)
    assert np.array_equal(table[:nt], before)                    # existing entries untouched
    ids = table[:nt2]
    assert len(set(ids.tolist())) == nt2 and ids.min() >= 0 and ids.max() < 400
    assert (table[nt2:] == -1).all()
    assert p.num_free_blocks() == 400 - nt2
    assert p.append_blocks(table, nt2, h, n) == nt2              # idempotent once covered


def test_append_blocks_errors_change_nothing():
    p = host_pool(NB=10)
    table = np.full(4, -1, dtype=np.int32)
    with pytest.raises(sc.SwiftCacheError) as e:                 # cap too small
        p.append_blocks(table, 0, 0, 16 * 5)
    assert e.value.status == sc.SC_ERR_CAPACITY and p.num_free_blocks() == 10 and (table == -1).all()
    big = np.full(32, -1, dtype=np.int32)
    with pytest.raises(sc.SwiftCacheError) as e:                 # pool too small
        p.append_blocks(big, 0, 0, 16 * 11)
    assert e.value.status == sc.SC_ERR_OUT_OF_BLOCKS and p.num_free_blocks() == 10
    with pytest.raises(sc.SwiftCacheError) as e:                 # table does not cover the history
        p.append_blocks(big, 1, 40, 8)
    assert e.value.status == sc.SC_ERR_INVALID_ARG


def test_two_conversations_get_disjoint_tables():
    p = host_pool(NB=64, seed=11)
    t1, t2 = np.full(32, -1, np.int32), np.full(32, -1, np.int32)
    n1 = p.append_blocks(t1, 0, 0, 100)
    n2 = p.append_blocks(t2, 0, 0, 37)
    for turn in range(3):
        n1 = p.append_blocks(t1, n1, 100 + 20 * turn, 20)
        n2 = p.append_blocks(t2, n2, 37 + 20 * turn, 20)
    assert not set(t1[:n1].tolist()) & set(t2[:n2].tolist())
    assert n1 == O.blocks_for(160, 16) and n2 == O.blocks_for(97, 16)


def test_data_calls_fail_loudly_without_device_memory():
    """No CPU fallback: a pool created without memory refuses every data call."""
    p = host_pool()
    for call in (lambda: p.store_prefix(0, 1, 1, 0, 16, 1, 1),
                 lambda: p.load_layer(0, 1, 1, 16, 0),
                 lambda: p.prefill_layer(0, 1, 1, 1, 1, 4, 16, 16, 0, sc.SC_ATTN_FUSED, 1),
                 lambda: p.prefill_turn(1, 1, 1, 1, sc.SC_MEM_DEVICE, 1, 4, [16], [0, 16], sc.SC_ATTN_FUSED, 0, 0)):
        with pytest.raises(sc.SwiftCacheError) as e:
            call()
        assert e.value.status == sc.SC_ERR_CUDA


def test_product_package_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_16135_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                for pat in (r"(import|from)\s+oracle", r"sc_oracle", r"oracle[/.]", r"sco_"):
                    assert not re.search(pat, src), (pat, os.path.join(dirpath, f))
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_16135_b200" not in src and "from paper_2606_16135_b200" not in src
            assert "swiftcache.h" not in src and "sc_internal" not in src
