"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-type the oracle's formula and compare it with itself: each
checks the oracle against an independent source -- values the paper prints
(tests/golden/), bit equality with the logically contiguous tensor (I1, I2),
the monolithic-causal definition (I3), closed forms (I4), an invariance (I5),
a pure-Python float64 triple loop and torch's SDPA (I6).
SURVEY.md section 8(c); DESIGN.md section 3.
"""
import math
import os

import numpy as np
import pytest

from oracle import sc_oracle as O
from paper_2606_16135_b200 import inputs as I

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                out.append(line.split())
    return out


# --------------------------------------------------------------- paper values
def test_table2_kv_bytes_per_token():
    """L*2*Hkv*D*2 bytes reproduces every printed MiB figure."""
    for L, H, D, printed in _rows("table2_kv_bytes_per_token.txt"):
        mib = O.kv_bytes_per_token(int(L), int(H), int(D), 2) / 2**20
        digits = len(printed.split(".")[1])
        assert abs(mib - float(printed)) <= 0.5 * 10 ** (-digits) + 1e-12, (L, H, D, mib, printed)


def test_block_bytes_eq1():
    """Eq. 1: LWM block of 16 tokens = 256 KiB per layer; GQA 64 KiB."""
    assert O.block_bytes(16, 32, 128, 2) == 256 * 1024
    assert O.block_bytes(16, 8, 128, 2) == 64 * 1024
    # Eq. 1 x L x (tokens/B) must agree with Table 2 x tokens
    assert O.block_bytes(16, 32, 128, 2) * 32 == O.kv_bytes_per_token(32, 32, 128, 2) * 16


def test_fig1_self_consistency():
    """75/(75+27) ~ 73.2 %; 5k tokens * 0.5 MiB / 32 GB/s ~ 75 ms."""
    (load, comp, share, gbs, hist), = _rows("fig1_consistency.txt")
    load, comp, share, gbs, hist = map(float, (load, comp, share, gbs, hist))
    assert abs(100 * load / (load + comp) - share) < 1.0
    ms = hist * O.kv_bytes_per_token(32, 32, 128, 2) / (gbs * 1e9) * 1e3
    assert 0.8 * load < ms < 1.25 * load


@pytest.mark.parametrize("h,n,B,want", [
    (0, 1, 16, 1), (0, 16, 16, 1), (0, 17, 16, 2), (512, 32, 16, 2), (5120, 256, 16, 16),
    (50000, 256, 16, 16), (4321, 256, 16, 16), (15, 1, 16, 0), (16, 1, 16, 1), (17, 15, 16, 0),
    (17, 16, 16, 1), (27359, 256, 16, 16), (1, 256, 16, 16), (509, 33, 16, 2),
])
def test_append_count(h, n, B, want):
    """O5: hand-counted cases of ceil((T_h+n)/B) - ceil(T_h/B)."""
    assert O.append_count(h, n, B) == want
    # brute force: count blocks newly touched by tokens h..h+n-1 that no token < h touches
    touched_before = {t // B for t in range(h)}
    new = {t // B for t in range(h, h + n)} - touched_before
    assert len(new) == want


# ------------------------------------------------------------------- helpers
def _tiny_case(seed=7, T_h=512, n=32, Hq=4, Hkv=4, D=64, variant="normal"):
    return I.make_qkv(n, T_h, Hq, Hkv, D, seed, variant)


def _brute_force_f64(q, K, V, T_h):
    """Independent pure-Python float64 triple loop (no numpy arithmetic)."""
    n, Hq, D = q.shape
    Hkv = K.shape[1]
    G = Hq // Hkv
    qf = I.bf16_bits_to_f32(q).astype(np.float64).tolist()
    Kf = I.bf16_bits_to_f32(K).astype(np.float64).tolist()
    Vf = I.bf16_bits_to_f32(V).astype(np.float64).tolist()
    out = np.zeros((n, Hq, D))
    for i in range(n):
        for h in range(Hq):
            g = h // G
            s = []
            for j in range(T_h + i + 1):
                acc = 0.0
                qi, kj = qf[i][h], Kf[j][g]
                for d in range(D):
                    acc += qi[d] * kj[d]
                s.append(acc / math.sqrt(D))
            m = max(s)
            e = [math.exp(x - m) for x in s]
            z = sum(e)
            for d in range(D):
                acc = 0.0
                for j in range(T_h + i + 1):
                    acc += e[j] / z * Vf[j][g][d]
                out[i, h, d] = acc
    return out


# ------------------------------------------------------------ I1 / I2 / I5
def test_I1_gather_bit_equal_contiguous():
    """I1: gathering through a permuted table returns the contiguous history bit for bit."""
    L, Hkv, D, B, NB, T = 2, 4, 64, 16, 64, 509          # ragged: 509 = 31*16 + 13
    table = I.block_table(1, NB, O.blocks_for(T, B))
    pool = O.Pool(L, Hkv, D, B, NB)
    X = {(l, kv): I.normal_bf16((T, Hkv, D), 100 + 2 * l + kv) for l in range(L) for kv in (0, 1)}
    for (l, kv), x in X.items():
        pool.store(l, kv, x, 0, table)
    for (l, kv), x in X.items():
        assert np.array_equal(pool.gather(l, kv, table, T), x)
    # a different conversation's blocks stay zero (zero-initialised pool, disjoint tables)
    other = np.setdiff1d(np.arange(NB, dtype=np.int32), table)[:4]
    assert not pool.gather(0, 0, other, 4 * B).any()


def test_I1_store_in_pieces_and_errors():
    """Storing in ragged pieces (mid-block starts) equals storing at once."""
    L, Hkv, D, B, NB, T = 1, 2, 16, 16, 16, 100
    table = I.block_table(1, NB, O.blocks_for(T, B))
    x = I.normal_bf16((T, Hkv, D), 5)
    pool = O.Pool(L, Hkv, D, B, NB)
    for a, b in [(0, 1), (1, 15), (15, 17), (17, 64), (64, 100)]:
        pool.store(0, 0, x[a:b], a, table)
    assert np.array_equal(pool.gather(0, 0, table, T), x)
    with pytest.raises(IndexError):
        pool.store(0, 0, x, 0, table[:3])
    with pytest.raises(IndexError):
        pool.gather(0, 0, np.array([NB], dtype=np.int32), 1)


def test_I2_scatter_then_gather_is_concat():
    """I2: after a turn, gathering T_h+n tokens returns [history ; k_new] bit-exactly."""
    L, Hq, Hkv, D, B, NB, T_h, n = 2, 4, 2, 32, 16, 48, 77, 33
    table = list(I.block_table(1, NB, O.blocks_for(T_h, B)))
    pool = O.Pool(L, Hkv, D, B, NB)
    hist = {}
    for l in range(L):
        q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 40 + l)
        pool.store(l, 0, kh, 0, table)
        pool.store(l, 1, vh, 0, table)
        hist[l] = (q, kh, vh, kn, vn)
    free = [b for b in I.permuted_ids(1, NB) if b not in set(table)]
    table += free[:O.append_count(T_h, n, B)]
    assert len(table) == O.blocks_for(T_h + n, B) and len(set(table)) == len(table)
    for l in range(L):
        q, kh, vh, kn, vn = hist[l]
        O.prefill_layer(pool, l, q, kn, vn, table, T_h)
        assert np.array_equal(pool.gather(l, 0, table, T_h + n), np.concatenate([kh, kn]))
        assert np.array_equal(pool.gather(l, 1, table, T_h + n), np.concatenate([vh, vn]))


def test_I5_permutation_invariance():
    """I5: re-placing the same logical data under a different table changes no output bit."""
    L, Hq, Hkv, D, B, NB, T_h, n = 1, 4, 2, 32, 16, 40, 200, 17
    q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 11)
    outs = []
    for cfg_seed, ident in ((1, False), (2, False), (1, True)):
        table = I.block_table(cfg_seed, NB, O.blocks_for(T_h + n, B), identity=ident)
        pool = O.Pool(L, Hkv, D, B, NB)
        pool.store(0, 0, kh, 0, table)
        pool.store(0, 1, vh, 0, table)
        outs.append(O.prefill_layer(pool, 0, q, kn, vn, table, T_h))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


# ------------------------------------------------------------------------ I3
def test_I3_last_rows_of_monolithic_causal():
    """I3: chunked-with-history output == last n rows of ONE causal attention over the
    concatenated T_h+n sequence (queries for the history rows are generated too)."""
    T_h, n, Hq, Hkv, D = 96, 32, 4, 2, 32
    q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 21)
    q_hist = I.normal_bf16((T_h, Hq, D), 22)
    K, V = np.concatenate([kh, kn]), np.concatenate([vh, vn])
    chunked = O.attention(q, K, V, T_h)
    mono = O.attention(np.concatenate([q_hist, q]), K, V, 0)   # T_h = 0: textbook causal
    assert np.array_equal(mono[T_h:], chunked)
    # and the textbook causal definition itself, via torch on CPU with an explicit mask
    import torch
    qa = torch.from_numpy(I.bf16_bits_to_f32(np.concatenate([q_hist, q]))).permute(1, 0, 2)
    Ka = torch.from_numpy(I.bf16_bits_to_f32(K)).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)
    Va = torch.from_numpy(I.bf16_bits_to_f32(V)).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)
    T = T_h + n
    mask = torch.tril(torch.ones(T, T, dtype=torch.bool))
    ref = torch.nn.functional.scaled_dot_product_attention(
        qa.double(), Ka.double(), Va.double(), attn_mask=mask).permute(1, 0, 2).numpy()
    assert np.abs(mono - ref).max() < 2e-6


def test_I3_n1_is_decode_over_all_keys():
    """n = 1: plain decode attention over all T_h+1 keys (no mask at all)."""
    T_h, Hq, Hkv, D = 70, 4, 4, 16
    q, kh, vh, kn, vn = I.make_qkv(1, T_h, Hq, Hkv, D, 31)
    K, V = np.concatenate([kh, kn]), np.concatenate([vh, vn])
    out = O.attention(q, K, V, T_h, dtype=np.float64)
    qf, Kf, Vf = (I.bf16_bits_to_f32(x).astype(np.float64) for x in (q, K, V))
    s = np.einsum("hd,jhd->hj", qf[0], Kf) / math.sqrt(D)
    p = np.exp(s - s.max(-1, keepdims=True))
    p /= p.sum(-1, keepdims=True)
    assert np.abs(out[0] - np.einsum("hj,jhd->hd", p, Vf)).max() < 1e-12


# ------------------------------------------------------------------------ I4
def test_I4_softmax_rows_sum_to_one_and_V_ones():
    T_h, n, Hq, Hkv, D = 300, 20, 4, 2, 64
    for variant in ("normal", "peaked", "adversarial"):
        q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 51, variant)
        K = np.concatenate([kh, kn])
        ones = np.full_like(K, 0x3F80)                     # bf16 1.0
        out, rs = O.attention(q, K, ones, T_h, return_rowsum=True)
        assert np.abs(rs - 1).max() <= 1e-5
        assert np.abs(out - 1).max() <= 2e-6
        p = O.softmax_row(q, K, T_h, n - 1, Hq - 1)
        assert p.shape == (T_h + n,) and abs(float(p.sum()) - 1) <= 1e-5 and (p >= 0).all()


def test_I4_softmax_row_against_a_python_loop():
    """sco_softmax_row_f32 against an independent pure-Python fp64 loop, e[j] / z written out:
    a wrong scale, a wrong kv-head mapping g = h // (Hq / Hkv), a missing max subtraction that
    overflows, or a wrong causal length T_h + i + 1 all fail here.  Config 1 (MHA) and a GQA case."""
    for (T_h, n, Hq, Hkv, D, variant) in ((512, 32, 4, 4, 64, "normal"), (70, 9, 8, 2, 32, "peaked")):
        q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 77, variant)
        K = np.concatenate([kh, kn])
        qf = I.bf16_bits_to_f32(q).astype(np.float64)
        Kf = I.bf16_bits_to_f32(K).astype(np.float64)
        G = Hq // Hkv
        for i, h in ((0, 0), (n // 2, Hq - 1), (n - 1, 1), (n - 1, Hq - 1)):
            nk = T_h + i + 1
            s = []
            for j in range(nk):
                acc = 0.0
                for d in range(D):
                    acc += float(qf[i, h, d]) * float(Kf[j, h // G, d])
                s.append(acc / math.sqrt(D))
            mx = max(s)
            e = [math.exp(x - mx) for x in s]
            z = sum(e)
            want = np.array([x / z for x in e])
            p = O.softmax_row(q, K, T_h, i, h)
            assert p.shape == (nk,)
            assert np.abs(p.astype(np.float64) - want).max() <= 1e-6, (T_h, i, h)
    # the unscaled scores of the peaked case reach ~ +-60: without the max subtraction exp() overflows fp32


def test_I4_uniform_closed_form():
    """q == 0 (or K constant) -> p uniform -> out[i] = mean(V[0 : T_h+i+1]) exactly."""
    T_h, n, Hq, Hkv, D = 45, 9, 4, 2, 16
    q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 61)
    K, V = np.concatenate([kh, kn]), np.concatenate([vh, vn])
    Vf = I.bf16_bits_to_f32(V).astype(np.float64)
    G = Hq // Hkv
    for qq, KK in ((np.zeros_like(q), K), (q, np.broadcast_to(K[:1], K.shape).copy())):
        out = O.attention(qq, KK, V, T_h, dtype=np.float64)
        for i in range(n):
            want = Vf[: T_h + i + 1].mean(axis=0)          # [Hkv][D]
            for h in range(Hq):
                assert np.abs(out[i, h] - want[h // G]).max() < 1e-12


def test_I4_one_hot_key_selects_value():
    """A key hugely aligned with the query makes softmax one-hot: out == that V row.
    Catches a transposed operand or wrong head mapping (g = h // G)."""
    T_h, n, Hq, Hkv, D = 40, 4, 4, 2, 16
    q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 71)
    G = Hq // Hkv
    q[:] = 0
    kh[:] = 0
    kn[:] = 0
    # head h looks along axis h; kv-head g's key at history position 3+g holds axes of its group
    for h in range(Hq):
        q[:, h, h] = I.f32_to_bf16_bits(np.float32([64.0]))[0]
        kh[3 + h // G, h // G, h] = I.f32_to_bf16_bits(np.float32([64.0]))[0]
    K, V = np.concatenate([kh, kn]), np.concatenate([vh, vn])
    out = O.attention(q, K, V, T_h)
    Vf = I.bf16_bits_to_f32(V)
    for h in range(Hq):
        assert np.abs(out[:, h] - Vf[3 + h // G, h // G]).max() < 1e-6


def test_causal_mask_excludes_future_new_tokens():
    """Changing k_new/v_new at position > i must not change row i; changing position i must."""
    T_h, n, Hq, Hkv, D = 33, 8, 2, 2, 16
    q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 81)
    base = O.attention(q, np.concatenate([kh, kn]), np.concatenate([vh, vn]), T_h)
    vn2 = vn.copy()
    vn2[5] = I.normal_bf16(vn[5].shape, 999)
    alt = O.attention(q, np.concatenate([kh, kn]), np.concatenate([vh, vn2]), T_h)
    assert np.array_equal(base[:5], alt[:5])
    assert not np.array_equal(base[5], alt[5]) and not np.array_equal(base[7], alt[7])


# ------------------------------------------------------------------------ I6
def test_I6_brute_force_tiny_config():
    """Pure-Python float64 triple loop over BASELINE.json config 1 (tiny, one layer),
    plus the fp32 oracle's own error against its float64 variant."""
    q, kh, vh, kn, vn = _tiny_case()
    K, V = np.concatenate([kh, kn]), np.concatenate([vh, vn])
    bf = _brute_force_f64(q, K, V, 512)
    o64 = O.attention(q, K, V, 512, dtype=np.float64)
    o32 = O.attention(q, K, V, 512, dtype=np.float32)
    assert np.abs(o64 - bf).max() < 1e-13
    rel = np.linalg.norm(o32 - bf) / np.linalg.norm(bf)
    assert rel < 2e-6 and np.abs(o32 - bf).max() < 1e-6


@pytest.mark.parametrize("T_h,n,Hq,Hkv,variant", [
    (0, 33, 4, 4, "normal"), (1, 1, 4, 1, "peaked"), (17, 31, 8, 2, "adversarial"),
    (509, 32, 4, 4, "peaked"),
])
def test_I6_sdpa_cross_check(T_h, n, Hq, Hkv, variant):
    """Library routine: torch SDPA, fp32 CPU, explicit boolean mask j <= T_h + i."""
    import torch
    D = 64
    q, kh, vh, kn, vn = I.make_qkv(n, T_h, Hq, Hkv, D, 91, variant)
    K, V = np.concatenate([kh, kn]), np.concatenate([vh, vn])
    out = O.attention(q, K, V, T_h)
    G = Hq // Hkv
    qa = torch.from_numpy(I.bf16_bits_to_f32(q)).permute(1, 0, 2)
    Ka = torch.from_numpy(I.bf16_bits_to_f32(K)).permute(1, 0, 2).repeat_interleave(G, 0)
    Va = torch.from_numpy(I.bf16_bits_to_f32(V)).permute(1, 0, 2).repeat_interleave(G, 0)
    j = torch.arange(T_h + n)[None, :]
    i = torch.arange(n)[:, None]
    ref = torch.nn.functional.scaled_dot_product_attention(qa, Ka, Va, attn_mask=(j <= T_h + i))
    ref = ref.permute(1, 0, 2).numpy()
    assert np.abs(out - ref).max() < 5e-5 * max(1.0, float(np.abs(ref).max()))
    assert np.linalg.norm(out - ref) / np.linalg.norm(ref) < 1e-5


# ------------------------------------------------------------------------ O6
def test_multi_turn_tables_stay_disjoint_and_history_grows():
    """O6 in miniature: 3 conversations, 3 turns, one shared pool."""
    L, Hq, Hkv, D, B, NB, n = 1, 2, 2, 16, 16, 64, 20
    hist = [37, 16, 5]
    tables, free = I.deal_tables(5, NB, [O.blocks_for(h, B) for h in hist])
    tables = [list(t) for t in tables]
    free = list(free)
    pool = O.Pool(L, Hkv, D, B, NB)
    logical = []
    for c, h in enumerate(hist):
        kh, vh = I.normal_bf16((h, Hkv, D), 200 + c), I.normal_bf16((h, Hkv, D), 300 + c)
        pool.store(0, 0, kh, 0, tables[c])
        pool.store(0, 1, vh, 0, tables[c])
        logical.append([kh, vh])
    for turn in range(3):
        for c in range(3):
            q, _, _, kn, vn = I.make_qkv(n, 0, Hq, Hkv, D, 1000 + 10 * turn + c)
            k = O.append_count(hist[c], n, B)
            tables[c] += [free.pop(0) for _ in range(k)]
            out = O.prefill_layer(pool, 0, q, kn, vn, tables[c], hist[c])
            mono = O.attention(q, np.concatenate([logical[c][0], kn]),
                               np.concatenate([logical[c][1], vn]), hist[c])
            assert np.array_equal(out, mono)
            logical[c] = [np.concatenate([logical[c][0], kn]), np.concatenate([logical[c][1], vn])]
            hist[c] += n
        allb = sum(tables, [])
        assert len(allb) == len(set(allb))
    for c in range(3):
        assert np.array_equal(pool.gather(0, 0, tables[c], hist[c]), logical[c][0])
        assert np.array_equal(pool.gather(0, 1, tables[c], hist[c]), logical[c][1])


# ------------------------------------------------------------------ sizing and elasticity (O7)
def test_lsc_rc_worked_example_from_the_paper():
    """L=10, K_master=100, K_1=9, K_2=8 -> N_LSC=17, N_RC=8, 25 blocks vs 10."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "lsc_rc_worked_example.txt")) if l.strip() and l[0] != "#"]
    for L, k_master, k1, k2, n_lsc, n_rc, total, conventional in (map(int, r) for r in rows):
        m_block = 4096                                   # any block size gives the same counts
        got = O.lsc_rc_sizing(k_master * m_block + 17, [k1 * m_block * L + 5, k2 * m_block * L], m_block, L)
        assert (got["k_master"], got["sum_k"]) == (k_master, k1 + k2)
        assert (got["n_lsc"], got["n_rc"], got["max_context_blocks"], got["conventional_blocks"]) == \
               (n_lsc, n_rc, total, conventional)


def test_lsc_fills_the_master_when_workers_offer_more():
    """Eq. 4-5: sum K_i >= K_master -> N_LSC = K_master and no regular cache."""
    got = O.lsc_rc_sizing(100 * 64, [90 * 64 * 4, 80 * 64 * 4], 64, 4)
    assert (got["n_lsc"], got["n_rc"]) == (100, 0)
    got = O.lsc_rc_sizing(100 * 64, [], 64, 4)           # no workers: all regular cache
    assert (got["n_lsc"], got["n_rc"], got["conventional_blocks"]) == (0, 25, 25)


def test_meu_is_the_lcm_split_brute_force():
    """Eq. 8-9 against a brute-force search of the least common multiple."""
    rng = np.random.default_rng(9)
    for _ in range(200):
        a, b = int(rng.integers(1, 400)), int(rng.integers(1, 400))
        lcm = next(x for x in range(max(a, b), a * b + 1, max(a, b)) if x % a == 0 and x % b == 0)
        mm, mi = O.meu(a, b)
        assert mm * a == mi * b == lcm
        assert math.gcd(mm, mi) == 1                     # the smallest such pair


def test_meu_of_the_papers_models():
    """Table 2 shapes: LWM 32/32/128 master, Qwen3-14B 40/8/128 worker, B=16."""
    be_m, be_i = O.block_elems(32, 16, 32, 128), O.block_elems(40, 16, 8, 128)
    assert (be_m, be_i) == (2097152, 655360)
    assert O.meu(be_m, be_i) == (5, 16)                  # 5 master blocks == 16 worker blocks, in elements
    assert O.meu(be_m, be_m) == (1, 1)


@pytest.mark.parametrize("n_i,b_i,meu_i,meu_m,length,want", [
    (10, 16, 3, 2, 160, (0, 0)),      # need 10 <= 10
    (10, 16, 3, 2, 161, (3, 2)),      # need 11, diff 1, k 1
    (10, 16, 3, 2, 200, (3, 2)),      # need 13, diff 3, k 1
    (10, 16, 3, 2, 209, (6, 4)),      # need 14, diff 4, k 2
    (0, 16, 16, 5, 1, (16, 5)),
])
def test_algorithm1_scale_up_hand_cases(n_i, b_i, meu_i, meu_m, length, want):
    assert O.scale_up(n_i, b_i, meu_i, meu_m, length) == want


@pytest.mark.parametrize("n_i,b_i,meu_i,meu_m,max_len,want", [
    (20, 16, 3, 2, 320, (0, 0)),      # max_need 20 >= 20
    (20, 16, 3, 2, 305, (0, 0)),      # max_need 20
    (20, 16, 3, 2, 290, (0, 0)),      # max_need 19, diff 1, k 0
    (20, 16, 3, 2, 100, (12, 8)),     # max_need 7, diff 13, k 4
    (32, 16, 16, 5, 0, (32, 10)),
])
def test_algorithm1_scale_down_hand_cases(n_i, b_i, meu_i, meu_m, max_len, want):
    assert O.scale_down(n_i, b_i, meu_i, meu_m, max_len) == want


def test_scale_up_then_down_returns_whole_units():
    """Both directions move multiples of (MEU_i, MEU_m) in the same ratio: no element is stranded."""
    mm, mi = O.meu(O.block_elems(32, 16, 32, 128), O.block_elems(36, 16, 8, 128))
    for length in (1, 500, 5000, 70000):
        dw, dm = O.scale_up(7, 16, mi, mm, length)
        assert dw % mi == 0 and dm % mm == 0 and dw // mi == dm // mm
        bw, bm = O.scale_down(7 + dw, 16, mi, mm, 16 * 7)
        assert bw % mi == 0 and bm % mm == 0 and bw // mi == bm // mm and bw <= dw
