"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: it only draws random
numbers, rounds them to bf16 and deals out block tables.  Both the CUDA path
and the CPU oracle receive what it returns; neither side's code lives here.

Recipe: values are fp32
N(0,1)*0.5 rounded to nearest-even bf16; block tables are the first entries of
a seeded permutation of the pool's block ids.  The shapes are those of the
paper's workloads -- LWM-1M-Text / Llama-2-7B MHA 32 layers x 32 heads x 128
(Table 2; Fig. 1) and a Qwen3-style GQA 32/8
shape -- and stand in for ShareGPT / L-Eval requests, which are not available.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 16135


@dataclass(frozen=True)
class Shape:
    """One BASELINE.json config.  hist/n_new are per conversation."""
    name: str
    config_id: int
    L: int
    Hq: int
    Hkv: int
    D: int
    B: int
    hist: tuple
    n_new: int
    n_blocks: int
    turns: int = 1
    pool_kind: str = "hbm"
    extra: dict = field(default_factory=dict)

    @property
    def tok_bytes(self) -> int:
        """K+V bytes of one token in one layer (bf16)."""
        return 2 * self.Hkv * self.D * 2

    @property
    def block_bytes(self) -> int:
        return self.B * self.tok_bytes


def config5_lengths() -> tuple:
    """8 history lengths, integers uniform on [1024, 32768], not rounded to B."""
    r = np.random.default_rng(BASE_SEED).integers(1024, 32769, size=8)
    return tuple(int(x) for x in r)


def _blocks(tokens: int, B: int) -> int:
    return -(-tokens // B)


def configs() -> dict:
    c5 = config5_lengths()
    c5_blocks = sum(_blocks(h + 10 * 256, 16) for h in c5)
    return {
        "tiny": Shape("tiny", 1, 2, 4, 4, 64, 16, (512,), 32, 64),
        "lwm_5k": Shape("lwm_5k", 2, 32, 32, 32, 128, 16, (5120,), 256, 320 + 16 + 48),
        "lwm_50k": Shape("lwm_50k", 3, 32, 32, 32, 128, 16, (50000,), 256, 3125 + 17 + 58),
        "gqa_128k": Shape("gqa_128k", 4, 32, 32, 8, 128, 16, (131072,), 256, 8192 + 16 + 48),
        "gqa_128k_host": Shape("gqa_128k_host", 4, 32, 32, 8, 128, 16, (131072,), 256,
                               8192 + 16 + 48, pool_kind="host"),
        "multiturn": Shape("multiturn", 5, 32, 32, 32, 128, 16, c5, 256, c5_blocks + 33, turns=10),
    }


def seed_for(config_id: int, layer: int, what: str, turn: int = 0, conv: int = 0) -> int:
    off = {"k": 0, "q": 25, "v": 50, "k_new": 10, "v_new": 60}[what]
    return BASE_SEED * 1000 + 100 * config_id + layer + off * 1000 + 7 * turn * 100000 + conv * 10000000


# ---------------------------------------------------------------- bf16 bits --
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16 bit pattern (uint16).  No NaN inputs."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal_bf16(shape, seed: int, scale: float = 0.5) -> np.ndarray:
    """fp32 N(0,1)*scale rounded to bf16; returned as uint16 bits (host)."""
    g = np.random.default_rng(seed)
    return f32_to_bf16_bits(g.standard_normal(shape, dtype=np.float32) * np.float32(scale))


def normal_bf16_device(shape, seed: int, device, scale: float = 0.5):
    """Same distribution drawn on the device with a seeded torch generator
    (for histories too large to ship from the host).  Returns a torch bf16
    tensor; the host copy of the same bits is ``t.view(torch.int16).cpu()``."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    x = torch.randn(shape, generator=g, device=device, dtype=torch.float32) * scale
    return x.to(torch.bfloat16)


# -------------------------------------------------------------- block tables --
def permuted_ids(config_id: int, n_blocks: int) -> np.ndarray:
    """Seeded permutation of the pool's physical block ids ("shuffled pool")."""
    return np.random.default_rng(BASE_SEED + config_id).permutation(n_blocks).astype(np.int32)


def block_table(config_id: int, n_blocks: int, n_entries: int, identity: bool = False) -> np.ndarray:
    if identity:
        return np.arange(n_entries, dtype=np.int32)
    return permuted_ids(config_id, n_blocks)[:n_entries].copy()


def deal_tables(config_id: int, n_blocks: int, counts) -> list:
    """Consecutive disjoint slices of one shared permutation, one per conversation."""
    perm = permuted_ids(config_id, n_blocks)
    out, o = [], 0
    for c in counts:
        out.append(perm[o:o + c].copy())
        o += c
    assert o <= n_blocks
    return out, perm[o:].copy()


# ------------------------------------------------------- score distributions --
def make_qkv(n_new: int, T_h: int, Hq: int, Hkv: int, D: int, seed: int, variant: str = "normal"):
    """(q, k_hist, v_hist, k_new, v_new) as bf16 bits for ONE layer.

    variant "normal": everything N(0,1)*0.5 (BASELINE.json).
    variant "peaked": q scaled x16 so the scores have std ~4 and the online
        softmax's running-max rescale is exercised.
    variant "adversarial": additionally the last history token and the last
        new token get, per KV head, a key that is the direction of an ACTUAL
        query row -- the last new token's query of the group's first query
        head -- scaled so its largest component is 4.  For that row the two
        planted keys score |q|^2 * 4 / max|q| (hundreds, against a spread of
        ~+-25 elsewhere): its largest score arrives in the last history tile
        and again at its own, last, new token.  Other rows see a large score
        of either sign there.
    """
    q = normal_bf16((n_new, Hq, D), seed + 1)
    kh = normal_bf16((T_h, Hkv, D), seed + 2)
    vh = normal_bf16((T_h, Hkv, D), seed + 3)
    kn = normal_bf16((n_new, Hkv, D), seed + 4)
    vn = normal_bf16((n_new, Hkv, D), seed + 5)
    if variant in ("peaked", "adversarial"):
        q = f32_to_bf16_bits(bf16_bits_to_f32(q) * np.float32(16.0))
    if variant == "adversarial":
        G = Hq // Hkv
        qf = bf16_bits_to_f32(q).reshape(n_new, Hkv, G, D)[n_new - 1, :, 0, :]  # [Hkv][D]: one real query row per KV head
        big = f32_to_bf16_bits(qf / np.maximum(np.abs(qf).max(axis=-1, keepdims=True), 1e-6) * np.float32(4.0))
        if T_h > 0:
            kh[T_h - 1] = big
        kn[n_new - 1] = big
    elif variant != "normal" and variant != "peaked":
        raise ValueError(variant)
    return q, kh, vh, kn, vn
