"""ctypes front end of the CPU oracle (oracle/sc_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / ``--impl reference`` legs, never by the product
package.  It imports nothing from ``paper_2606_16135_b200``.

Every array is numpy; bf16 tensors are ``uint16`` bit patterns.  The steps
(O1..O6) and the passages they follow are listed in sc_oracle.c's header and
in DESIGN.md section 3.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sc_oracle.c")
_LIB = os.path.join(_HERE, "libsc_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile sc_oracle.c with gcc (-O2 -fopenmp) next to its source."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True, capture_output=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        lib = C.CDLL(build())
        u16p, i32p = C.POINTER(C.c_uint16), C.POINTER(C.c_int32)
        f32p, f64p = C.POINTER(C.c_float), C.POINTER(C.c_double)
        lib.sco_pool_new.restype = C.c_void_p
        lib.sco_pool_new.argtypes = [C.c_int32] * 5
        lib.sco_pool_free.argtypes = [C.c_void_p]
        lib.sco_block_bytes.restype = C.c_int64
        lib.sco_block_bytes.argtypes = [C.c_int32] * 4
        lib.sco_kv_bytes_per_token.restype = C.c_int64
        lib.sco_kv_bytes_per_token.argtypes = [C.c_int32] * 4
        lib.sco_store.argtypes = [C.c_void_p, C.c_int32, C.c_int32, u16p, C.c_int32, C.c_int32,
                                  i32p, C.c_int32]
        lib.sco_gather.argtypes = [C.c_void_p, C.c_int32, C.c_int32, i32p, C.c_int32, C.c_int32, u16p]
        lib.sco_blocks_for.argtypes = [C.c_int32, C.c_int32]
        lib.sco_append_count.argtypes = [C.c_int32] * 3
        common = [u16p, u16p, u16p] + [C.c_int32] * 5
        lib.sco_attention_f32.argtypes = common + [f32p, f32p]
        lib.sco_attention_f64.argtypes = common + [f64p, f64p]
        lib.sco_softmax_row_f32.argtypes = [u16p, u16p] + [C.c_int32] * 6 + [f32p]
        i64p = C.POINTER(C.c_int64)
        lib.sco_lsc_rc_sizing.argtypes = [C.c_int64, i64p, C.c_int32, C.c_int64, C.c_int32, i64p]
        lib.sco_block_elems.restype = C.c_int64
        lib.sco_block_elems.argtypes = [C.c_int32] * 4
        lib.sco_meu.argtypes = [C.c_int64, C.c_int64, i64p, i64p]
        lib.sco_scale_up.restype = None
        lib.sco_scale_up.argtypes = [C.c_int64] * 5 + [i64p, i64p]
        lib.sco_scale_down.restype = None
        lib.sco_scale_down.argtypes = [C.c_int64] * 5 + [i64p, i64p]
        _lib = lib
        return lib


def _u16(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a, a.ctypes.data_as(C.POINTER(C.c_uint16))


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int32))


def openmp_threads() -> int:
    return int(_load().sco_openmp_threads())


def block_bytes(B: int, Hkv: int, D: int, dtype_bytes: int = 2) -> int:
    """Eq. 1."""
    return int(_load().sco_block_bytes(B, Hkv, D, dtype_bytes))


def kv_bytes_per_token(L: int, Hkv: int, D: int, dtype_bytes: int = 2) -> int:
    """Table 2."""
    return int(_load().sco_kv_bytes_per_token(L, Hkv, D, dtype_bytes))


def blocks_for(tokens: int, B: int) -> int:
    return int(_load().sco_blocks_for(tokens, B))


def append_count(hist_len: int, n_new: int, B: int) -> int:
    """O5: new table entries needed so the table covers hist_len+n_new tokens."""
    return int(_load().sco_append_count(hist_len, n_new, B))


def lsc_rc_sizing(c_master: int, c_workers, m_block: int, L: int) -> dict:
    """Eq. 2-5: LSC and RC capacities in blocks."""
    cw = (C.c_int64 * max(len(c_workers), 1))(*c_workers)
    out = (C.c_int64 * 6)()
    if _load().sco_lsc_rc_sizing(c_master, cw, len(c_workers), m_block, L, out):
        raise ValueError("sco_lsc_rc_sizing")
    keys = ("k_master", "sum_k", "n_lsc", "n_rc", "max_context_blocks", "conventional_blocks")
    return dict(zip(keys, (int(x) for x in out)))


def block_elems(L: int, B: int, Hkv: int, D: int) -> int:
    """Eq. 6 / 7."""
    return int(_load().sco_block_elems(L, B, Hkv, D))


def meu(be_m: int, be_i: int):
    """Eq. 8-9: (MEU_m, MEU_i)."""
    a, b = C.c_int64(), C.c_int64()
    if _load().sco_meu(be_m, be_i, C.byref(a), C.byref(b)):
        raise ValueError("sco_meu")
    return int(a.value), int(b.value)


def scale_up(n_i, b_i, meu_i, meu_m, request_len):
    """Algorithm 1 ScaleUp: (blocks the worker gains, blocks the master gives up)."""
    a, b = C.c_int64(), C.c_int64()
    _load().sco_scale_up(n_i, b_i, meu_i, meu_m, request_len, C.byref(a), C.byref(b))
    return int(a.value), int(b.value)


def scale_down(n_i, b_i, meu_i, meu_m, max_len):
    """Algorithm 1 ScaleDown: (blocks the worker releases, blocks the master gains)."""
    a, b = C.c_int64(), C.c_int64()
    _load().sco_scale_down(n_i, b_i, meu_i, meu_m, max_len, C.byref(a), C.byref(b))
    return int(a.value), int(b.value)


class Pool:
    """O1: block-major pool of NB full-layer blocks."""

    def __init__(self, L: int, Hkv: int, D: int, B: int, NB: int):
        self.L, self.Hkv, self.D, self.B, self.NB = L, Hkv, D, B, NB
        self._lib = _load()
        self._p = self._lib.sco_pool_new(L, Hkv, D, B, NB)
        if not self._p:
            raise MemoryError("sco_pool_new")

    def __del__(self):
        if getattr(self, "_p", None):
            self._lib.sco_pool_free(self._p)
            self._p = None

    def store(self, layer: int, kv: int, X: np.ndarray, start: int, table) -> None:
        """O2: X [n][Hkv][D] (bf16 bits) -> logical tokens start..start+n-1."""
        X, xp = _u16(X)
        assert X.ndim == 3 and X.shape[1:] == (self.Hkv, self.D), X.shape
        table, tp = _i32(table)
        rc = self._lib.sco_store(self._p, layer, kv, xp, start, X.shape[0], tp, len(table))
        if rc:
            raise IndexError("sco_store: table too short or block id out of range")

    def gather(self, layer: int, kv: int, table, T: int) -> np.ndarray:
        """O3: logical tokens 0..T-1 of one layer as [T][Hkv][D] bf16 bits."""
        table, tp = _i32(table)
        out = np.empty((T, self.Hkv, self.D), dtype=np.uint16)
        rc = self._lib.sco_gather(self._p, layer, kv, tp, len(table), T,
                                  out.ctypes.data_as(C.POINTER(C.c_uint16)))
        if rc:
            raise IndexError("sco_gather: table too short or block id out of range")
        return out


def attention(q, K, V, T_h: int, dtype=np.float32, return_rowsum: bool = False):
    """O4.  q [n][Hq][D], K/V [T_h+n][Hkv][D] as bf16 bits -> out [n][Hq][D] `dtype`."""
    lib = _load()
    q, qp = _u16(q)
    K, kp = _u16(K)
    V, vp = _u16(V)
    n, Hq, D = q.shape
    assert K.shape == V.shape and K.shape[0] == T_h + n and K.shape[2] == D, (K.shape, V.shape)
    Hkv = K.shape[1]
    out = np.empty((n, Hq, D), dtype=dtype)
    rs = np.empty((n, Hq), dtype=dtype)
    if dtype == np.float32:
        fn, ptr = lib.sco_attention_f32, C.POINTER(C.c_float)
    elif dtype == np.float64:
        fn, ptr = lib.sco_attention_f64, C.POINTER(C.c_double)
    else:
        raise TypeError(dtype)
    rc = fn(qp, kp, vp, n, T_h, Hq, Hkv, D, out.ctypes.data_as(ptr), rs.ctypes.data_as(ptr))
    if rc:
        raise ValueError(f"sco_attention rc={rc}")
    return (out, rs) if return_rowsum else out


def softmax_row(q, K, T_h: int, i: int, h: int) -> np.ndarray:
    """Softmax weights of new token i, head h over keys 0..T_h+i (fp32)."""
    lib = _load()
    q, qp = _u16(q)
    K, kp = _u16(K)
    _, Hq, D = q.shape
    p = np.empty(T_h + i + 1, dtype=np.float32)
    rc = lib.sco_softmax_row_f32(qp, kp, T_h, i, h, Hq, K.shape[1], D,
                                 p.ctypes.data_as(C.POINTER(C.c_float)))
    if rc:
        raise ValueError("sco_softmax_row_f32")
    return p


def prefill_layer(pool: Pool, layer: int, q, k_new, v_new, table, hist_len: int,
                  dtype=np.float32):
    """One layer of one turn, in the paper's order: O3 gather the history into
    the (oracle's) LSC, O5/O2 scatter the new K/V into the pool, O4 attend
    over [LSC ; new].  `table` must already cover hist_len+n tokens.
    Returns out [n][Hq][D]."""
    lsc_k = pool.gather(layer, 0, table, hist_len)
    lsc_v = pool.gather(layer, 1, table, hist_len)
    pool.store(layer, 0, k_new, hist_len, table)
    pool.store(layer, 1, v_new, hist_len, table)
    K = np.concatenate([lsc_k, np.ascontiguousarray(k_new)], axis=0)
    V = np.concatenate([lsc_v, np.ascontiguousarray(v_new)], axis=0)
    return attention(q, K, V, hist_len, dtype=dtype)
