"""ctypes binding of libswiftcache.so: the same names as include/swiftcache.h.

Argument marshalling only -- every step of the path runs in the library's
CUDA kernels.  There is no CPU fallback: if the shared library is missing the
import of :func:`lib` raises, and every data call on a machine without a CUDA
device returns SC_ERR_CUDA, which :func:`check` turns into an exception.

torch is used by callers for device memory and streams; this module itself
needs only pointers (``tensor.data_ptr()``) and stream handles
(``torch.cuda.current_stream().cuda_stream``).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libswiftcache.so")

SC_OK, SC_ERR_INVALID_ARG, SC_ERR_OUT_OF_BLOCKS, SC_ERR_CAPACITY = 0, 1, 2, 3
SC_ERR_BAD_BLOCK_ID, SC_ERR_CUDA, SC_ERR_UNSUPPORTED = 4, 5, 6
SC_POOL_HBM, SC_POOL_HOST_PINNED, SC_POOL_PEER = 0, 1, 2
SC_ATTN_STAGED, SC_ATTN_FUSED = 0, 1
SC_MEM_DEVICE, SC_MEM_HOST_PINNED = 0, 1
SC_ENGINE_AUTO, SC_ENGINE_MMA_SYNC, SC_ENGINE_TCGEN05, SC_ENGINE_DECODE = 0, 1, 2, 3
SC_COPY_AUTO, SC_COPY_LDG, SC_COPY_BULK = 0, 1, 2
SC_MAX_SEQS = 32
SC_STATIC_SCRATCH_BYTES = 32 << 20

STATUS_NAMES = {0: "SC_OK", 1: "SC_ERR_INVALID_ARG", 2: "SC_ERR_OUT_OF_BLOCKS", 3: "SC_ERR_CAPACITY",
                4: "SC_ERR_BAD_BLOCK_ID", 5: "SC_ERR_CUDA", 6: "SC_ERR_UNSUPPORTED"}

# every symbol include/swiftcache.h declares (tests check the library exports them all)
SYMBOLS = [
    "sc_version", "sc_last_error", "sc_pool_bytes_required", "sc_pool_create", "sc_pool_destroy",
    "sc_pool_info", "sc_cell_offset", "sc_lsc_offset", "sc_set_engine", "sc_set_split_tiles",
    "sc_alloc_blocks", "sc_free_blocks", "sc_num_free_blocks", "sc_append_blocks", "sc_store_prefix",
    "sc_read_tokens", "sc_load_layer", "sc_prefill_layer", "sc_load_layer_batched",
    "sc_prefill_layer_batched", "sc_prefill_turn", "sc_launch_count", "sc_profile_enable",
    "sc_profile_collect", "sc_lsc_rc_sizing", "sc_elastic_units", "sc_scale_up", "sc_scale_down",
    "sc_pool_resize", "sc_set_resident_blocks", "sc_prefill_turn_ex", "sc_prefill_layer_static",
]


class sc_pool_config_t(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("block_size", C.c_int32), ("n_blocks", C.c_int32),
                ("pool_kind", C.c_int32), ("lsc_blocks", C.c_int32), ("max_new_tokens", C.c_int32),
                ("max_seqs", C.c_int32), ("alloc_seed", C.c_uint64)]


class sc_pool_info_t(C.Structure):
    _fields_ = [("chunk_bytes", C.c_int64), ("cell_bytes", C.c_int64), ("block_bytes", C.c_int64),
                ("pool_bytes", C.c_int64), ("lsc_buffer_bytes", C.c_int64), ("lsc_bytes", C.c_int64),
                ("scratch_bytes", C.c_int64), ("n_free_blocks", C.c_int32), ("max_splits", C.c_int32)]


class sc_sizing_t(C.Structure):
    _fields_ = [("k_master", C.c_int64), ("sum_k", C.c_int64), ("n_lsc", C.c_int64), ("n_rc", C.c_int64),
                ("max_context_blocks", C.c_int64), ("conventional_blocks", C.c_int64)]


LAYER_HOOK = C.CFUNCTYPE(None, C.c_int32, C.c_void_p, C.c_void_p)


class sc_turn_options_t(C.Structure):
    _fields_ = [("lsc_buffers", C.c_int32), ("after_attention", LAYER_HOOK), ("user", C.c_void_p)]


class SwiftCacheError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


_lib = None


def lib() -> C.CDLL:
    """Load libswiftcache.so (built by ``python -m paper_2606_16135_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_16135_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    i32, i64, vp, sz = C.c_int32, C.c_int64, C.c_void_p, C.c_size_t
    i32p = C.POINTER(C.c_int32)
    L.sc_version.restype = C.c_char_p
    L.sc_last_error.restype = C.c_char_p
    sig = {
        "sc_pool_bytes_required": [C.POINTER(sc_pool_config_t), C.POINTER(sz), C.POINTER(sz)],
        "sc_pool_create": [C.POINTER(sc_pool_config_t), vp, sz, vp, sz, i32, C.POINTER(vp)],
        "sc_pool_destroy": [vp],
        "sc_pool_info": [vp, C.POINTER(sc_pool_info_t)],
        "sc_cell_offset": [vp, i32, i32, i32, i32, i32, i32, C.POINTER(i64)],
        "sc_lsc_offset": [vp, i32, i32, i32, i32, i32, i32, C.POINTER(i64)],
        "sc_set_engine": [vp, i32, i32],
        "sc_set_split_tiles": [vp, i32],
        "sc_alloc_blocks": [vp, i32, i32p],
        "sc_free_blocks": [vp, i32p, i32],
        "sc_num_free_blocks": [vp, i32p],
        "sc_append_blocks": [vp, i32p, i32p, i32, i32, i32],
        "sc_store_prefix": [vp, i32, vp, vp, i32, i32, vp, i32, vp],
        "sc_read_tokens": [vp, i32, i32, vp, i32, i32, i32, i32, vp, vp, vp],
        "sc_load_layer": [vp, i32, vp, i32, i32, i32, vp],
        "sc_prefill_layer": [vp, i32, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp],
        "sc_load_layer_batched": [vp, i32, vp, i32, i32, i32p, i32p, i32, vp],
        "sc_prefill_layer_batched": [vp, i32, vp, vp, vp, vp, i32, i32, i32p, i32p, i32, i32, vp, vp],
        "sc_prefill_turn": [vp, vp, vp, vp, vp, i32, vp, i32, i32, i32p, i32p, i32, vp, vp],
        "sc_prefill_turn_ex": [vp, vp, vp, vp, vp, i32, vp, i32, i32, i32p, i32p, i32, vp, vp,
                               C.POINTER(sc_turn_options_t)],
        "sc_launch_count": [vp, C.POINTER(i64)],
        "sc_profile_enable": [vp, i32],
        "sc_profile_collect": [vp, C.POINTER(C.c_double), C.POINTER(i64)],
        "sc_lsc_rc_sizing": [C.POINTER(sc_pool_config_t), i64, C.POINTER(i64), i32, C.POINTER(sc_sizing_t)],
        "sc_elastic_units": [C.POINTER(sc_pool_config_t), C.POINTER(sc_pool_config_t), C.POINTER(i64), C.POINTER(i64)],
        "sc_scale_up": [i64, i32, i64, i64, i64, C.POINTER(i64), C.POINTER(i64)],
        "sc_scale_down": [i64, i32, i64, i64, i64, C.POINTER(i64), C.POINTER(i64)],
        "sc_pool_resize": [vp, i32, sz, i32, vp],
        "sc_set_resident_blocks": [vp, i32],
        "sc_prefill_layer_static": [C.POINTER(sc_pool_config_t), vp, i32, vp, vp, vp, vp, i32, i32, i32, i32, vp, vp],
    }
    for name, argtypes in sig.items():
        fn = getattr(L, name)
        fn.argtypes = argtypes
        fn.restype = i32
    _lib = L
    return L


def check(status: int) -> None:
    if status != SC_OK:
        raise SwiftCacheError(status, lib().sc_last_error().decode())


def _i32_array(x):
    a = np.ascontiguousarray(x, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int32))


def sc_version() -> str:
    return lib().sc_version().decode()


def sc_pool_bytes_required(cfg: sc_pool_config_t):
    p, l = C.c_size_t(), C.c_size_t()
    check(lib().sc_pool_bytes_required(C.byref(cfg), C.byref(p), C.byref(l)))
    return int(p.value), int(l.value)


def sc_lsc_rc_sizing(cfg: sc_pool_config_t, c_master_bytes: int, c_worker_bytes) -> dict:
    cw = (C.c_int64 * max(len(c_worker_bytes), 1))(*c_worker_bytes)
    out = sc_sizing_t()
    check(lib().sc_lsc_rc_sizing(C.byref(cfg), c_master_bytes, cw, len(c_worker_bytes), C.byref(out)))
    return {k: int(getattr(out, k)) for k, _ in sc_sizing_t._fields_}


def sc_elastic_units(master: sc_pool_config_t, worker: sc_pool_config_t):
    a, b = C.c_int64(), C.c_int64()
    check(lib().sc_elastic_units(C.byref(master), C.byref(worker), C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def sc_scale_up(n_worker_blocks, block_size, meu_worker, meu_master, request_len):
    a, b = C.c_int64(), C.c_int64()
    check(lib().sc_scale_up(n_worker_blocks, block_size, meu_worker, meu_master, request_len, C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def sc_scale_down(n_worker_blocks, block_size, meu_worker, meu_master, max_len):
    a, b = C.c_int64(), C.c_int64()
    check(lib().sc_scale_down(n_worker_blocks, block_size, meu_worker, meu_master, max_len, C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def sc_prefill_layer_static(cfg: sc_pool_config_t, pool_ptr: int, layer: int, q_ptr: int, k_new_ptr: int,
                            v_new_ptr: int, table_ptr: int, n_table: int, hist_len: int, n_new: int,
                            tiles_per_split: int, out_ptr: int, stream: int = 0) -> None:
    """One layer of prefill without a Pool object and without any allocation (see swiftcache.h):
    for processes that have given all their HBM to the block pool, or that must not stall the GPU
    with cudaMalloc.  The split-KV partials live in a fixed SC_STATIC_SCRATCH_BYTES array inside the
    library, ONE per GPU: calls that could overlap on the GPU must be ordered by the caller.
    ``k_new_ptr`` / ``v_new_ptr`` may both be 0 when the new tokens are in the pool already."""
    check(lib().sc_prefill_layer_static(C.byref(cfg), pool_ptr or None, layer, q_ptr or None, k_new_ptr or None,
                                        v_new_ptr or None, table_ptr or None, n_table, hist_len, n_new,
                                        tiles_per_split, out_ptr or None, stream or None))


def make_config(L, Hq, Hkv, D, B, n_blocks, lsc_blocks, max_new_tokens, max_seqs=1,
                pool_kind=SC_POOL_HBM, alloc_seed=0) -> sc_pool_config_t:
    return sc_pool_config_t(L, Hq, Hkv, D, B, n_blocks, pool_kind, lsc_blocks, max_new_tokens,
                            max_seqs, alloc_seed)


class Pool:
    """Thin handle around sc_pool_t*; method names are the C names without ``sc_``.

    ``pool_ptr`` / ``lsc_ptr`` are raw addresses of caller-owned memory (0 for a
    host-only pool).  Keep the owning tensors alive for the life of the pool.
    """

    def __init__(self, cfg: sc_pool_config_t, pool_ptr: int = 0, pool_bytes: int = 0,
                 lsc_ptr: int = 0, lsc_bytes: int = 0, zero_fill: bool = True):
        self.cfg = cfg
        self._h = C.c_void_p()
        check(lib().sc_pool_create(C.byref(cfg), pool_ptr or None, pool_bytes, lsc_ptr or None,
                                   lsc_bytes, int(zero_fill), C.byref(self._h)))

    def destroy(self):
        if self._h:
            check(lib().sc_pool_destroy(self._h))
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- geometry
    def info(self) -> sc_pool_info_t:
        i = sc_pool_info_t()
        check(lib().sc_pool_info(self._h, C.byref(i)))
        return i

    def cell_offset(self, block, layer, kv, head, slot, d) -> int:
        o = C.c_int64()
        check(lib().sc_cell_offset(self._h, block, layer, kv, head, slot, d, C.byref(o)))
        return int(o.value)

    def lsc_offset(self, buf, lblock, kv, head, slot, d) -> int:
        o = C.c_int64()
        check(lib().sc_lsc_offset(self._h, buf, lblock, kv, head, slot, d, C.byref(o)))
        return int(o.value)

    def set_engine(self, attn_engine=SC_ENGINE_AUTO, copy_engine=SC_COPY_AUTO):
        check(lib().sc_set_engine(self._h, attn_engine, copy_engine))

    def set_split_tiles(self, tiles_per_split: int):
        check(lib().sc_set_split_tiles(self._h, tiles_per_split))

    def resize(self, new_n_blocks: int, new_pool_bytes: int = 0, zero_fill: bool = True, stream=0):
        check(lib().sc_pool_resize(self._h, new_n_blocks, new_pool_bytes, int(zero_fill), stream or None))
        self.cfg.n_blocks = new_n_blocks

    def set_resident_blocks(self, n_blocks: int):
        check(lib().sc_set_resident_blocks(self._h, n_blocks))

    def launch_count(self) -> int:
        n = C.c_int64()
        check(lib().sc_launch_count(self._h, C.byref(n)))
        return int(n.value)

    def profile_enable(self, on: bool):
        check(lib().sc_profile_enable(self._h, int(on)))

    def profile_collect(self):
        """{kind: (summed ms, launches)} for gather / scatter / attention / combine."""
        ms = (C.c_double * 4)()
        cnt = (C.c_int64 * 4)()
        check(lib().sc_profile_collect(self._h, ms, cnt))
        names = ("gather", "scatter", "attention", "combine")
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(names)}

    # ---- allocator / tables (host)
    def alloc_blocks(self, n: int) -> np.ndarray:
        ids = np.empty(max(n, 1), dtype=np.int32)
        check(lib().sc_alloc_blocks(self._h, n, ids.ctypes.data_as(C.POINTER(C.c_int32))))
        return ids[:n]

    def free_blocks(self, ids) -> None:
        a, p = _i32_array(ids)
        check(lib().sc_free_blocks(self._h, p, len(a)))

    def num_free_blocks(self) -> int:
        n = C.c_int32()
        check(lib().sc_num_free_blocks(self._h, C.byref(n)))
        return int(n.value)

    def append_blocks(self, table: np.ndarray, n_table: int, hist_len: int, n_new: int) -> int:
        """`table` is an int32 numpy array of capacity len(table); returns the new n_table."""
        assert table.dtype == np.int32 and table.flags["C_CONTIGUOUS"]
        n = C.c_int32(n_table)
        check(lib().sc_append_blocks(self._h, table.ctypes.data_as(C.POINTER(C.c_int32)), C.byref(n),
                                     len(table), hist_len, n_new))
        return int(n.value)

    # ---- data calls (pointers are ints; streams are cudaStream_t handles as ints)
    def store_prefix(self, layer, k_ptr, v_ptr, start_token, n_tokens, table_ptr, n_table, stream=0):
        check(lib().sc_store_prefix(self._h, layer, k_ptr, v_ptr, start_token, n_tokens, table_ptr,
                                    n_table, stream or None))

    def read_tokens(self, layer, src, table_ptr, n_table, lsc_block_off, start_token, n_tokens,
                    k_out_ptr, v_out_ptr, stream=0):
        check(lib().sc_read_tokens(self._h, layer, src, table_ptr or None, n_table, lsc_block_off,
                                   start_token, n_tokens, k_out_ptr, v_out_ptr, stream or None))

    def load_layer(self, layer, table_ptr, n_table, hist_len, buf, stream=0):
        check(lib().sc_load_layer(self._h, layer, table_ptr, n_table, hist_len, buf, stream or None))

    def prefill_layer(self, layer, q_ptr, k_new_ptr, v_new_ptr, table_ptr, n_table, hist_len, n_new,
                      buf, mode, out_ptr, stream=0):
        check(lib().sc_prefill_layer(self._h, layer, q_ptr, k_new_ptr, v_new_ptr, table_ptr, n_table,
                                     hist_len, n_new, buf, mode, out_ptr, stream or None))

    def load_layer_batched(self, layer, tables_ptr, max_blocks, hist_lens, cu_new, buf, stream=0):
        h, hp = _i32_array(hist_lens)
        c, cp = _i32_array(cu_new)
        check(lib().sc_load_layer_batched(self._h, layer, tables_ptr, max_blocks, len(h), hp, cp, buf,
                                          stream or None))

    def prefill_layer_batched(self, layer, q_ptr, k_new_ptr, v_new_ptr, tables_ptr, max_blocks,
                              hist_lens, cu_new, buf, mode, out_ptr, stream=0):
        h, hp = _i32_array(hist_lens)
        c, cp = _i32_array(cu_new)
        check(lib().sc_prefill_layer_batched(self._h, layer, q_ptr, k_new_ptr, v_new_ptr, tables_ptr,
                                             max_blocks, len(h), hp, cp, buf, mode, out_ptr,
                                             stream or None))

    def prefill_turn(self, q_all_ptr, k_all_ptr, v_all_ptr, out_all_ptr, io_kind, tables_ptr,
                     max_blocks, hist_lens, cu_new, mode, copy_stream, compute_stream):
        h, hp = _i32_array(hist_lens)
        c, cp = _i32_array(cu_new)
        check(lib().sc_prefill_turn(self._h, q_all_ptr, k_all_ptr, v_all_ptr, out_all_ptr, io_kind,
                                    tables_ptr, max_blocks, len(h), hp, cp, mode, copy_stream or None,
                                    compute_stream or None))

    def prefill_turn_ex(self, q_all_ptr, k_all_ptr, v_all_ptr, out_all_ptr, io_kind, tables_ptr,
                        max_blocks, hist_lens, cu_new, mode, copy_stream, compute_stream,
                        lsc_buffers=2, after_attention=None):
        """`after_attention(layer, compute_stream_handle)` is a Python callable run on the host
        after each layer has been enqueued (it may enqueue work on the compute stream).

        ctypes cannot carry a Python exception through the C frames of the library (it prints it
        and goes on), so the trampoline keeps the FIRST exception the hook raises, skips the hook
        for the remaining layers, and this method re-raises it once the C call has returned.  The
        library has by then enqueued every layer: the turn's own results are complete, only the
        hook's work is missing from that layer on."""
        h, hp = _i32_array(hist_lens)
        c, cp = _i32_array(cu_new)
        raised = []

        def trampoline(layer, stream, user):
            if raised:
                return
            try:
                after_attention(layer, stream)
            except BaseException as e:      # noqa: BLE001 -- re-raised below, outside the C frames
                raised.append(e)

        hook = LAYER_HOOK(trampoline) if after_attention else LAYER_HOOK()
        opt = sc_turn_options_t(lsc_buffers, hook, None)
        status = lib().sc_prefill_turn_ex(self._h, q_all_ptr, k_all_ptr, v_all_ptr, out_all_ptr, io_kind,
                                          tables_ptr, max_blocks, len(h), hp, cp, mode, copy_stream or None,
                                          compute_stream or None, C.byref(opt))
        if raised:
            raise raised[0]
        check(status)
