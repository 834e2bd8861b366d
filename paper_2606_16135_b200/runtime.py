"""Plumbing around the C ABI: torch owns device / pinned memory and streams, the
library does the work.  Nothing here computes anything on the path.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as sc


def bits_to_torch(bits: np.ndarray, device=None) -> torch.Tensor:
    """uint16 bf16 bit patterns (numpy) -> torch.bfloat16 tensor (same bits)."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    return t.to(device) if device is not None else t


def torch_to_bits(t: torch.Tensor) -> np.ndarray:
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def _aligned_bytes(nbytes: int, device, pinned: bool = False, align: int = 1024):
    """A uint8 tensor of nbytes whose data_ptr is `align`-byte aligned (and its owner)."""
    if pinned:
        raw = torch.empty(nbytes + align, dtype=torch.uint8, pin_memory=True)
    else:
        raw = torch.empty(nbytes + align, dtype=torch.uint8, device=device)
    off = (-raw.data_ptr()) % align
    return raw[off:off + nbytes], raw


class Session:
    """One pool + LSC + two streams on one GPU."""

    def __init__(self, L, Hq, Hkv, D, B, n_blocks, lsc_blocks, max_new_tokens, max_seqs=1,
                 pool_kind=sc.SC_POOL_HBM, alloc_seed=0, device="cuda:0", zero_fill=True, fill_byte=None,
                 pool_ptr=None):
        """`pool_ptr`: address of a pool region the caller already owns and has mapped on `device`
        (SC_POOL_PEER: another GPU's memory); otherwise the session allocates the region itself."""
        if not torch.cuda.is_available():
            raise RuntimeError("swiftcache needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.cfg = sc.make_config(L, Hq, Hkv, D, B, n_blocks, lsc_blocks, max_new_tokens, max_seqs,
                                  pool_kind, alloc_seed)
        pool_bytes, lsc_bytes = sc.sc_pool_bytes_required(self.cfg)
        if pool_ptr is None:
            self.pool_mem, self._pool_owner = _aligned_bytes(
                pool_bytes, self.device, pinned=(pool_kind == sc.SC_POOL_HOST_PINNED))
            pool_ptr = self.pool_mem.data_ptr()
        else:
            self.pool_mem = self._pool_owner = None
        self.lsc_mem, self._lsc_owner = _aligned_bytes(max(lsc_bytes, 1024), self.device)
        if fill_byte is not None:          # tests: what the borrowed memory holds before the pool exists
            if self.pool_mem is not None:  # a region the caller passed in (pool_ptr) is the caller's to fill
                self.pool_mem.fill_(fill_byte)
            self.lsc_mem.fill_(fill_byte)
        self.pool = sc.Pool(self.cfg, pool_ptr, pool_bytes,
                            self.lsc_mem.data_ptr() if lsc_blocks else 0, lsc_bytes, zero_fill=zero_fill)
        self.L, self.Hq, self.Hkv, self.D, self.B = L, Hq, Hkv, D, B
        # the compute stream outranks the copy stream: when an SM frees up, an attention CTA (which
        # needs a whole SM) is placed before the next wave of gather CTAs
        self.compute_stream = torch.cuda.Stream(device=self.device, priority=-1)
        self.copy_stream = torch.cuda.Stream(device=self.device, priority=0)

    def close(self):
        torch.cuda.synchronize(self.device)
        self.pool.destroy()

    # -- small helpers (marshalling only)
    def table_dev(self, table) -> torch.Tensor:
        return torch.from_numpy(np.ascontiguousarray(table, dtype=np.int32)).to(self.device)

    def store_prefix(self, layer, k: torch.Tensor, v: torch.Tensor, start, table_dev, stream=None):
        st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
        self.pool.store_prefix(layer, k.data_ptr(), v.data_ptr(), start, k.shape[0], table_dev.data_ptr(),
                               table_dev.numel(), st)

    def read_tokens(self, layer, src, table_dev, start, n, lsc_block_off=0, stream=None):
        st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
        k = torch.empty((n, self.Hkv, self.D), dtype=torch.bfloat16, device=self.device)
        v = torch.empty_like(k)
        self.pool.read_tokens(layer, src, table_dev.data_ptr() if table_dev is not None else 0,
                              table_dev.numel() if table_dev is not None else 0, lsc_block_off, start, n,
                              k.data_ptr(), v.data_ptr(), st)
        return k, v
