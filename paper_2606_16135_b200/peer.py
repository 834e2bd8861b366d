"""Lending a pool region from one process to another through CUDA IPC.

In the paper the donor of the pool is ANOTHER model's GPU: "stored on a worker GPU ... preloads
... into the LSC of the master GPU" over NVLink.  With one process per
GPU the worker process allocates the region on its device and exports a handle; the master
process opens the handle and passes the mapped pointer to sc_pool_create as pool_base with
pool_kind = SC_POOL_PEER.  The library never sees the handle, only the pointer.

Plumbing only (allocation and address mapping through the CUDA runtime, via cuda-python): no
step of the method runs here.  The region comes from cudaMalloc DIRECTLY, not from a torch
tensor: an IPC handle names a whole cudaMalloc allocation and opens at that allocation's base,
whereas a tensor of torch's caching allocator may sit anywhere inside a larger segment -- the
opener would then write the pool over the lender's other tensors.
"""
from __future__ import annotations

try:                                     # cuda-python >= 12.8 names it cuda.bindings.runtime
    from cuda.bindings import runtime as cudart
except ImportError:                      # pragma: no cover - older cuda-python
    from cuda import cudart

ALIGN = 1024                             # sc_pool_create wants pool_base 1024-byte aligned


def _ok(err, what: str) -> None:
    if int(err) != 0:
        raise RuntimeError(f"{what}: {cudart.cudaGetErrorString(err)[1].decode()} ({int(err)})")


class LentRegion:
    """Owner side: `nbytes` usable bytes of device memory on the CURRENT device, starting at a
    1024-byte aligned address, plus what another process needs to map them (`ticket()`)."""

    def __init__(self, nbytes: int, device: int | None = None):
        self.nbytes = int(nbytes)
        if device is not None:
            _ok(cudart.cudaSetDevice(int(device))[0], "cudaSetDevice")
        err, base = cudart.cudaMalloc(self.nbytes + ALIGN)
        _ok(err, "cudaMalloc(lent pool region)")
        self.base = int(base)
        self.offset = (-self.base) % ALIGN          # from the allocation base to the region
        self.ptr = self.base + self.offset
        err, handle = cudart.cudaIpcGetMemHandle(self.base)
        if int(err) != 0:
            cudart.cudaFree(self.base)
            _ok(err, "cudaIpcGetMemHandle")
        self._handle = bytes(handle.reserved)

    def ticket(self) -> tuple:
        """Picklable: (handle bytes, offset of the region from the allocation base, usable bytes)."""
        return (self._handle, self.offset, self.nbytes)

    def fill(self, byte: int) -> None:
        """Synchronous memset of the usable bytes (tests: what the lent memory held before)."""
        _ok(cudart.cudaMemset(self.ptr, int(byte), self.nbytes)[0], "cudaMemset")
        _ok(cudart.cudaDeviceSynchronize()[0], "cudaDeviceSynchronize")

    def to_host(self):
        """The usable bytes as a numpy uint8 array (synchronous copy)."""
        import numpy as np
        host = np.empty(self.nbytes, dtype=np.uint8)
        _ok(cudart.cudaMemcpy(host.ctypes.data, self.ptr, self.nbytes,
                              cudart.cudaMemcpyKind.cudaMemcpyDeviceToHost)[0], "cudaMemcpy(D2H)")
        return host

    def free(self) -> None:
        """Only after every opener has closed its mapping."""
        if self.base:
            _ok(cudart.cudaFree(self.base)[0], "cudaFree(lent pool region)")
            self.base = self.ptr = 0


class OpenedRegion:
    """Borrower side: maps a ticket on the CURRENT device.  `ptr` is valid there (peer access is
    enabled lazily by the runtime when the lender is another GPU) and addresses the same bytes as
    the lender's `ptr`."""

    def __init__(self, ticket: tuple, need_bytes: int = 0, device: int | None = None):
        raw, offset, nbytes = ticket
        if need_bytes > nbytes:
            raise ValueError(f"lent region holds {nbytes} bytes, the pool needs {need_bytes}")
        if device is not None:
            _ok(cudart.cudaSetDevice(int(device))[0], "cudaSetDevice")
        h = cudart.cudaIpcMemHandle_t()
        h.reserved = raw
        err, base = cudart.cudaIpcOpenMemHandle(h, cudart.cudaIpcMemLazyEnablePeerAccess)
        _ok(err, "cudaIpcOpenMemHandle (is there a P2P path between the two GPUs?)")
        self.base = int(base)
        self.ptr = self.base + int(offset)
        self.nbytes = int(nbytes)
        if self.ptr % ALIGN:
            # the mapping's base is congruent to the lender's modulo 1024 on every driver seen so
            # far (both are at least 2 MiB-granular); if not, say so instead of mis-addressing
            self.close()
            raise RuntimeError(f"mapped base {self.base:#x} + offset {offset} is not {ALIGN}-byte aligned")

    def close(self) -> None:
        if self.base:
            _ok(cudart.cudaIpcCloseMemHandle(self.base)[0], "cudaIpcCloseMemHandle")
            self.base = self.ptr = 0
