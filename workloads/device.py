"""Device side of the harness: seeded fill of the source pool on the GPU (bit-identical to values.py) and the
stand-in contraction that keeps the compute stream busy in the offload-overlap measurement (config 5).
Harness only — the product never imports this."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "csrc", "bsworkload.cu")
_LIBDIR = os.path.join(_HERE, "lib")
_SO = os.path.join(_LIBDIR, "libbsworkload.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        os.makedirs(_LIBDIR, exist_ok=True)
        tmp = _SO + f".{os.getpid()}.tmp"
        nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
        subprocess.run([nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                        "-Xcompiler", "-fPIC", "-cudart", "static", "-shared", _SRC, "-o", tmp], check=True)
        os.replace(tmp, _SO)
    return _SO


def _L():
    global _lib
    if _lib is None:
        so = _SO
        if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            so = build()
        lib = C.CDLL(so)
        lib.wl_fill_blocks.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
        lib.wl_contract.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]
        lib.wl_memcpy_each.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
        _lib = lib
    return _lib


def fill_pool_device(bset, device="cuda", pool=None):
    """Allocate (or reuse) the source pool on the device and fill every block with its seeded values.
    Returns (pool uint8 tensor, addr numpy uint64 device addresses)."""
    import torch

    if pool is None:
        pool = torch.zeros(max(int(bset.pool_bytes), 16), dtype=torch.uint8, device=device)
    addr = (np.uint64(pool.data_ptr()) + bset.pool_off).astype(np.uint64)
    d_addr = torch.from_numpy(addr.view(np.int64)).to(device)
    d_nel = torch.from_numpy(bset.nelems.astype(np.uint64).view(np.int64)).to(device)
    rc = _L().wl_fill_blocks(d_addr.data_ptr(), d_nel.data_ptr(), 0, bset.n_blocks, bset.seed,
                             torch.cuda.current_stream().cuda_stream)
    if rc:
        raise RuntimeError(f"wl_fill_blocks: cudaError {rc}")
    torch.cuda.current_stream().synchronize()
    return pool, addr


class StandInContraction:
    """Batched fp64 block GEMMs C_i = A_i * M_i on the sector shapes of the set (SURVEY §8(d) config-5 protocol):
    A_i = block i (d_l x d_r), M_i = a d_r x d_r matrix, C_i = scratch.  Harness load, efficiency irrelevant."""

    def __init__(self, bset, addr: np.ndarray, device="cuda", max_items: int | None = None, seed: int = 99):
        import torch

        dim = bset.dim.astype(np.int64)
        m = dim[:, 0]
        n = dim[:, 1] * dim[:, 2]
        sel = np.nonzero((m > 0) & (n > 0))[0]
        if max_items is not None:
            sel = sel[:max_items]
        nmax = int(n[sel].max()) if len(sel) else 1
        cmax = int((m[sel] * n[sel]).max()) if len(sel) else 1
        self.mat = torch.rand(nmax * nmax, dtype=torch.float64, device=device)
        self.out = torch.zeros(cmax * 8, dtype=torch.float64, device=device)
        items = np.zeros(len(sel), dtype=[("a", "<u8"), ("b", "<u8"), ("c", "<u8"), ("m", "<u4"), ("n", "<u4"),
                                          ("k", "<u4"), ("pad", "<u4")])
        items["a"] = addr[sel]
        items["b"] = self.mat.data_ptr()
        items["c"] = self.out.data_ptr() + (np.arange(len(sel)) % 8) * cmax * 8
        items["m"], items["n"], items["k"] = m[sel], n[sel], n[sel]
        self.items = torch.from_numpy(items.view(np.uint8).reshape(-1).copy()).to(device)
        self.n_items = len(sel)
        self.flops = float(2 * (m[sel] * n[sel] * n[sel]).sum())

    def run(self, reps: int = 1, stream: int | None = None, grid: int = 0):
        import torch

        s = torch.cuda.current_stream().cuda_stream if stream is None else stream
        for _ in range(reps):
            rc = _L().wl_contract(self.items.data_ptr(), self.n_items, grid, s)
            if rc:
                raise RuntimeError(f"wl_contract: cudaError {rc}")


def memcpy_each(dsts: np.ndarray, srcs: np.ndarray, sizes: np.ndarray, stream: int) -> None:
    """One cudaMemcpyAsync (device to device) per entry of the host arrays of device pointers / sizes (uint64): the
    library comparator of the pack step."""
    dsts, srcs, sizes = (np.ascontiguousarray(a, dtype=np.uint64) for a in (dsts, srcs, sizes))
    rc = _L().wl_memcpy_each(dsts.ctypes.data, srcs.ctypes.data, sizes.ctypes.data, len(sizes), stream)
    if rc:
        raise RuntimeError(f"cudaMemcpyAsync: cudaError {rc}")
