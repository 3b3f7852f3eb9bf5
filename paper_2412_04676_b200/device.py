"""Device-memory plumbing with PyTorch: holds the descriptor arrays / workspace / result words as torch
tensors and hands raw pointers to the C ABI.  No data-path arithmetic here."""
from __future__ import annotations

import ctypes as C

import numpy as np
import torch

from . import _binding as B

_TENSOR_DTYPE = np.dtype([("rank", "<u4"), ("first_block", "<u4"), ("n_blocks", "<u4"), ("dq", "<i4", (2,)),
                          ("sign", "i1", (4,)), ("tag", "<u4"), ("reserved", "<u4")])


def current_stream(device=None) -> int:
    return int(torch.cuda.current_stream(device).cuda_stream)


def _to_dev(a: np.ndarray, device) -> torch.Tensor:
    a = np.ascontiguousarray(a)
    t = torch.from_numpy(a.view(np.uint8).reshape(-1).copy()) if a.size else torch.empty(0, dtype=torch.uint8)
    return t.to(device)


class DeviceSet:
    """The four device arrays of one bs_set_desc, as torch uint8 tensors."""

    def __init__(self, tensors: torch.Tensor, qn: torch.Tensor, dim: torch.Tensor, addr: torch.Tensor, n_tensors: int,
                 n_blocks: int, dtype: int = B.F64):
        self.tensors, self.qn, self.dim, self.addr = tensors, qn, dim, addr
        self.n_tensors, self.n_blocks, self.dtype = n_tensors, n_blocks, dtype

    @property
    def legs(self) -> int:
        """Legs per block of the qn / dim arrays: 4 for a BS_RANK4 set (wire format v3), else 3."""
        return 4 if self.dtype & B.RANK4 else 3

    @classmethod
    def from_host(cls, tensors: np.ndarray, qn: np.ndarray, dim: np.ndarray, addr: np.ndarray, device="cuda",
                  dtype: int = B.F64):
        assert tensors.dtype.itemsize == 32
        legs = 4 if dtype & B.RANK4 else 3
        return cls(_to_dev(tensors, device), _to_dev(qn.astype(np.int32, copy=False), device),
                   _to_dev(dim.astype(np.uint32, copy=False), device), _to_dev(addr.astype(np.uint64, copy=False), device),
                   len(tensors), int(np.asarray(dim).reshape(-1, legs).shape[0]), dtype)

    @classmethod
    def empty(cls, cap_tensors: int, cap_blocks: int, device="cuda", fill: int | None = None, rank4: bool = False):
        def mk(n):
            t = torch.empty(max(n, 16), dtype=torch.uint8, device=device)
            if fill is not None:
                t.fill_(fill)
            return t
        legs = 4 if rank4 else 3
        return cls(mk(32 * cap_tensors), mk(8 * legs * cap_blocks), mk(4 * legs * cap_blocks), mk(8 * cap_blocks), cap_tensors,
                   cap_blocks, B.RANK4 if rank4 else B.F64)

    @property
    def desc(self) -> B.SetDesc:
        return B.make_desc(self.n_tensors, self.n_blocks, self.tensors.data_ptr(), self.qn.data_ptr(), self.dim.data_ptr(),
                           self.addr.data_ptr(), self.dtype)

    def to_host(self, n_tensors: int | None = None, n_blocks: int | None = None) -> dict:
        T = self.n_tensors if n_tensors is None else n_tensors
        Bn = self.n_blocks if n_blocks is None else n_blocks
        return dict(
            tensors=self.tensors[: 32 * T].cpu().numpy().view(_TENSOR_DTYPE).copy(),
            qn=self.qn[: 8 * self.legs * Bn].cpu().numpy().view(np.int32).reshape(Bn, self.legs, 2).copy(),
            dim=self.dim[: 4 * self.legs * Bn].cpu().numpy().view(np.uint32).reshape(Bn, self.legs).copy(),
            addr=self.addr[: 8 * Bn].cpu().numpy().view(np.uint64).copy(),
        )


_STRUCT_DTYPE = np.dtype([("rank", "<u4"), ("first_block", "<u4"), ("n_blocks", "<u4"), ("dq", "<i4", (2,)),
                          ("sign", "i1", (4,)), ("layer_bytes", "<u8")])
_LAYER_DTYPE = np.dtype([("structure", "<u4"), ("tag", "<u4"), ("offset", "<u8")])


class DeviceLayeredSet:
    """The five device arrays of one bs_layered_desc (wire format v2), as torch uint8 tensors."""

    def __init__(self, structs, layers, qn, dim, addr, n_structs: int, n_struct_blocks: int, n_layers: int, n_addr: int,
                 dtype: int = B.F64):
        self.structs, self.layers, self.qn, self.dim, self.addr = structs, layers, qn, dim, addr
        self.n_structs, self.n_struct_blocks, self.n_layers, self.n_addr = n_structs, n_struct_blocks, n_layers, n_addr
        self.dtype = dtype

    @classmethod
    def from_host(cls, structs: np.ndarray, layers: np.ndarray, qn: np.ndarray, dim: np.ndarray, addr: np.ndarray,
                  device="cuda", dtype: int = B.F64):
        assert structs.dtype.itemsize == 32 and layers.dtype.itemsize == 16
        return cls(_to_dev(structs, device), _to_dev(layers, device), _to_dev(qn.astype(np.int32, copy=False), device),
                   _to_dev(dim.astype(np.uint32, copy=False), device), _to_dev(addr.astype(np.uint64, copy=False), device),
                   len(structs), int(np.asarray(dim).reshape(-1, 3).shape[0]), len(layers), int(np.asarray(addr).size), dtype)

    @classmethod
    def empty(cls, cap_structs: int, cap_struct_blocks: int, cap_layers: int, cap_addr: int, device="cuda",
              fill: int | None = None):
        def mk(n):
            t = torch.empty(max(n, 16), dtype=torch.uint8, device=device)
            if fill is not None:
                t.fill_(fill)
            return t
        return cls(mk(32 * cap_structs), mk(16 * cap_layers), mk(24 * cap_struct_blocks), mk(12 * cap_struct_blocks),
                   mk(8 * cap_addr), cap_structs, cap_struct_blocks, cap_layers, cap_addr)

    @property
    def desc(self) -> B.LayeredDesc:
        return B.make_layered_desc(self.n_structs, self.n_struct_blocks, self.n_layers, self.n_addr, self.structs.data_ptr(),
                                   self.layers.data_ptr(), self.qn.data_ptr(), self.dim.data_ptr(), self.addr.data_ptr(), self.dtype)

    def to_host(self, n_structs: int, n_struct_blocks: int, n_layers: int, n_addr: int) -> dict:
        return dict(
            structs=self.structs[: 32 * n_structs].cpu().numpy().view(_STRUCT_DTYPE).copy(),
            layers=self.layers[: 16 * n_layers].cpu().numpy().view(_LAYER_DTYPE).copy(),
            qn=self.qn[: 24 * n_struct_blocks].cpu().numpy().view(np.int32).reshape(n_struct_blocks, 3, 2).copy(),
            dim=self.dim[: 12 * n_struct_blocks].cpu().numpy().view(np.uint32).reshape(n_struct_blocks, 3).copy(),
            addr=self.addr[: 8 * n_addr].cpu().numpy().view(np.uint64).copy(),
        )


class Workspace:
    """Device workspace + the 64-byte bs_result word of one call site."""

    def __init__(self, n_tensors: int, n_blocks: int, stream_capacity: int, device="cuda", layered=None, packages=False):
        """layered = (n_structs, n_struct_blocks, n_layers, n_addr) sizes the workspace for wire format v2 instead;
        packages=True adds the room bs_package_unpack needs for the assembled header region."""
        if packages and layered is not None:
            self.nbytes = B.layered_package_workspace_bytes(*layered, stream_capacity)
        elif packages:
            self.nbytes = B.package_workspace_bytes(n_tensors, n_blocks, stream_capacity)
        elif layered is not None:
            self.nbytes = B.layered_workspace_bytes(*layered, stream_capacity)
        else:
            self.nbytes = B.workspace_bytes(n_tensors, n_blocks, stream_capacity)
        self.buf = torch.empty(self.nbytes, dtype=torch.uint8, device=device)
        self.result = torch.zeros(64, dtype=torch.uint8, device=device)
        assert self.buf.data_ptr() % 256 == 0

    @property
    def ptr(self) -> int:
        return self.buf.data_ptr()

    @property
    def result_ptr(self) -> int:
        return self.result.data_ptr()

    def read_result(self) -> dict:
        """Synchronising read of the deferred outcome."""
        raw = self.result.cpu().numpy().tobytes()
        r = B.Result.from_buffer_copy(raw)
        return dict(total_bytes=int(r.total_bytes), header_bytes=int(r.header_bytes), payload_bytes=int(r.payload_bytes),
                    pool_bytes=int(r.pool_bytes), status=int(r.status), n_tensors=int(r.n_tensors), n_blocks=int(r.n_blocks),
                    n_structs=int(r.reserved[0]), n_struct_blocks=int(r.reserved[1]), dtype=int(r.reserved[2]),
                    n_packages=int(r.reserved[3]))
