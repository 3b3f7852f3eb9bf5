"""ctypes face of oracle/bs_oracle_v3.c — wire format v3, tensors of rank 2, 3 or 4 (TEST INFRASTRUCTURE ONLY; argument
marshalling, no arithmetic).  numpy arrays in, numpy arrays out."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

from .bs_oracle import TENSOR_DTYPE, OracleError

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bs_oracle_v3.c")
_LIBDIR = os.path.join(_HERE, "lib")
_SO = os.path.join(_LIBDIR, "libbsoracle_v3.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    with _lock:
        stale = force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC)
        if stale:
            os.makedirs(_LIBDIR, exist_ok=True)
            tmp = _SO + f".{os.getpid()}.tmp"
            subprocess.run(["gcc", "-std=c99", "-O2", "-Wall", "-Wextra", "-shared", "-fPIC", _SRC, "-o", tmp], check=True)
            os.replace(tmp, _SO)
    return _SO


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        u64, vp, u32 = C.c_uint64, C.c_void_p, C.c_uint32
        pu64, pu32 = C.POINTER(C.c_uint64), C.POINTER(C.c_uint32)
        lib.orc3_header_bytes.restype = u64
        lib.orc3_header_bytes.argtypes = [u64, u64]
        lib.orc3_plan.argtypes = [u64, vp, u32, vp, vp, vp, pu64]
        lib.orc3_serialized_size.argtypes = [u64, u64, vp, u32, pu64, pu64]
        lib.orc3_serialize.argtypes = [u64, u64, vp, vp, vp, vp, u32, vp, u64, pu64]
        lib.orc3_stream_info.argtypes = [vp, u64, pu64, pu64, pu64, pu64, pu32]
        lib.orc3_validate_stream.argtypes = [vp, u64]
        lib.orc3_pool_bytes.argtypes = [vp, u64, pu64]
        lib.orc3_deserialize.argtypes = [vp, u64, vp, vp, vp, vp, vp, u64, u32]
        lib.orc3_validate_set.argtypes = [u64, u64, vp, vp]
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dim(dim):
    return np.ascontiguousarray(dim, dtype=np.uint32).reshape(-1, 4)


def _tensors(t):
    t = np.ascontiguousarray(t)
    assert t.dtype.itemsize == 32
    return t


def header_bytes(T: int, B: int) -> int:
    return int(_L().orc3_header_bytes(T, B))


def plan(dim, dtype: int = 0):
    dim = _dim(dim)
    B = dim.shape[0]
    nbytes, stored, offset = np.zeros(B, np.uint64), np.zeros(B, np.uint64), np.zeros(B, np.uint64)
    P = C.c_uint64(0)
    rc = _L().orc3_plan(B, _p(dim), dtype, _p(nbytes), _p(stored), _p(offset), C.byref(P))
    if rc:
        raise OracleError(rc, "v3 plan")
    return nbytes, stored, offset, int(P.value)


def serialized_size(n_tensors: int, dim, dtype: int = 0):
    dim = _dim(dim)
    hb, tot = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc3_serialized_size(n_tensors, dim.shape[0], _p(dim), dtype, C.byref(hb), C.byref(tot))
    if rc:
        raise OracleError(rc, "v3 serialized_size")
    return int(hb.value), int(tot.value)


def serialize(tensors, qn, dim, addr, dtype: int = 0, capacity: int | None = None, out: np.ndarray | None = None) -> np.ndarray:
    """The whole v3 stream.  qn [B][4][2], dim [B][4]; ``addr``: HOST addresses of the dense row-major blocks."""
    tensors, dim = _tensors(tensors), _dim(dim)
    qn = np.ascontiguousarray(qn, dtype=np.int32).reshape(-1, 4, 2)
    addr = np.ascontiguousarray(addr, dtype=np.uint64)
    T, B = len(tensors), dim.shape[0]
    if capacity is None:
        capacity = serialized_size(T, dim, dtype)[1]
    if out is None:
        out = np.full(max(capacity, 1), 0xCD, dtype=np.uint8)
    written = C.c_uint64(0)
    rc = _L().orc3_serialize(T, B, _p(tensors), _p(qn), _p(dim), _p(addr), dtype, _p(out), capacity, C.byref(written))
    if rc:
        e = OracleError(rc, "v3 serialize")
        e.required = int(written.value)
        raise e
    return out[: int(written.value)]


def stream_info(stream: np.ndarray):
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    T, B, hb, P, dt = C.c_uint64(0), C.c_uint64(0), C.c_uint64(0), C.c_uint64(0), C.c_uint32(0)
    rc = _L().orc3_stream_info(_p(s), s.size, C.byref(T), C.byref(B), C.byref(hb), C.byref(P), C.byref(dt))
    if rc:
        raise OracleError(rc, "v3 stream_info")
    return dict(n_tensors=int(T.value), n_blocks=int(B.value), header_bytes=int(hb.value), payload_bytes=int(P.value),
                dtype=int(dt.value))


def validate_stream(stream: np.ndarray) -> int:
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    return int(_L().orc3_validate_stream(_p(s), s.size))


def pool_bytes(stream: np.ndarray) -> int:
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    n = C.c_uint64(0)
    rc = _L().orc3_pool_bytes(_p(s), s.size, C.byref(n))
    if rc:
        raise OracleError(rc, "v3 pool_bytes")
    return int(n.value)


def deserialize(stream: np.ndarray, pool: np.ndarray | None = None, scatter_addr=None, scatter_dim=None):
    """dict(tensors, qn [B][4][2], dim [B][4], addr, pool); pool layout unless scatter_* are given."""
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    info = stream_info(s)
    T, B = info["n_tensors"], info["n_blocks"]
    tensors = np.zeros(T, dtype=TENSOR_DTYPE)
    qn = np.zeros((B, 4, 2), np.int32)
    if scatter_addr is None:
        rc0 = validate_stream(s)
        if rc0:
            raise OracleError(rc0, "v3 deserialize")
        need = pool_bytes(s)
        if pool is None:
            pool = np.full(max(need, 1), 0xEE, dtype=np.uint8)
        dim = np.zeros((B, 4), np.uint32)
        addr = np.zeros(B, np.uint64)
        flags = 0
    else:
        dim = _dim(scatter_dim).copy()
        addr = np.ascontiguousarray(scatter_addr, dtype=np.uint64).copy()
        flags = 1
        if pool is None:
            pool = np.zeros(1, np.uint8)
    rc = _L().orc3_deserialize(_p(s), s.size, _p(tensors), _p(qn), _p(dim), _p(addr), _p(pool), pool.size, flags)
    if rc:
        raise OracleError(rc, "v3 deserialize")
    return dict(tensors=tensors, qn=qn, dim=dim, addr=addr, pool=pool, dtype=info["dtype"])


def validate_set(tensors, qn) -> int:
    tensors = _tensors(tensors)
    qn = np.ascontiguousarray(qn, dtype=np.int32).reshape(-1, 4, 2)
    return int(_L().orc3_validate_set(len(tensors), qn.shape[0], _p(tensors), _p(qn)))
