"""ctypes face of oracle/bs_oracle_v2.c — wire format v2, structure-shared layers (TEST INFRASTRUCTURE ONLY;
argument marshalling, no arithmetic).  numpy arrays in, numpy arrays out."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

from .bs_oracle import OracleError

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bs_oracle_v2.c")
_LIBDIR = os.path.join(_HERE, "lib")
_SO = os.path.join(_LIBDIR, "libbsoracle_v2.so")
_lock = threading.Lock()
_lib = None

# 32-byte structure record and 16-byte layer record (re-typed here on purpose)
STRUCT_DTYPE = np.dtype([("rank", "<u4"), ("first_block", "<u4"), ("n_blocks", "<u4"), ("dq", "<i4", (2,)),
                         ("sign", "i1", (4,)), ("layer_bytes", "<u8")])
LAYER_DTYPE = np.dtype([("structure", "<u4"), ("tag", "<u4"), ("offset", "<u8")])
assert STRUCT_DTYPE.itemsize == 32 and LAYER_DTYPE.itemsize == 16


def build(force: bool = False) -> str:
    with _lock:
        stale = force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC)
        if stale:
            os.makedirs(_LIBDIR, exist_ok=True)
            tmp = _SO + f".{os.getpid()}.tmp"
            subprocess.run(["gcc", "-std=c99", "-O2", "-Wall", "-Wextra", "-shared", "-fPIC", _SRC, "-o", tmp],
                           check=True)
            os.replace(tmp, _SO)
    return _SO


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        u64, vp, u32 = C.c_uint64, C.c_void_p, C.c_uint32
        pu64 = C.POINTER(C.c_uint64)
        lib.orc2_header_bytes.restype = u64
        lib.orc2_header_bytes.argtypes = [u64, u64, u64]
        lib.orc2_plan.argtypes = [u64, u64, u64, vp, vp, vp, u32, vp, vp, vp, pu64, pu64]
        lib.orc2_serialized_size.argtypes = [u64, u64, u64, vp, vp, vp, u32, pu64, pu64]
        lib.orc2_serialize.argtypes = [u64, u64, u64, vp, vp, vp, vp, vp, u32, vp, u64, pu64]
        lib.orc2_stream_info.argtypes = [vp, u64, pu64, pu64, pu64, pu64, pu64]
        lib.orc2_stream_dtype.argtypes = [vp, u64, C.POINTER(u32)]
        lib.orc2_validate_stream.argtypes = [vp, u64]
        lib.orc2_counts.argtypes = [vp, u64, pu64, pu64]
        lib.orc2_deserialize.argtypes = [vp, u64, vp, vp, vp, vp, vp, vp, u64, u32]
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _args(structs, layers, dim):
    structs = np.ascontiguousarray(structs)
    layers = np.ascontiguousarray(layers)
    assert structs.dtype.itemsize == 32 and layers.dtype.itemsize == 16
    dim = np.ascontiguousarray(dim, dtype=np.uint32).reshape(-1, 3)
    return structs, layers, dim


def header_bytes(n_structs: int, n_layers: int, n_struct_blocks: int) -> int:
    return int(_L().orc2_header_bytes(n_structs, n_layers, n_struct_blocks))


def plan(structs, layers, dim, dtype: int = 0):
    """dict(rel_offset[Bs], layer_bytes[C], layer_offset[T], n_addr, payload_bytes).  dtype: 0 f64, 1 f32, 2 c64, 3 c128."""
    structs, layers, dim = _args(structs, layers, dim)
    Cn, Bs, T = len(structs), dim.shape[0], len(layers)
    rel = np.zeros(Bs, np.uint64)
    lb = np.zeros(Cn, np.uint64)
    lo = np.zeros(T, np.uint64)
    na, P = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc2_plan(Cn, Bs, T, _p(structs), _p(layers), _p(dim), dtype, _p(rel), _p(lb), _p(lo), C.byref(na), C.byref(P))
    if rc:
        raise OracleError(rc, "v2 plan")
    return dict(rel_offset=rel, layer_bytes=lb, layer_offset=lo, n_addr=int(na.value), payload_bytes=int(P.value))


def serialized_size(structs, layers, dim, dtype: int = 0):
    structs, layers, dim = _args(structs, layers, dim)
    hb, tot = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc2_serialized_size(len(structs), dim.shape[0], len(layers), _p(structs), _p(layers), _p(dim), dtype,
                                   C.byref(hb), C.byref(tot))
    if rc:
        raise OracleError(rc, "v2 serialized_size")
    return int(hb.value), int(tot.value)


def serialize(structs, layers, qn, dim, addr, capacity: int | None = None, out: np.ndarray | None = None,
              dtype: int = 0) -> np.ndarray:
    """The whole v2 stream.  ``addr``: HOST addresses of the blocks, layer-major.  dtype: the element type (reading E-2)."""
    structs, layers, dim = _args(structs, layers, dim)
    qn = np.ascontiguousarray(qn, dtype=np.int32).reshape(-1, 3, 2)
    addr = np.ascontiguousarray(addr, dtype=np.uint64)
    if capacity is None:
        capacity = serialized_size(structs, layers, dim, dtype)[1]
    if out is None:
        out = np.full(max(capacity, 1), 0xCD, dtype=np.uint8)
    written = C.c_uint64(0)
    rc = _L().orc2_serialize(len(structs), dim.shape[0], len(layers), _p(structs), _p(layers), _p(qn), _p(dim), _p(addr),
                             dtype, _p(out), capacity, C.byref(written))
    if rc:
        e = OracleError(rc, "v2 serialize")
        e.required = int(written.value)
        raise e
    return out[: int(written.value)]


def stream_info(stream: np.ndarray):
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    v = [C.c_uint64(0) for _ in range(5)]
    rc = _L().orc2_stream_info(_p(s), s.size, *[C.byref(x) for x in v])
    if rc:
        raise OracleError(rc, "v2 stream_info")
    dt = C.c_uint32(0)
    _L().orc2_stream_dtype(_p(s), s.size, C.byref(dt))
    return dict(n_structs=int(v[0].value), n_struct_blocks=int(v[1].value), n_layers=int(v[2].value),
                header_bytes=int(v[3].value), payload_bytes=int(v[4].value), dtype=int(dt.value))


def validate_stream(stream: np.ndarray) -> int:
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    return int(_L().orc2_validate_stream(_p(s), s.size))


def counts(stream: np.ndarray):
    """(n_addr, pool_bytes) of a v2 stream."""
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    na, pb = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc2_counts(_p(s), s.size, C.byref(na), C.byref(pb))
    if rc:
        raise OracleError(rc, "v2 counts")
    return int(na.value), int(pb.value)


def deserialize(stream: np.ndarray, pool: np.ndarray | None = None, scatter_addr=None, scatter_dim=None):
    """dict(structs, layers, qn, dim, addr, pool); pool layout unless scatter_* are given."""
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    info = stream_info(s)
    Cn, Bs, T = info["n_structs"], info["n_struct_blocks"], info["n_layers"]
    rc0 = validate_stream(s)
    if rc0:
        raise OracleError(rc0, "v2 deserialize")
    na, need = counts(s)
    structs = np.zeros(Cn, dtype=STRUCT_DTYPE)
    layers = np.zeros(T, dtype=LAYER_DTYPE)
    qn = np.zeros((Bs, 3, 2), np.int32)
    if scatter_addr is None:
        if pool is None:
            pool = np.full(max(need, 1), 0xEE, dtype=np.uint8)
        dim = np.zeros((Bs, 3), np.uint32)
        addr = np.zeros(na, np.uint64)
        flags = 0
    else:
        dim = np.ascontiguousarray(scatter_dim, dtype=np.uint32).reshape(-1, 3).copy()
        addr = np.ascontiguousarray(scatter_addr, dtype=np.uint64).copy()
        assert dim.shape[0] == Bs and addr.size == na
        flags = 1
        if pool is None:
            pool = np.zeros(1, np.uint8)
    rc = _L().orc2_deserialize(_p(s), s.size, _p(structs), _p(layers), _p(qn), _p(dim), _p(addr), _p(pool), pool.size, flags)
    if rc:
        raise OracleError(rc, "v2 deserialize")
    return dict(structs=structs, layers=layers, qn=qn, dim=dim, addr=addr, pool=pool)
