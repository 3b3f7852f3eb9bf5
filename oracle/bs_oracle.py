"""ctypes face of oracle/bs_oracle.c (TEST INFRASTRUCTURE ONLY — argument marshalling, no arithmetic).

numpy arrays in, numpy arrays out.  ``build()`` compiles the C file with the box's gcc (-O2, one
thread, no SIMD flags) into oracle/lib/libbsoracle.so; the library is rebuilt when the source is newer.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

OK, ERR_ARG, ERR_CAPACITY, ERR_CORRUPT, ERR_UNSUPPORTED = 0, -1, -2, -3, -4

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bs_oracle.c")
_LIBDIR = os.path.join(_HERE, "lib")
_SO = os.path.join(_LIBDIR, "libbsoracle.so")
_lock = threading.Lock()
_lib = None

# same 32-byte layout as the descriptor's tensor record (re-typed here on purpose)
TENSOR_DTYPE = np.dtype(
    [("rank", "<u4"), ("first_block", "<u4"), ("n_blocks", "<u4"), ("dq", "<i4", (2,)),
     ("sign", "i1", (4,)), ("tag", "<u4"), ("reserved", "<u4")]
)


class OracleError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"oracle {what}: error {code}")
        self.code = code


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than the source."""
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
        lib.orc_header_bytes.restype = u64
        lib.orc_header_bytes.argtypes = [u64, u64]
        lib.orc_plan_al.argtypes = [u64, vp, u32, vp, vp, vp, pu64]
        lib.orc_serialized_size_al.argtypes = [u64, u64, vp, u32, pu64, pu64]
        lib.orc_emit_header_al.argtypes = [u64, u64, vp, vp, vp, u32, vp, u64]
        lib.orc_emit_payload_range_al.argtypes = [u64, u64, vp, vp, vp, u32, u64, u64, vp, u64, pu64, pu64]
        lib.orc_serialize_al.argtypes = [u64, u64, vp, vp, vp, vp, u32, vp, u64, pu64]
        lib.orc_stream_align.argtypes = [vp, u64, C.POINTER(u32)]
        lib.orc_stream_info.argtypes = [vp, u64, pu64, pu64, pu64, pu64]
        lib.orc_validate_stream.argtypes = [vp, u64]
        lib.orc_pool_bytes.argtypes = [vp, u64, pu64]
        lib.orc_deserialize.argtypes = [vp, u64, vp, vp, vp, vp, vp, u64, u32]
        lib.orc_validate_set.argtypes = [u64, u64, vp, vp]
        assert lib.orc_selftest_endian() == 1, "oracle assumes a little-endian host"
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _c(a, dtype, shape_tail=None):
    a = np.ascontiguousarray(a, dtype=dtype)
    if shape_tail is not None:
        a = a.reshape((-1,) + shape_tail)
    return a


def _tensors(t):
    t = np.ascontiguousarray(t)
    assert t.dtype.itemsize == 32
    return t


def header_bytes(T: int, B: int) -> int:
    return int(_L().orc_header_bytes(T, B))


def plan(dim, align: int = 16):
    """(nbytes, stored, offset, payload_bytes) of SURVEY §8(c) serialize step 2.  align: 16, or 8 (reading D19: unpadded)."""
    dim = _c(dim, np.uint32, (3,))
    B = dim.shape[0]
    nbytes = np.zeros(B, np.uint64)
    stored = np.zeros(B, np.uint64)
    offset = np.zeros(B, np.uint64)
    P = C.c_uint64(0)
    rc = _L().orc_plan_al(B, _p(dim), align, _p(nbytes), _p(stored), _p(offset), C.byref(P))
    if rc:
        raise OracleError(rc, "plan")
    return nbytes, stored, offset, int(P.value)


def serialized_size(n_tensors: int, dim, align: int = 16):
    dim = _c(dim, np.uint32, (3,))
    hb, tot = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc_serialized_size_al(n_tensors, dim.shape[0], _p(dim), align, C.byref(hb), C.byref(tot))
    if rc:
        raise OracleError(rc, "serialized_size")
    return int(hb.value), int(tot.value)


def emit_header(tensors, qn, dim, align: int = 16) -> np.ndarray:
    tensors, qn, dim = _tensors(tensors), _c(qn, np.int32, (3, 2)), _c(dim, np.uint32, (3,))
    T, B = len(tensors), dim.shape[0]
    out = np.full(header_bytes(T, B), 0xCD, dtype=np.uint8)   # poisoned: every byte must be written
    rc = _L().orc_emit_header_al(T, B, _p(tensors), _p(qn), _p(dim), align, _p(out), out.size)
    if rc:
        raise OracleError(rc, "emit_header")
    return out


def emit_payload_range(tensors, dim, addr, t0: int, t1: int, capacity: int, out: np.ndarray | None = None, align: int = 16):
    """Payload bytes of tensors [t0, t1).  Returns (first_offset, bytes ndarray).  ``out``: a caller buffer of at least
    ``capacity`` bytes to write into (e.g. a slice of one large stream buffer) instead of a fresh poisoned one."""
    tensors, dim = _tensors(tensors), _c(dim, np.uint32, (3,))
    addr = _c(addr, np.uint64)
    if out is None:
        out = np.full(max(capacity, 1), 0xCD, dtype=np.uint8)
    assert out.dtype == np.uint8 and out.flags["C_CONTIGUOUS"] and out.size >= capacity
    first, nb = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc_emit_payload_range_al(len(tensors), dim.shape[0], _p(tensors), _p(dim), _p(addr), align, t0, t1,
                                        _p(out), capacity, C.byref(first), C.byref(nb))
    if rc:
        raise OracleError(rc, "emit_payload_range")
    return int(first.value), out[: int(nb.value)]


def serialize(tensors, qn, dim, addr, capacity: int | None = None, out: np.ndarray | None = None, align: int = 16) -> np.ndarray:
    """The whole stream.  ``addr`` holds HOST addresses (uint64) of the dense row-major blocks.  align: 16 or 8 (D19)."""
    tensors, qn, dim = _tensors(tensors), _c(qn, np.int32, (3, 2)), _c(dim, np.uint32, (3,))
    addr = _c(addr, np.uint64)
    T, B = len(tensors), dim.shape[0]
    if capacity is None:
        capacity = serialized_size(T, dim, align)[1]
    if out is None:
        out = np.full(max(capacity, 1), 0xCD, dtype=np.uint8)
    written = C.c_uint64(0)
    rc = _L().orc_serialize_al(T, B, _p(tensors), _p(qn), _p(dim), _p(addr), align, _p(out), capacity, C.byref(written))
    if rc:
        e = OracleError(rc, "serialize")
        e.required = int(written.value)
        raise e
    return out[: int(written.value)]


def stream_info(stream: np.ndarray):
    s = _c(stream, np.uint8)
    T, B, hb, P = C.c_uint64(0), C.c_uint64(0), C.c_uint64(0), C.c_uint64(0)
    rc = _L().orc_stream_info(_p(s), s.size, C.byref(T), C.byref(B), C.byref(hb), C.byref(P))
    if rc:
        raise OracleError(rc, "stream_info")
    al = C.c_uint32(0)
    _L().orc_stream_align(_p(s), s.size, C.byref(al))
    return dict(n_tensors=int(T.value), n_blocks=int(B.value), header_bytes=int(hb.value),
                payload_bytes=int(P.value), align=int(al.value))


def validate_stream(stream: np.ndarray) -> int:
    s = _c(stream, np.uint8)
    return int(_L().orc_validate_stream(_p(s), s.size))


def pool_bytes(stream: np.ndarray) -> int:
    s = _c(stream, np.uint8)
    n = C.c_uint64(0)
    rc = _L().orc_pool_bytes(_p(s), s.size, C.byref(n))
    if rc:
        raise OracleError(rc, "pool_bytes")
    return int(n.value)


def deserialize(stream: np.ndarray, pool: np.ndarray | None = None, scatter_addr=None, scatter_dim=None):
    """Returns dict(tensors, qn, dim, addr, pool).  addr = host addresses; pool layout unless scatter_*."""
    s = _c(stream, np.uint8)
    info = stream_info(s)
    T, B = info["n_tensors"], info["n_blocks"]
    tensors = np.zeros(T, dtype=TENSOR_DTYPE)
    qn = np.zeros((B, 3, 2), np.int32)
    if scatter_addr is None:
        rc0 = validate_stream(s)
        if rc0:
            raise OracleError(rc0, "deserialize")
        need = pool_bytes(s)
        if pool is None:
            pool = np.full(max(need, 1), 0xEE, dtype=np.uint8)
        dim = np.zeros((B, 3), np.uint32)
        addr = np.zeros(B, np.uint64)
        flags = 0
    else:
        dim = _c(scatter_dim, np.uint32, (3,)).copy()
        addr = _c(scatter_addr, np.uint64).copy()
        flags = 1
        if pool is None:
            pool = np.zeros(1, np.uint8)
    rc = _L().orc_deserialize(_p(s), s.size, _p(tensors), _p(qn), _p(dim), _p(addr), _p(pool), pool.size, flags)
    if rc:
        raise OracleError(rc, "deserialize")
    return dict(tensors=tensors, qn=qn, dim=dim, addr=addr, pool=pool)


def validate_set(tensors, qn) -> int:
    tensors, qn = _tensors(tensors), _c(qn, np.int32, (3, 2))
    return int(_L().orc_validate_set(len(tensors), qn.shape[0], _p(tensors), _p(qn)))
