"""ctypes face of oracle/bs_oracle_pkg.c — self-contained packages (TEST INFRASTRUCTURE ONLY; marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

from .bs_oracle import OracleError

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bs_oracle_pkg.c")
_SO = os.path.join(_HERE, "lib", "libbsoracle_pkg.so")
_lock = threading.Lock()
_lib = None
PKG_HEADER = 64
NO_BLOCK = 0xFFFFFFFF


def build(force: bool = False) -> str:
    with _lock:
        if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
            os.makedirs(os.path.dirname(_SO), exist_ok=True)
            tmp = _SO + f".{os.getpid()}.tmp"
            subprocess.run(["gcc", "-std=c99", "-O2", "-Wall", "-Wextra", "-shared", "-fPIC", _SRC, "-o", tmp], check=True)
            os.replace(tmp, _SO)
    return _SO


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        u64, vp = C.c_uint64, C.c_void_p
        pu64 = C.POINTER(C.c_uint64)
        lib.orcp_count.restype = u64
        lib.orcp_count.argtypes = [u64, u64, u64]
        lib.orcp_range.argtypes = [u64, u64, u64, u64, pu64, pu64]
        lib.orcp_emit.argtypes = [vp, u64, u64, u64, u64, vp, u64, pu64]
        lib.orcp_assemble.argtypes = [vp, u64, u64, u64, vp, u64, pu64]
        _lib = lib
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def count(header_bytes: int, total_bytes: int, cap: int) -> int:
    return int(_L().orcp_count(header_bytes, total_bytes, cap))


def package_range(header_bytes: int, total_bytes: int, cap: int, index: int):
    lo, hi = C.c_uint64(0), C.c_uint64(0)
    rc = _L().orcp_range(header_bytes, total_bytes, cap, index, C.byref(lo), C.byref(hi))
    if rc:
        raise OracleError(rc, "pkg range")
    return int(lo.value), int(hi.value)


def emit(stream: np.ndarray, cap: int, stream_id: int, index: int) -> np.ndarray:
    """Package `index` (64-byte header + bytes) of a v1 stream."""
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    out = np.full(PKG_HEADER + cap, 0xCD, np.uint8)
    w = C.c_uint64(0)
    rc = _L().orcp_emit(_p(s), s.size, cap, stream_id, index, _p(out), out.size, C.byref(w))
    if rc:
        raise OracleError(rc, "pkg emit")
    return out[: int(w.value)]


def emit_slots(stream: np.ndarray, cap: int, stream_id: int, slot_bytes: int, slot_of=None, n_slots=None, poison=0x00):
    """All packages of a stream, package k written to slot slot_of[k] (identity by default)."""
    s = np.ascontiguousarray(stream, dtype=np.uint8)
    hb = int(np.frombuffer(s[48:56].tobytes(), "<u8")[0])
    n = count(hb, s.size, cap)
    if slot_of is None:
        slot_of = np.arange(n)
    if n_slots is None:
        n_slots = n
    slots = np.full((n_slots, slot_bytes), poison, np.uint8)
    for k in range(n):
        pk = emit(s, cap, stream_id, k)
        slots[int(slot_of[k]), : pk.size] = pk
    return slots


def assemble(slots: np.ndarray, stream_id: int, capacity: int | None = None) -> np.ndarray:
    slots = np.ascontiguousarray(slots, dtype=np.uint8)
    n_slots, slot_bytes = slots.shape
    if capacity is None:
        capacity = n_slots * slot_bytes
    out = np.full(max(capacity, 1), 0xCD, np.uint8)
    tot = C.c_uint64(0)
    rc = _L().orcp_assemble(_p(slots), slot_bytes, n_slots, stream_id, _p(out), capacity, C.byref(tot))
    if rc:
        e = OracleError(rc, "pkg assemble")
        e.required = int(tot.value)
        raise e
    return out[: int(tot.value)]
