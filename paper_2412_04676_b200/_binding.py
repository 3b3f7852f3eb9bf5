"""ctypes binding of libbsstream.so (include/bs.h).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels.  There is no CPU fallback — if the shared library cannot be
loaded this module raises, and every device call fails with BS_ERR_CUDA on a box without a GPU."""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

OK, PENDING = 0, 1
ERR_ARG, ERR_CAPACITY, ERR_CORRUPT, ERR_UNSUPPORTED, ERR_CUDA, ERR_IO = -1, -2, -3, -4, -5, -6
F64, F32, C64, C128 = 0, 1, 2, 3
ALIGN8 = 0x100   # OR-ed into a set's dtype: serialize an unpadded stream (bs.h BS_ALIGN8)
RANK4 = 0x200    # OR-ed into a set's dtype: qn / dim have four legs per block, wire format v3 (bs.h BS_RANK4)
LAYOUT_POOL, SCATTER_TO_ADDR = 0, 1
VARIANT_DEFAULT, VARIANT_LDG, VARIANT_TMA = 0, 1, 2


class BsError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {strerror(code)} ({code})" + (f", cudaError {last_cuda_error()}" if code == ERR_CUDA else ""))
        self.code = code


class TensorRec(C.Structure):
    _fields_ = [("rank", C.c_uint32), ("first_block", C.c_uint32), ("n_blocks", C.c_uint32), ("dq", C.c_int32 * 2),
                ("sign", C.c_int8 * 4), ("tag", C.c_uint32), ("reserved", C.c_uint32)]


class SetDesc(C.Structure):
    _fields_ = [("n_tensors", C.c_uint32), ("n_blocks", C.c_uint32), ("n_qn", C.c_uint32), ("dtype", C.c_uint32),
                ("tensors", C.c_void_p), ("qn", C.c_void_p), ("dim", C.c_void_p), ("addr", C.c_void_p)]


class StructRec(C.Structure):
    _fields_ = [("rank", C.c_uint32), ("first_block", C.c_uint32), ("n_blocks", C.c_uint32), ("dq", C.c_int32 * 2),
                ("sign", C.c_int8 * 4), ("layer_bytes", C.c_uint64)]


class LayerRec(C.Structure):
    _fields_ = [("structure", C.c_uint32), ("tag", C.c_uint32), ("offset", C.c_uint64)]


class LayeredDesc(C.Structure):
    _fields_ = [("n_structs", C.c_uint32), ("n_struct_blocks", C.c_uint32), ("n_layers", C.c_uint32), ("n_qn", C.c_uint32),
                ("dtype", C.c_uint32), ("reserved", C.c_uint32), ("n_addr", C.c_uint64), ("structs", C.c_void_p),
                ("layers", C.c_void_p), ("qn", C.c_void_p), ("dim", C.c_void_p), ("addr", C.c_void_p)]


class LayeredStreamInfo(C.Structure):
    _fields_ = [("n_structs", C.c_uint64), ("n_struct_blocks", C.c_uint64), ("n_layers", C.c_uint64),
                ("header_bytes", C.c_uint64), ("payload_bytes", C.c_uint64), ("total_bytes", C.c_uint64),
                ("dtype", C.c_uint64)]


class Result(C.Structure):
    _fields_ = [("total_bytes", C.c_uint64), ("header_bytes", C.c_uint64), ("payload_bytes", C.c_uint64),
                ("pool_bytes", C.c_uint64), ("status", C.c_int32), ("n_tensors", C.c_uint32), ("n_blocks", C.c_uint32),
                ("reserved", C.c_uint32 * 5)]


class StreamInfo(C.Structure):
    _fields_ = [("n_tensors", C.c_uint64), ("n_blocks", C.c_uint64), ("header_bytes", C.c_uint64),
                ("payload_bytes", C.c_uint64), ("total_bytes", C.c_uint64), ("dtype", C.c_uint64), ("align", C.c_uint64),
                ("max_rank", C.c_uint64)]


class Opts(C.Structure):
    _fields_ = [("variant", C.c_uint32), ("tile_bytes", C.c_uint32), ("ctas_per_sm", C.c_uint32), ("stages", C.c_uint32),
                ("warps", C.c_uint32), ("tune", C.c_uint32), ("fuse", C.c_uint32), ("pace", C.c_uint32)]


def make_opts(opts) -> "Opts":
    """dict / Opts / None -> Opts (zeros = library defaults)."""
    if isinstance(opts, Opts):
        return opts
    o = Opts()
    for k in ("variant", "tile_bytes", "ctas_per_sm", "stages", "warps", "tune", "fuse", "pace"):
        setattr(o, k, int((opts or {}).get(k, 0) or 0))
    return o


class EngineCfg(C.Structure):
    _fields_ = [("chunk_bytes", C.c_uint64), ("n_staging", C.c_uint32), ("max_tensors", C.c_uint32),
                ("max_blocks", C.c_uint32), ("max_stream_bytes", C.c_uint64), ("opts", Opts)]


class TicketStats(C.Structure):
    _fields_ = [("bytes", C.c_uint64), ("n_chunks", C.c_uint32), ("status", C.c_int32), ("dma_ms", C.c_float),
                ("total_ms", C.c_float)]


class QueueStats(C.Structure):
    _fields_ = [("saves", C.c_uint64), ("loads", C.c_uint64), ("bytes_saved", C.c_uint64), ("bytes_loaded", C.c_uint64),
                ("host_bytes_live", C.c_uint64), ("host_bytes_peak", C.c_uint64), ("keys_live", C.c_uint64),
                ("device_bytes", C.c_uint64), ("in_flight", C.c_uint32), ("max_in_flight", C.c_uint32),
                ("bytes_spilled", C.c_uint64), ("bytes_filled", C.c_uint64)]


assert C.sizeof(TensorRec) == 32 and C.sizeof(Result) == 64 and C.sizeof(StructRec) == 32 and C.sizeof(LayerRec) == 16

_lib = None


def lib():
    """Load libbsstream.so, building it in-tree first if it is missing or stale (nvcc, sm_100a)."""
    global _lib
    if _lib is not None:
        return _lib
    so = _build.SO
    if _build.is_stale():
        try:
            so = _build.build()
        except Exception as e:  # no nvcc on this box and no prebuilt library: fail loudly
            if not os.path.exists(so):
                raise ImportError(f"libbsstream.so is not built and cannot be built here: {e}") from e
    L = C.CDLL(so)
    u32, u64, vp, i32 = C.c_uint32, C.c_uint64, C.c_void_p, C.c_int
    pu64 = C.POINTER(C.c_uint64)
    L.bs_version.restype = u32
    L.bs_strerror.restype = C.c_char_p
    L.bs_strerror.argtypes = [i32]
    L.bs_last_cuda_error.restype = i32
    L.bs_header_bytes.restype = u64
    L.bs_header_bytes.argtypes = [u64, u64]
    L.bs_header_bytes_rank4.restype = u64
    L.bs_header_bytes_rank4.argtypes = [u64, u64]
    L.bs_workspace_bytes.restype = u64
    L.bs_workspace_bytes.argtypes = [u32, u32, u64]
    L.bs_stream_info.argtypes = [vp, C.POINTER(StreamInfo)]
    L.bs_serialized_size.argtypes = [C.POINTER(SetDesc), vp, u64, pu64, pu64, vp]
    L.bs_serialize.argtypes = [C.POINTER(SetDesc), vp, u64, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_serialize_range.argtypes = [C.POINTER(SetDesc), vp, u64, u64, i32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_noalloc_scratch_bytes.restype = u64
    L.bs_noalloc_scratch_bytes.argtypes = []
    L.bs_serialize_noalloc.argtypes = [C.POINTER(SetDesc), vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_deserialize.argtypes = [vp, u64, C.POINTER(SetDesc), vp, u64, u32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_deserialize_range.argtypes = [vp, u64, u64, vp, C.POINTER(SetDesc), u32, vp, u64, C.POINTER(Opts), vp]
    L.bs_engine_create.argtypes = [C.POINTER(vp), C.POINTER(EngineCfg)]
    L.bs_engine_destroy.argtypes = [vp]
    L.bs_offload_async.argtypes = [vp, C.POINTER(SetDesc), u64, vp, u64, vp, C.POINTER(vp)]
    L.bs_prefetch_async.argtypes = [vp, vp, u64, C.POINTER(SetDesc), vp, u64, u32, vp, C.POINTER(vp)]
    LD = C.POINTER(LayeredDesc)
    L.bs_layered_header_bytes.restype = u64
    L.bs_layered_header_bytes.argtypes = [u64, u64, u64]
    L.bs_layered_workspace_bytes.restype = u64
    L.bs_layered_workspace_bytes.argtypes = [u32, u32, u32, u64, u64]
    L.bs_layered_stream_info.argtypes = [vp, C.POINTER(LayeredStreamInfo)]
    L.bs_layered_serialized_size.argtypes = [LD, vp, u64, pu64, pu64, vp]
    L.bs_layered_serialize.argtypes = [LD, vp, u64, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_layered_serialize_range.argtypes = [LD, vp, u64, u64, i32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_layered_deserialize.argtypes = [vp, u64, LD, vp, u64, u32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_offload_layered_async.argtypes = [vp, LD, u64, vp, u64, vp, C.POINTER(vp)]
    L.bs_prefetch_layered_async.argtypes = [vp, vp, u64, LD, vp, u64, u32, vp, C.POINTER(vp)]
    pu32 = C.POINTER(C.c_uint32)
    L.bs_package_count.restype = u64
    L.bs_package_count.argtypes = [u64, u64, u64]
    L.bs_package_range.argtypes = [u64, u64, u64, u64, pu64, pu64]
    L.bs_package_workspace_bytes.restype = u64
    L.bs_package_workspace_bytes.argtypes = [u32, u32, u64]
    L.bs_package_emit.argtypes = [C.POINTER(SetDesc), u64, u64, u64, vp, u64, u64, pu32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_package_unpack.argtypes = [vp, u64, u64, u64, C.POINTER(SetDesc), vp, u64, u32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_layered_package_workspace_bytes.restype = u64
    L.bs_layered_package_workspace_bytes.argtypes = [u32, u32, u32, u64, u64]
    L.bs_layered_package_emit.argtypes = [LD, u64, u64, u64, vp, u64, u64, pu32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_layered_package_unpack.argtypes = [vp, u64, u64, u64, LD, vp, u64, u32, vp, u64, vp, C.POINTER(Opts), vp]
    L.bs_offload_packages_async.argtypes = [vp, C.POINTER(SetDesc), u64, u64, u64, vp, u64, u64, pu32, vp, C.POINTER(vp)]
    L.bs_prefetch_packages_async.argtypes = [vp, vp, u64, u64, u64, C.POINTER(SetDesc), vp, u64, u32, vp, C.POINTER(vp)]
    L.bs_offload_layered_packages_async.argtypes = [vp, LD, u64, u64, u64, vp, u64, u64, pu32, vp, C.POINTER(vp)]
    L.bs_prefetch_layered_packages_async.argtypes = [vp, vp, u64, u64, u64, LD, vp, u64, u32, vp, C.POINTER(vp)]
    L.bs_queue_create.argtypes = [C.POINTER(vp), C.POINTER(EngineCfg)]
    L.bs_queue_destroy.argtypes = [vp]
    L.bs_queue_save.argtypes = [vp, u64, C.POINTER(SetDesc), u64, vp, u64, vp]
    L.bs_queue_adopt.argtypes = [vp, u64, vp, u64]
    L.bs_queue_save_layered.argtypes = [vp, u64, C.POINTER(LayeredDesc), u64, vp, u64, vp]
    L.bs_queue_load_layered.argtypes = [vp, u64, C.POINTER(LayeredDesc), vp, u64, u32, vp]
    L.bs_queue_load.argtypes = [vp, u64, C.POINTER(SetDesc), vp, u64, u32, vp]
    L.bs_queue_checkpoint.argtypes = [vp, u64, vp]
    L.bs_queue_wait.argtypes = [vp, u64, C.POINTER(TicketStats), C.POINTER(TicketStats)]
    L.bs_queue_query.argtypes = [vp, u64]
    L.bs_queue_forget.argtypes = [vp, u64]
    L.bs_queue_drain.argtypes = [vp]
    L.bs_queue_get_stats.argtypes = [vp, C.POINTER(QueueStats)]
    L.bs_queue_spill.argtypes = [vp, u64, C.c_char_p]
    L.bs_queue_fill.argtypes = [vp, u64, C.c_char_p, vp, u64]
    L.bs_queue_io_wait.argtypes = [vp, u64, pu64, C.POINTER(C.c_double)]
    L.bs_ticket_wait.argtypes = [vp, C.POINTER(TicketStats)]
    L.bs_ticket_query.argtypes = [vp]
    L.bs_ticket_destroy.argtypes = [vp]
    L.bs_ticket_stream_wait.argtypes = [vp, vp]
    _lib = L
    return L


def _check(rc: int, what: str) -> int:
    if rc < 0:
        raise BsError(rc, what)
    return rc


def _opts(opts):
    if opts is None:
        return None
    return C.byref(make_opts(opts))


def version() -> int:
    return int(lib().bs_version())


def strerror(code: int) -> str:
    return lib().bs_strerror(code).decode()


def last_cuda_error() -> int:
    return int(lib().bs_last_cuda_error())


def header_bytes(n_tensors: int, n_blocks: int) -> int:
    return int(lib().bs_header_bytes(n_tensors, n_blocks))


def header_bytes_rank4(n_tensors: int, n_blocks: int) -> int:
    return int(lib().bs_header_bytes_rank4(n_tensors, n_blocks))


def workspace_bytes(n_tensors: int, n_blocks: int, stream_capacity: int) -> int:
    return int(lib().bs_workspace_bytes(n_tensors, n_blocks, stream_capacity))


def stream_info(first_64_bytes) -> dict:
    """Parse the fixed header from HOST bytes (bytes / bytearray / numpy uint8)."""
    buf = (C.c_ubyte * 64).from_buffer_copy(bytes(first_64_bytes[:64]).ljust(64, b"\0"))
    info = StreamInfo()
    _check(lib().bs_stream_info(C.addressof(buf), C.byref(info)), "bs_stream_info")
    return {k: int(getattr(info, k)) for k, _ in StreamInfo._fields_}


def make_desc(n_tensors: int, n_blocks: int, tensors_ptr: int, qn_ptr: int, dim_ptr: int, addr_ptr: int,
              dtype: int = F64) -> SetDesc:
    return SetDesc(n_tensors, n_blocks, 2, dtype, tensors_ptr, qn_ptr, dim_ptr, addr_ptr)


def serialized_size(desc: SetDesc, ws_ptr: int, ws_bytes: int, stream: int = 0):
    hb, tot = C.c_uint64(0), C.c_uint64(0)
    _check(lib().bs_serialized_size(C.byref(desc), ws_ptr, ws_bytes, C.byref(hb), C.byref(tot), stream), "bs_serialized_size")
    return int(hb.value), int(tot.value)


def serialize(desc: SetDesc, stream_ptr: int, capacity: int, ws_ptr: int, ws_bytes: int, result_ptr: int,
              opts=None, stream: int = 0) -> int:
    return _check(lib().bs_serialize(C.byref(desc), stream_ptr, capacity, ws_ptr, ws_bytes, result_ptr, _opts(opts), stream),
                  "bs_serialize")


NOALLOC_MAX_BLOCKS = 65536
NOALLOC_MAX_STREAM_BYTES = 1 << 30


def noalloc_scratch_bytes() -> int:
    return int(lib().bs_noalloc_scratch_bytes())


def serialize_noalloc(desc: SetDesc, stream_ptr: int, capacity: int, result_ptr: int, opts=None, stream: int = 0) -> int:
    """bs_serialize on the library's built-in workspace: for callers that cannot allocate device memory (bs.h)."""
    return _check(lib().bs_serialize_noalloc(C.byref(desc), stream_ptr, capacity, result_ptr, _opts(opts), stream),
                  "bs_serialize_noalloc")


def serialize_range(desc: SetDesc, dst_ptr: int, lo: int, hi: int, run_scan: bool, ws_ptr: int, ws_bytes: int,
                    result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_serialize_range(C.byref(desc), dst_ptr, lo, hi, int(run_scan), ws_ptr, ws_bytes, result_ptr,
                                           _opts(opts), stream), "bs_serialize_range")


def deserialize(stream_ptr: int, nbytes: int, out: SetDesc, pool_ptr: int, pool_bytes: int, flags: int, ws_ptr: int,
                ws_bytes: int, result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_deserialize(stream_ptr, nbytes, C.byref(out), pool_ptr, pool_bytes, flags, ws_ptr, ws_bytes,
                                       result_ptr, _opts(opts), stream), "bs_deserialize")


def deserialize_range(src_ptr: int, lo: int, hi: int, header_ptr: int, out: SetDesc, flags: int, ws_ptr: int, ws_bytes: int,
                      opts=None, stream: int = 0) -> int:
    return _check(lib().bs_deserialize_range(src_ptr, lo, hi, header_ptr, C.byref(out), flags, ws_ptr, ws_bytes, _opts(opts),
                                             stream), "bs_deserialize_range")


# ---- wire format v2: structure-shared layers ----------------------------------------------------------------------
def layered_header_bytes(n_structs: int, n_layers: int, n_struct_blocks: int) -> int:
    return int(lib().bs_layered_header_bytes(n_structs, n_layers, n_struct_blocks))


def layered_workspace_bytes(n_structs: int, n_struct_blocks: int, n_layers: int, n_addr: int, stream_capacity: int) -> int:
    return int(lib().bs_layered_workspace_bytes(n_structs, n_struct_blocks, n_layers, n_addr, stream_capacity))


def layered_stream_info(first_64_bytes) -> dict:
    buf = (C.c_ubyte * 64).from_buffer_copy(bytes(first_64_bytes[:64]).ljust(64, b"\0"))
    info = LayeredStreamInfo()
    _check(lib().bs_layered_stream_info(C.addressof(buf), C.byref(info)), "bs_layered_stream_info")
    return {k: int(getattr(info, k)) for k, _ in LayeredStreamInfo._fields_}


def make_layered_desc(n_structs: int, n_struct_blocks: int, n_layers: int, n_addr: int, structs_ptr: int, layers_ptr: int,
                      qn_ptr: int, dim_ptr: int, addr_ptr: int, dtype: int = F64) -> LayeredDesc:
    return LayeredDesc(n_structs, n_struct_blocks, n_layers, 2, dtype, 0, n_addr, structs_ptr, layers_ptr, qn_ptr, dim_ptr,
                       addr_ptr)


def layered_serialized_size(desc: LayeredDesc, ws_ptr: int, ws_bytes: int, stream: int = 0):
    hb, tot = C.c_uint64(0), C.c_uint64(0)
    _check(lib().bs_layered_serialized_size(C.byref(desc), ws_ptr, ws_bytes, C.byref(hb), C.byref(tot), stream),
           "bs_layered_serialized_size")
    return int(hb.value), int(tot.value)


def layered_serialize(desc: LayeredDesc, stream_ptr: int, capacity: int, ws_ptr: int, ws_bytes: int, result_ptr: int,
                      opts=None, stream: int = 0) -> int:
    return _check(lib().bs_layered_serialize(C.byref(desc), stream_ptr, capacity, ws_ptr, ws_bytes, result_ptr, _opts(opts),
                                             stream), "bs_layered_serialize")


def layered_serialize_range(desc: LayeredDesc, dst_ptr: int, lo: int, hi: int, run_scan: bool, ws_ptr: int, ws_bytes: int,
                            result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_layered_serialize_range(C.byref(desc), dst_ptr, lo, hi, int(run_scan), ws_ptr, ws_bytes, result_ptr,
                                                   _opts(opts), stream), "bs_layered_serialize_range")


def layered_deserialize(stream_ptr: int, nbytes: int, out: LayeredDesc, pool_ptr: int, pool_bytes: int, flags: int,
                        ws_ptr: int, ws_bytes: int, result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_layered_deserialize(stream_ptr, nbytes, C.byref(out), pool_ptr, pool_bytes, flags, ws_ptr, ws_bytes,
                                               result_ptr, _opts(opts), stream), "bs_layered_deserialize")


# ---- self-contained packages ----------------------------------------------------------------------
PKG_HEADER = 64
PKG_NO_BLOCK = 0xFFFFFFFF


def _slot_map(slot_of):
    if slot_of is None:
        return None
    return (C.c_uint32 * len(slot_of))(*[int(x) for x in slot_of])


def package_count(header_bytes: int, total_bytes: int, cap: int) -> int:
    return int(lib().bs_package_count(header_bytes, total_bytes, cap))


def package_range(header_bytes: int, total_bytes: int, cap: int, index: int):
    lo, hi = C.c_uint64(0), C.c_uint64(0)
    _check(lib().bs_package_range(header_bytes, total_bytes, cap, index, C.byref(lo), C.byref(hi)), "bs_package_range")
    return int(lo.value), int(hi.value)


def package_workspace_bytes(n_tensors: int, n_blocks: int, stream_capacity: int) -> int:
    return int(lib().bs_package_workspace_bytes(n_tensors, n_blocks, stream_capacity))


def package_emit(desc: SetDesc, total_bytes: int, cap: int, stream_id: int, slots_ptr: int, slot_bytes: int, n_slots: int,
                 slot_of, ws_ptr: int, ws_bytes: int, result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_package_emit(C.byref(desc), total_bytes, cap, stream_id, slots_ptr, slot_bytes, n_slots,
                                        _slot_map(slot_of), ws_ptr, ws_bytes, result_ptr, _opts(opts), stream),
                  "bs_package_emit")


def package_unpack(slots_ptr: int, slot_bytes: int, n_slots: int, stream_id: int, out: SetDesc, pool_ptr: int,
                   pool_bytes: int, flags: int, ws_ptr: int, ws_bytes: int, result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_package_unpack(slots_ptr, slot_bytes, n_slots, stream_id, C.byref(out), pool_ptr, pool_bytes, flags,
                                          ws_ptr, ws_bytes, result_ptr, _opts(opts), stream), "bs_package_unpack")


def layered_package_workspace_bytes(n_structs: int, n_struct_blocks: int, n_layers: int, n_addr: int, stream_capacity: int) -> int:
    return int(lib().bs_layered_package_workspace_bytes(n_structs, n_struct_blocks, n_layers, n_addr, stream_capacity))


def layered_package_emit(desc: LayeredDesc, total_bytes: int, cap: int, stream_id: int, slots_ptr: int, slot_bytes: int,
                         n_slots: int, slot_of, ws_ptr: int, ws_bytes: int, result_ptr: int, opts=None, stream: int = 0) -> int:
    return _check(lib().bs_layered_package_emit(C.byref(desc), total_bytes, cap, stream_id, slots_ptr, slot_bytes, n_slots,
                                                _slot_map(slot_of), ws_ptr, ws_bytes, result_ptr, _opts(opts), stream),
                  "bs_layered_package_emit")


def layered_package_unpack(slots_ptr: int, slot_bytes: int, n_slots: int, stream_id: int, out: LayeredDesc, pool_ptr: int,
                           pool_bytes: int, flags: int, ws_ptr: int, ws_bytes: int, result_ptr: int, opts=None,
                           stream: int = 0) -> int:
    return _check(lib().bs_layered_package_unpack(slots_ptr, slot_bytes, n_slots, stream_id, C.byref(out), pool_ptr, pool_bytes,
                                                  flags, ws_ptr, ws_bytes, result_ptr, _opts(opts), stream),
                  "bs_layered_package_unpack")


class Ticket:
    def __init__(self, handle: int):
        self._h = handle

    def query(self) -> int:
        return int(lib().bs_ticket_query(self._h))

    def wait(self) -> dict:
        st = TicketStats()
        rc = lib().bs_ticket_wait(self._h, C.byref(st))
        out = dict(status=int(rc), bytes=int(st.bytes), n_chunks=int(st.n_chunks), dma_ms=float(st.dma_ms),
                   total_ms=float(st.total_ms))
        return out

    def stream_wait(self, stream: int) -> None:
        _check(lib().bs_ticket_stream_wait(self._h, stream), "bs_ticket_stream_wait")

    def destroy(self):
        if self._h:
            lib().bs_ticket_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Engine:
    """bs_engine_create / bs_offload_async / bs_prefetch_async."""

    def __init__(self, max_tensors: int, max_blocks: int, max_stream_bytes: int, chunk_bytes: int = 0, n_staging: int = 0,
                 opts=None):
        o = make_opts(opts)
        cfg = EngineCfg(chunk_bytes, n_staging, max_tensors, max_blocks, max_stream_bytes, o)
        h = C.c_void_p(0)
        _check(lib().bs_engine_create(C.byref(h), C.byref(cfg)), "bs_engine_create")
        self._h = h.value

    def offload_async(self, desc: SetDesc, total_bytes: int, h_pinned_ptr: int, h_capacity: int, producer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_offload_async(self._h, C.byref(desc), total_bytes, h_pinned_ptr, h_capacity, producer, C.byref(t)),
               "bs_offload_async")
        return Ticket(t.value)

    def prefetch_async(self, h_pinned_ptr: int, nbytes: int, out: SetDesc, pool_ptr: int, pool_bytes: int, flags: int = 0,
                       consumer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_prefetch_async(self._h, h_pinned_ptr, nbytes, C.byref(out), pool_ptr, pool_bytes, flags, consumer,
                                       C.byref(t)), "bs_prefetch_async")
        return Ticket(t.value)

    def offload_packages_async(self, desc: SetDesc, total_bytes: int, cap: int, stream_id: int, h_slots_ptr: int,
                               slot_bytes: int, n_slots: int, slot_of=None, producer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_offload_packages_async(self._h, C.byref(desc), total_bytes, cap, stream_id, h_slots_ptr, slot_bytes,
                                               n_slots, _slot_map(slot_of), producer, C.byref(t)), "bs_offload_packages_async")
        return Ticket(t.value)

    def prefetch_packages_async(self, h_slots_ptr: int, slot_bytes: int, n_slots: int, stream_id: int, out: SetDesc,
                                pool_ptr: int, pool_bytes: int, flags: int = 0, consumer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_prefetch_packages_async(self._h, h_slots_ptr, slot_bytes, n_slots, stream_id, C.byref(out), pool_ptr,
                                                pool_bytes, flags, consumer, C.byref(t)), "bs_prefetch_packages_async")
        return Ticket(t.value)

    def offload_layered_packages_async(self, desc: LayeredDesc, total_bytes: int, cap: int, stream_id: int, h_slots_ptr: int,
                                       slot_bytes: int, n_slots: int, slot_of=None, producer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_offload_layered_packages_async(self._h, C.byref(desc), total_bytes, cap, stream_id, h_slots_ptr, slot_bytes,
                                                       n_slots, _slot_map(slot_of), producer, C.byref(t)),
               "bs_offload_layered_packages_async")
        return Ticket(t.value)

    def prefetch_layered_packages_async(self, h_slots_ptr: int, slot_bytes: int, n_slots: int, stream_id: int, out: LayeredDesc,
                                        pool_ptr: int, pool_bytes: int, flags: int = 0, consumer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_prefetch_layered_packages_async(self._h, h_slots_ptr, slot_bytes, n_slots, stream_id, C.byref(out), pool_ptr,
                                                        pool_bytes, flags, consumer, C.byref(t)), "bs_prefetch_layered_packages_async")
        return Ticket(t.value)

    def offload_layered_async(self, desc: LayeredDesc, total_bytes: int, h_pinned_ptr: int, h_capacity: int,
                              producer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_offload_layered_async(self._h, C.byref(desc), total_bytes, h_pinned_ptr, h_capacity, producer,
                                              C.byref(t)), "bs_offload_layered_async")
        return Ticket(t.value)

    def prefetch_layered_async(self, h_pinned_ptr: int, nbytes: int, out: LayeredDesc, pool_ptr: int, pool_bytes: int,
                               flags: int = 0, consumer: int = 0) -> Ticket:
        t = C.c_void_p(0)
        _check(lib().bs_prefetch_layered_async(self._h, h_pinned_ptr, nbytes, C.byref(out), pool_ptr, pool_bytes, flags,
                                               consumer, C.byref(t)), "bs_prefetch_layered_async")
        return Ticket(t.value)

    def destroy(self):
        if self._h:
            lib().bs_engine_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Queue:
    """bs_queue_*: a save lane and a load lane (one per PCIe direction) + keys ordered by events."""

    def __init__(self, max_tensors: int, max_blocks: int, max_stream_bytes: int, chunk_bytes: int = 0, n_staging: int = 0,
                 opts=None):
        cfg = EngineCfg(chunk_bytes, n_staging, max_tensors, max_blocks, max_stream_bytes, make_opts(opts))
        h = C.c_void_p(0)
        _check(lib().bs_queue_create(C.byref(h), C.byref(cfg)), "bs_queue_create")
        self._h = h.value
        self._keys = set()   # which keys exist (BS_ERR_ARG is also a deferred status, so wait() must tell them apart)

    def save(self, key: int, desc: SetDesc, total_bytes: int, h_pinned_ptr: int, h_capacity: int, producer: int = 0) -> None:
        _check(lib().bs_queue_save(self._h, key, C.byref(desc), total_bytes, h_pinned_ptr, h_capacity, producer), "bs_queue_save")
        self._keys.add(key)

    def save_layered(self, key: int, desc: LayeredDesc, total_bytes: int, h_pinned_ptr: int, h_capacity: int, producer: int = 0) -> None:
        _check(lib().bs_queue_save_layered(self._h, key, C.byref(desc), total_bytes, h_pinned_ptr, h_capacity, producer),
               "bs_queue_save_layered")
        self._keys.add(key)

    def load_layered(self, key: int, out: LayeredDesc, pool_ptr: int, pool_bytes: int, flags: int = 0, consumer: int = 0) -> None:
        _check(lib().bs_queue_load_layered(self._h, key, C.byref(out), pool_ptr, pool_bytes, flags, consumer), "bs_queue_load_layered")

    def adopt(self, key: int, h_pinned_ptr: int, nbytes: int) -> None:
        _check(lib().bs_queue_adopt(self._h, key, h_pinned_ptr, nbytes), "bs_queue_adopt")
        self._keys.add(key)

    def load(self, key: int, out: SetDesc, pool_ptr: int, pool_bytes: int, flags: int = 0, consumer: int = 0) -> None:
        _check(lib().bs_queue_load(self._h, key, C.byref(out), pool_ptr, pool_bytes, flags, consumer), "bs_queue_load")

    def checkpoint(self, key: int, stream: int = 0) -> None:
        _check(lib().bs_queue_checkpoint(self._h, key, stream), "bs_queue_checkpoint")

    def wait(self, key: int) -> dict:
        """Host-blocking.  Returns the first deferred status and the two operations' stats (no exception for deferred errors)."""
        s, l = TicketStats(), TicketStats()
        if key not in self._keys:
            raise BsError(ERR_ARG, "bs_queue_wait: unknown key")
        rc = lib().bs_queue_wait(self._h, key, C.byref(s), C.byref(l))
        f = lambda st: dict(status=int(st.status), bytes=int(st.bytes), n_chunks=int(st.n_chunks), dma_ms=float(st.dma_ms),
                            total_ms=float(st.total_ms))
        return dict(status=int(rc), save=f(s), load=f(l))

    def query_raw(self, key: int) -> int:
        return int(lib().bs_queue_query(self._h, key))

    def forget(self, key: int) -> None:
        _check(lib().bs_queue_forget(self._h, key), "bs_queue_forget")
        self._keys.discard(key)

    def spill(self, key: int, path: str) -> None:
        _check(lib().bs_queue_spill(self._h, key, os.fsencode(path)), "bs_queue_spill")

    def fill(self, key: int, path: str, h_pinned_ptr: int, h_capacity: int) -> None:
        _check(lib().bs_queue_fill(self._h, key, os.fsencode(path), h_pinned_ptr, h_capacity), "bs_queue_fill")
        self._keys.add(key)

    def io_wait(self, key: int) -> dict:
        """Host-blocking: outcome of the key's last storage job (no exception for BS_ERR_IO)."""
        n, sec = C.c_uint64(0), C.c_double(0.0)
        rc = lib().bs_queue_io_wait(self._h, key, C.byref(n), C.byref(sec))
        return dict(status=int(rc), bytes=int(n.value), seconds=float(sec.value))

    def drain(self) -> None:
        _check(lib().bs_queue_drain(self._h), "bs_queue_drain")

    def stats(self) -> dict:
        st = QueueStats()
        _check(lib().bs_queue_get_stats(self._h, C.byref(st)), "bs_queue_get_stats")
        return {k: int(getattr(st, k)) for k, _ in QueueStats._fields_}

    def destroy(self):
        if self._h:
            lib().bs_queue_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
