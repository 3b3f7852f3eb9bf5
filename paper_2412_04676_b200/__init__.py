"""paper_2412_04676_b200 — B200-native serialization / offload of U(1) block-sparse DMRG scratch data.

Python face of the C-ABI library ``libbsstream.so`` (include/bs.h): same names, argument marshalling only.
PyTorch is used for device memory and streams, nothing else; every step of the path (size/offset scan, header
write, pack, header parse, unpack, chunked offload/prefetch) runs in the library's hand-written CUDA kernels.
There is no CPU fallback.
"""
from ._binding import (  # noqa: F401
    ALIGN8, RANK4, C64, C128, ERR_ARG, ERR_CAPACITY, ERR_CORRUPT, ERR_CUDA, ERR_IO, ERR_UNSUPPORTED, F32, F64, LAYOUT_POOL, OK, PENDING, SCATTER_TO_ADDR,
    VARIANT_DEFAULT, VARIANT_LDG, VARIANT_TMA,
    BsError, Engine, LayeredDesc, Opts, Queue, Result, SetDesc, Ticket,
    layered_deserialize, layered_header_bytes, layered_serialize, layered_serialize_range, layered_serialized_size,
    layered_stream_info, layered_workspace_bytes, make_layered_desc,
    deserialize, deserialize_range, header_bytes, header_bytes_rank4, last_cuda_error, lib, make_desc, serialize, serialize_noalloc, serialize_range, serialized_size,
    NOALLOC_MAX_BLOCKS, NOALLOC_MAX_STREAM_BYTES, noalloc_scratch_bytes,
    stream_info, strerror, version, workspace_bytes,
    PKG_HEADER, PKG_NO_BLOCK, layered_package_emit, layered_package_unpack, layered_package_workspace_bytes, package_count, package_emit, package_range, package_unpack, package_workspace_bytes,
)
from .device import DeviceLayeredSet, DeviceSet, Workspace, current_stream  # noqa: F401
