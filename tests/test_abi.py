"""The C-ABI library loads and exports every symbol include/bs.h declares; host-only entry points work without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2412_04676_b200 as bs
from tests.util import read_hex_fixture

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "bs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(bs_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_every_declared_symbol_is_exported():
    lib = bs.lib()
    names = declared_functions()
    assert {"bs_serialize", "bs_deserialize", "bs_offload_async", "bs_prefetch_async", "bs_serialized_size",
            "bs_stream_info", "bs_engine_create", "bs_ticket_wait"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/bs.h but not exported"


def test_struct_layouts_match_the_header():
    assert ctypes.sizeof(bs.SetDesc) == 48
    assert ctypes.sizeof(bs.Result) == 64
    assert ctypes.sizeof(bs.Opts) == 32


def test_host_only_entry_points():
    assert bs.version() == 0x00010200
    assert bs.header_bytes(1, 2) == 256 and bs.header_bytes(0, 0) == 128
    assert bs.header_bytes(2000, 446140) == (64 + 32 * 2000 + 48 * 446140 + 127) // 128 * 128
    assert bs.workspace_bytes(1, 7, 1 << 20) % 256 == 0
    assert bs.workspace_bytes(9008, 3299211, 45 << 30) < 200 << 20      # O(B) + 4 B per 16 KiB of stream
    raw = read_hex_fixture(os.path.join(ROOT, "tests", "golden", "p7_golden_stream.hex"))
    assert bs.stream_info(raw) == dict(n_tensors=1, n_blocks=2, header_bytes=256, payload_bytes=32, total_bytes=288, dtype=0, align=16, max_rank=3)
    g7 = read_hex_fixture(os.path.join(ROOT, "tests", "golden", "g7_golden_stream_align8.hex"))
    assert bs.stream_info(g7) == dict(n_tensors=1, n_blocks=2, header_bytes=256, payload_bytes=24, total_bytes=280, dtype=0, align=8, max_rank=3)
    g8 = read_hex_fixture(os.path.join(ROOT, "tests", "golden", "g8_golden_stream_v3.hex"))
    assert bs.stream_info(g8) == dict(n_tensors=2, n_blocks=3, header_bytes=384, payload_bytes=64, total_bytes=448, dtype=0, align=16, max_rank=4)
    assert bs.header_bytes_rank4(2, 3) == 384
    f32 = read_hex_fixture(os.path.join(ROOT, "tests", "golden", "g4_golden_stream_f32.hex"))
    assert bs.stream_info(f32)["dtype"] == bs.F32
    for pos in (0, 8, 12, 16, 20, 24, 28, 48):
        bad = bytearray(raw)
        bad[pos] ^= 4 if pos in (16, 28) else 1      # align words 16 and 8 are both formats (16 ^ 4 = 20 is none)      # dtype words 0..3 are element types
        with pytest.raises(bs.BsError) as e:
            bs.stream_info(bad)
        assert e.value.code == bs.ERR_CORRUPT
    assert "corrupt" in bs.strerror(bs.ERR_CORRUPT) and bs.strerror(0) == "ok"


def test_argument_errors_need_no_device():
    d = bs.make_desc(1, 1, 16, 16, 16, 16)
    d.n_qn = 3
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d, 256, 1024, 256, 1 << 20, 0)
    assert e.value.code == bs.ERR_UNSUPPORTED
    d = bs.make_desc(1, 1, 8, 16, 16, 16)          # tensors not 16-byte aligned
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d, 256, 1024, 256, 1 << 20, 0)
    assert e.value.code == bs.ERR_ARG
    d = bs.make_desc(1, 1, 16, 16, 16, 16)
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d, 256, 1024, 256, 64, 0)     # workspace too small
    assert e.value.code == bs.ERR_CAPACITY


def test_rank4_sets_need_16_byte_aligned_label_and_extent_arrays():
    """A BS_RANK4 set's qn / dim rows are 32 / 16 bytes and move as 16-byte words: arrays 8 (or 4) off that grid — a sub-view
    of a larger allocation — are BS_ERR_ARG up front, not a misaligned-address fault in the kernel.  Plain sets keep 8 / 4."""
    for qn, dim, ok in ((32, 32, True), (40, 32, False), (32, 40, False), (32, 36, False)):
        d = bs.make_desc(1, 1, 16, qn, dim, 16, dtype=bs.F64 | bs.RANK4)
        if ok:      # passes the descriptor check; the (too small) workspace is what is refused next
            with pytest.raises(bs.BsError) as e:
                bs.serialize(d, 256, 1024, 256, 64, 0)
            assert e.value.code == bs.ERR_CAPACITY
            continue
        for call in (lambda: bs.serialize(d, 256, 1024, 256, 1 << 20, 0),
                     lambda: bs.deserialize(256, 1024, d, 256, 1 << 20, bs.LAYOUT_POOL, 256, 1 << 20, 0),
                     lambda: bs.serialize_noalloc(d, 256, 1024, 256)):
            with pytest.raises(bs.BsError) as e:
                call()
            assert e.value.code == bs.ERR_ARG
    d = bs.make_desc(1, 1, 16, 40, 36, 16)         # three legs: 8- and 4-byte alignment is enough
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d, 256, 1024, 256, 64, 0)
    assert e.value.code == bs.ERR_CAPACITY


def test_launch_shapes_are_checked_without_a_device():
    """bs_opts: a TMA tile is any multiple of 1 KiB from 4 KiB to 64 KiB (round 2), an LDG tile a multiple of 16 KiB; rings
    must fit the shared memory.  A shape the kernels cannot run is BS_ERR_ARG before anything touches the device."""
    d = bs.make_desc(1, 1, 16, 16, 16, 16)
    bad = [dict(variant=bs.VARIANT_TMA, tile_bytes=6000, stages=3, warps=1), dict(variant=bs.VARIANT_TMA, tile_bytes=2048, stages=3, warps=1),
           dict(variant=bs.VARIANT_TMA, tile_bytes=66560, stages=3, warps=1), dict(variant=bs.VARIANT_LDG, tile_bytes=8192),
           dict(variant=bs.VARIANT_LDG, tile_bytes=20480), dict(variant=bs.VARIANT_TMA, tile_bytes=20480, stages=6, warps=2),
           dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=2, warps=1), dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=9, warps=1),
           dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=17), dict(variant=7),
           # the named switches (round 3; they used to ride in bs_opts.reserved[], where garbage could not be refused)
           dict(variant=bs.VARIANT_TMA, fuse=3), dict(variant=bs.VARIANT_TMA, tune=0x4), dict(variant=bs.VARIANT_TMA, tune=0x80000010),
           dict(variant=bs.VARIANT_LDG, tile_bytes=16384, tune=0x2000)]
    for o in bad:
        with pytest.raises(bs.BsError) as e:
            bs.serialize(d, 256, 1024, 256, 1 << 20, 0, o)
        assert e.value.code == bs.ERR_ARG, o
    import torch
    if not torch.cuda.is_available():   # a good shape gets as far as the device: there is none here
        for o in (dict(variant=bs.VARIANT_TMA, tile_bytes=20480, stages=5, warps=2), dict(variant=bs.VARIANT_TMA, tile_bytes=5120, stages=8, warps=4),
                  dict(variant=bs.VARIANT_TMA, tile_bytes=65536, stages=3, warps=1, pace=6500, tune=0x1018), dict(variant=bs.VARIANT_LDG, tile_bytes=49152)):
            with pytest.raises(bs.BsError) as e:
                bs.serialize(d, 256, 1024, 256, 1 << 20, 0, o)
            assert e.value.code == bs.ERR_CUDA, o


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("box has a GPU")
    d = bs.make_desc(0, 0, 0, 0, 0, 0)
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d, 256, 1024, 256, 1 << 20, 0)
    assert e.value.code == bs.ERR_CUDA
