"""bs_serialize_noalloc: the entry point for callers that cannot allocate device memory.

Who needs it: the solver this library serves gives the HBM that is left to its own block pool, and it saves scratch data
exactly when memory is tight, so a cudaMalloc for a workspace can fail at that moment; a plug-in inside
such a program is not allowed to allocate behind the pool's back at all; and cudaMalloc / cudaFree synchronise the whole
device, which a caller that hides its offload behind side streams cannot afford.  For them the library carries a fixed
1.5 MiB array per GPU and uses it as the workspace (include/bs.h, csrc/bs_noalloc.cu).

What is checked: the stream and the result word of the new call equal those of bs_serialize on a caller-owned workspace —
byte for byte, the tolerance of every parity test here is 0 — on two calls IN A ROW on different sets, so the second call
finds the first one's tables, scan state and counters in the shared array; then the first set again, behind the larger
one.  The limits are refused up front, and that needs no GPU.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide the other files)
and passes on its own in a fresh process as well as behind the rest of the suite.
"""
import numpy as np
import pytest
import torch

import paper_2412_04676_b200 as bs
import workloads as W


def test_limits_are_stated_and_refused_before_the_device_is_touched():
    # the array is large enough for the stated limits
    assert bs.workspace_bytes(0, bs.NOALLOC_MAX_BLOCKS, bs.NOALLOC_MAX_STREAM_BYTES) <= bs.noalloc_scratch_bytes() == 1536 * 1024
    d = bs.make_desc(1, bs.NOALLOC_MAX_BLOCKS + 1, 16, 16, 16, 16)
    with pytest.raises(bs.BsError) as e:
        bs.serialize_noalloc(d, 256, 1 << 20, 256)
    assert e.value.code == bs.ERR_CAPACITY
    d = bs.make_desc(1, 1, 16, 16, 16, 16)
    with pytest.raises(bs.BsError) as e:
        bs.serialize_noalloc(d, 256, bs.NOALLOC_MAX_STREAM_BYTES + 16, 256)
    assert e.value.code == bs.ERR_CAPACITY
    d.n_qn = 3                                   # descriptor errors come out as for bs_serialize
    with pytest.raises(bs.BsError) as e:
        bs.serialize_noalloc(d, 256, 1 << 20, 256)
    assert e.value.code == bs.ERR_UNSUPPORTED


def _both_ways(bset, opts=None):
    """(stream, result) of bs_serialize on its own workspace and of bs_serialize_noalloc, same set, poisoned buffers."""
    from tests.gpu_util import DEV, Uploaded, gpu_serialize
    up = Uploaded(bset)
    total = bs.serialized_size(up.dset.desc, *_ws(up.dset, DEV), bs.current_stream())[1]
    cap = total + 4096
    ref_t, ref_res = gpu_serialize(up.dset, cap, opts)
    got_t = torch.full((cap,), 0xCD, dtype=torch.uint8, device=DEV)
    result = torch.full((64,), 0xA5, dtype=torch.uint8, device=DEV)
    bs.serialize_noalloc(up.dset.desc, got_t.data_ptr(), cap, result.data_ptr(), opts, bs.current_stream())
    r = bs.Result.from_buffer_copy(result.cpu().numpy().tobytes())
    got_res = dict(status=int(r.status), total_bytes=int(r.total_bytes), header_bytes=int(r.header_bytes),
                   payload_bytes=int(r.payload_bytes), n_tensors=int(r.n_tensors), n_blocks=int(r.n_blocks))
    return total, ref_t.cpu().numpy(), ref_res, got_t.cpu().numpy(), got_res


_keep = []


def _ws(dset, dev):
    w = bs.Workspace(dset.n_tensors, dset.n_blocks, 1 << 30, dev)
    _keep.append(w)
    return w.ptr, w.nbytes


def _same(bset, opts=None):
    total, ref, ref_res, got, got_res = _both_ways(bset, opts)
    assert ref_res["status"] == bs.OK and got_res["status"] == bs.OK, (ref_res, got_res)
    for k in got_res:
        assert got_res[k] == ref_res[k], (k, got_res, ref_res)
    assert got_res["total_bytes"] == total
    bad = np.nonzero(got != ref)[0]               # the stream AND the untouched poison behind it
    assert bad.size == 0, f"{bset.name}: first difference from bs_serialize at byte {bad[0]} of {total}"


@pytest.mark.gpu
def test_two_calls_in_a_row_write_what_bs_serialize_writes():
    small, larger = W.make_config("1"), W.make_config("2")     # 1 item of the pass / 23 items, 77 MB: several hundred tiles
    assert larger.n_blocks <= bs.NOALLOC_MAX_BLOCKS
    _same(small)            # first use of the array on this device (or not, behind the rest of the suite: both must work)
    _same(larger)           # finds the small set's leftovers
    _same(small)            # finds the larger set's: more scan items and table entries than this call writes
    # the two-launch form and the tile counter use further words of the shared head
    _same(larger, dict(variant=bs.VARIANT_TMA, fuse=1, tune=0x10))
    _same(small, dict(variant=bs.VARIANT_LDG, tile_bytes=16384))
    _keep.clear()


@pytest.mark.gpu
def test_a_stream_larger_than_the_callers_buffer_is_the_usual_deferred_error():
    from tests.gpu_util import DEV, Uploaded
    up = Uploaded(W.make_config("1"))
    total = bs.serialized_size(up.dset.desc, *_ws(up.dset, DEV), bs.current_stream())[1]
    out = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    result = torch.zeros(64, dtype=torch.uint8, device=DEV)
    bs.serialize_noalloc(up.dset.desc, out.data_ptr(), total - 16, result.data_ptr(), None, bs.current_stream())
    r = bs.Result.from_buffer_copy(result.cpu().numpy().tobytes())
    assert int(r.status) == bs.ERR_CAPACITY and int(r.total_bytes) == total
    assert (out.cpu().numpy() == 0xCD).all(), "nothing may be written when the stream does not fit"
    _keep.clear()
