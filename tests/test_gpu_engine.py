"""S8/S9: the asynchronous offload / prefetch engine against the oracle (concat(chunks) == stream)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from tests.gpu_util import DEV, Uploaded
from tests.util import oracle_stream

pytestmark = pytest.mark.gpu


def pinned(n, fill):
    t = torch.empty(max(n, 16), dtype=torch.uint8, pin_memory=True)
    t.fill_(fill)
    return t


@pytest.mark.parametrize("chunk,n_staging,opts", [(65536, 2, None), (65536 * 5, 1, None), (65536 * 16, 3, None), (1 << 28, 2, None),
                                                  # every chunk's tiles handed out by the counter (what chunks of 128 MiB and more do)
                                                  (65536 * 5, 2, dict(variant=2, tune=0x10)), (65536 * 16, 3, dict(variant=2, tune=0x10))])
def test_offload_then_prefetch_round_trip(chunk, n_staging, opts):
    bset = W.make_config("2")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total + 4096, chunk_bytes=chunk, n_staging=n_staging, opts=opts)
    host = pinned(total + 4096, 0xCD)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    hb, tot = bs.serialized_size(up.dset.desc, ws.ptr, ws.nbytes, bs.current_stream())
    assert tot == total
    t = eng.offload_async(up.dset.desc, tot, host.data_ptr(), host.numel(), bs.current_stream())
    st = t.wait()
    assert st["status"] == bs.OK and st["bytes"] == total and st["n_chunks"] == -(-total // chunk)
    got = host.numpy()
    assert (got[:total] == want).all(), "concat(chunks) != oracle stream"
    assert (got[total:] == 0xCD).all()

    # load it back through the engine
    ref = oracle.deserialize(want)
    need = oracle.pool_bytes(want)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    t2 = eng.prefetch_async(host.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, bs.current_stream())
    # the consumer stream waits on the ticket's event: work enqueued now sees the data (checkpoint)
    snapshot = pool.clone()
    st2 = t2.wait()
    assert st2["status"] == bs.OK, st2
    assert (snapshot.cpu().numpy() == ref["pool"][:need]).all()
    h = out.to_host()
    assert h["tensors"].tobytes() == bset.tensors.tobytes() and (h["qn"] == bset.qn).all() and (h["dim"] == bset.dim).all()
    eng.destroy()


def test_offload_size_zero_means_query_and_mismatch_is_an_error():
    bset = W.make_config("1")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    eng = bs.Engine(4, 64, 1 << 20, chunk_bytes=65536)
    host = pinned(1 << 20, 0xCD)
    t = eng.offload_async(up.dset.desc, 0, host.data_ptr(), host.numel(), bs.current_stream())
    assert t.wait()["status"] == bs.OK
    assert (host.numpy()[:len(want)] == want).all()
    t = eng.offload_async(up.dset.desc, len(want) + 16, host.data_ptr(), host.numel(), bs.current_stream())
    assert t.wait()["status"] == bs.ERR_ARG                      # size prediction re-checked on the device
    with pytest.raises(bs.BsError) as e:
        eng.offload_async(up.dset.desc, len(want), host.data_ptr(), len(want) - 16, bs.current_stream())
    assert e.value.code == bs.ERR_CAPACITY
    eng.destroy()


def test_prefetch_rejects_corrupt_streams():
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    want, _, _ = oracle_stream(bset)
    need = oracle.pool_bytes(want)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, len(want), chunk_bytes=65536)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    host = pinned(len(want), 0)
    # a corrupt block record: caught by the device-side header validation, nothing written
    bad = want.copy()
    bad[64 + 32 * bset.n_tensors + 48 + 40] ^= 0x10
    host.numpy()[:] = bad
    t = eng.prefetch_async(host.data_ptr(), len(want), out.desc, pool.data_ptr(), need)
    assert t.wait()["status"] == bs.ERR_CORRUPT
    torch.cuda.synchronize()
    assert (pool == 0xEE).all() and (out.qn == 0xAB).all()
    # a corrupt fixed header: caught on the host at once
    bad = want.copy()
    bad[0] ^= 1
    host.numpy()[:] = bad
    with pytest.raises(bs.BsError) as e:
        eng.prefetch_async(host.data_ptr(), len(want), out.desc, pool.data_ptr(), need)
    assert e.value.code == bs.ERR_CORRUPT
    # a non-zero pad byte: the payload is checked as it streams through the unpack kernel
    odd = int(np.nonzero(bset.nelems % 2 == 1)[0][0])
    _, _, off, _ = oracle.plan(bset.dim)
    bad = want.copy()
    bad[oracle.header_bytes(bset.n_tensors, bset.n_blocks) + int(off[odd]) + int(bset.nelems[odd]) * 8] ^= 1
    host.numpy()[:] = bad
    t = eng.prefetch_async(host.data_ptr(), len(want), out.desc, pool.data_ptr(), need)
    assert t.wait()["status"] == bs.ERR_CORRUPT
    eng.destroy()


def test_prefetch_rejects_a_payload_without_blocks():
    """T = 0, B = 0, payload_bytes != 0 through the engine (the LDG variant used to index the block table at B - 1)."""
    import struct
    P = 65536 + 32
    bad = np.zeros(128 + P, np.uint8)
    bad[:64] = np.frombuffer(b"BSPARSE1" + struct.pack("<IIIIIIQQQQ", 1, 0x01020304, 0, 2, 3, 16, 0, 0, 128, P), np.uint8)
    assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
    host = pinned(len(bad), 0)
    host.numpy()[:] = bad
    for opts in (None, dict(variant=bs.VARIANT_LDG)):
        eng = bs.Engine(4, 64, len(bad), chunk_bytes=65536, opts=opts)
        pool = torch.full((4096,), 0xEE, dtype=torch.uint8, device=DEV)
        out = bs.DeviceSet.empty(4, 64, DEV, fill=0xAB)
        t = eng.prefetch_async(host.data_ptr(), len(bad), out.desc, pool.data_ptr(), 4096)
        assert t.wait()["status"] == bs.ERR_CORRUPT
        torch.cuda.synchronize()
        assert (pool == 0xEE).all() and (out.qn == 0xAB).all()
        eng.destroy()


def test_engine_checks_what_the_direct_calls_check():
    """A descriptor or a launch shape bs_serialize would refuse is refused by the engine too, at once — not saved as a
    stream no loader accepts, not a device fault."""
    bset = W.make_config("1")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    host = pinned(1 << 20, 0xCD)
    for bad in (dict(variant=bs.VARIANT_TMA, tile_bytes=6000, stages=3, warps=1),      # not a multiple of 1 KiB
                dict(variant=bs.VARIANT_LDG, tile_bytes=8192)):                         # LDG: not a multiple of 16 KiB
        with pytest.raises(bs.BsError) as e:
            bs.Engine(4, 64, 1 << 20, chunk_bytes=65536, opts=bad)
        assert e.value.code == bs.ERR_ARG
    eng = bs.Engine(4, 64, 1 << 20, chunk_bytes=65536)
    cs = bs.current_stream()
    d = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, up.addr, DEV, dtype=7)            # unknown element type
    with pytest.raises(bs.BsError) as e:
        eng.offload_async(d.desc, 0, host.data_ptr(), host.numel(), cs)
    assert e.value.code == bs.ERR_UNSUPPORTED
    with pytest.raises(bs.BsError) as e:
        eng.offload_packages_async(d.desc, 0, 16384, 1, host.data_ptr(), 64 + 16384, 8, None, cs)
    assert e.value.code == bs.ERR_UNSUPPORTED
    nul = bs.make_desc(bset.n_tensors, bset.n_blocks, up.dset.tensors.data_ptr(), 0, up.dset.dim.data_ptr(),
                       up.dset.addr.data_ptr())                                               # NULL label array
    with pytest.raises(bs.BsError) as e:
        eng.offload_async(nul, len(want), host.data_ptr(), host.numel(), cs)
    assert e.value.code == bs.ERR_ARG
    host.numpy()[:len(want)] = want
    out = bs.DeviceSet.empty(4, 64, DEV, fill=0xAB)
    bad_out = bs.make_desc(4, 64, out.tensors.data_ptr(), out.qn.data_ptr(), 0, out.addr.data_ptr())
    with pytest.raises(bs.BsError) as e:
        eng.prefetch_async(host.data_ptr(), len(want), bad_out, 0, 0)
    assert e.value.code == bs.ERR_ARG
    assert (host.numpy()[len(want):] == 0xCD).all()
    eng.destroy()


def test_a_failed_offload_leaves_no_valid_header_on_the_host():
    """On a deferred error the pack kernels write nothing but the DMA of every chunk still runs: the staging buffers hold
    the stream of the call before.  The engine has the 64 bytes of the fixed header blanked, so the host never sees a
    stale stream as valid (chunks and packages)."""
    bset = W.make_config("1")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    eng = bs.Engine(4, 64, 1 << 20, chunk_bytes=65536)
    cs = bs.current_stream()
    host = pinned(1 << 20, 0xCD)
    assert eng.offload_async(up.dset.desc, total, host.data_ptr(), host.numel(), cs).wait()["status"] == bs.OK
    assert bs.stream_info(host.numpy()[:64].tobytes())["total_bytes"] == total
    host.fill_(0xCD)
    t = eng.offload_async(up.dset.desc, total + 16, host.data_ptr(), host.numel(), cs)      # wrong size prediction
    assert t.wait()["status"] == bs.ERR_ARG
    with pytest.raises(bs.BsError):
        bs.stream_info(host.numpy()[:64].tobytes())
    assert (host.numpy()[:64] == 0).all()
    # packages: every slot header of the failed call is blank
    cap = 16384
    n = bs.package_count(bs.header_bytes(bset.n_tensors, bset.n_blocks), total, cap)
    slots = pinned((n + 1) * (64 + cap), 0xCD)      # one spare slot: the wrong size below may cut one package more
    assert eng.offload_packages_async(up.dset.desc, total, cap, 5, slots.data_ptr(), 64 + cap, n, None, cs).wait()["status"] == bs.OK
    assert bytes(slots.numpy()[:8]) == b"BSPKG001"
    slots.fill_(0xCD)
    t = eng.offload_packages_async(up.dset.desc, total + 16, cap, 5, slots.data_ptr(), 64 + cap, n + 1, None, cs)
    assert t.wait()["status"] == bs.ERR_ARG
    sl = slots.numpy().reshape(n + 1, 64 + cap)
    assert not any(bytes(sl[k, :8]) == b"BSPKG001" for k in range(n + 1))
    eng.destroy()


def test_offload_overlaps_a_busy_compute_stream():
    """The producer stream is not blocked and the result is the same stream while a stand-in contraction runs."""
    from workloads.device import StandInContraction
    bset = W.make_config("2")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total, chunk_bytes=1 << 22)
    host = pinned(total, 0xCD)
    work = StandInContraction(bset, up.addr, DEV)
    t = eng.offload_async(up.dset.desc, total, host.data_ptr(), host.numel(), bs.current_stream())
    work.run(reps=3)                      # enqueued after the offload call returned; reads the same blocks
    st = t.wait()
    torch.cuda.synchronize()
    assert st["status"] == bs.OK
    assert (host.numpy()[:total] == want).all()
    eng.destroy()
