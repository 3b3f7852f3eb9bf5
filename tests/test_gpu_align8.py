"""Unpadded streams on the GPU (bs.h BS_ALIGN8; DESIGN.md §18 reading D19): wire format v1 with the
header's align word = 8, through the C ABI against the oracles (bs_oracle.c `_al` entry points for fp64, the independent
numpy oracle bs_oracle_dtype.py for the other element types).  Bit-exact.  Every test needs a GPU."""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from oracle import dt
from tests.gpu_util import DEV, Uploaded
from tests.util import host_addrs, read_hex_fixture

pytestmark = pytest.mark.gpu

SHAPES = [None, dict(variant=bs.VARIANT_TMA, fuse=1), dict(variant=bs.VARIANT_TMA, fuse=2),
          dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=4, warps=1), dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=3, warps=1),
          dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=4, fuse=2), dict(variant=bs.VARIANT_TMA, tile_bytes=65536),
          # what sets of half a GB and more select for themselves (tests/test_gpu_fullsize.py runs it at that size): tiles
          # from the counter (tune 0x10), the table two iterations ahead (0x1000), one ring of 3 x 48 KiB
          dict(variant=bs.VARIANT_TMA, tune=0x10), dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=3, warps=1, tune=0x1010),
          dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=3, warps=1, tune=0x1010, fuse=2)]


def sets():
    return [W.make_config("1"), W.make_config("2"),
            W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial"),
            W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)]


def a8_set(up, dtype=bs.F64):
    b = up.bset
    return bs.DeviceSet.from_host(b.tensors, b.qn, b.dim, up.addr, DEV, dtype=dtype | bs.ALIGN8)


def serialize(dset, capacity, opts=None, ws=None):
    out = torch.full((max(capacity, 16),), 0xCD, dtype=torch.uint8, device=DEV)
    ws = ws or bs.Workspace(dset.n_tensors, dset.n_blocks, max(capacity, 1 << 16), DEV)
    bs.serialize(dset.desc, out.data_ptr(), capacity, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    return out, ws.read_result()


def deserialize(stream_t, nbytes, cap_t, cap_b, pool_bytes, opts=None, flags=bs.LAYOUT_POOL, out=None):
    out = out or bs.DeviceSet.empty(cap_t, cap_b, DEV, fill=0xAB)
    pool = torch.full((max(pool_bytes, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(cap_t, cap_b, max(nbytes, 1 << 16), DEV)
    bs.deserialize(stream_t.data_ptr(), nbytes, out.desc, pool.data_ptr(), pool_bytes, flags, ws.ptr, ws.nbytes, ws.result_ptr,
                   opts, bs.current_stream())
    return out, pool, ws.read_result()


def test_golden_align8_stream_from_the_gpu():
    from tests.test_oracle_golden import golden_set
    gold = read_hex_fixture(os.path.join(os.path.dirname(__file__), "golden", "g7_golden_stream_align8.hex"))
    tensors, qn, dim, blocks = golden_set()
    raw = np.zeros(2 * 64, np.uint8)
    raw[0:8] = blocks[0].view(np.uint8)
    raw[64:80] = blocks[1].view(np.uint8)
    d_pool = torch.from_numpy(raw).to(DEV)
    addr = np.array([d_pool.data_ptr(), d_pool.data_ptr() + 64], np.uint64)
    dset = bs.DeviceSet.from_host(tensors, qn, dim, addr, DEV, dtype=bs.F64 | bs.ALIGN8)
    out, res = serialize(dset, 1024)
    assert res["status"] == bs.OK and res["total_bytes"] == 280 and res["dtype"] == (bs.F64 | bs.ALIGN8), res
    got = out.cpu().numpy()
    assert got[:280].tobytes() == gold and (got[280:] == 0xCD).all()
    assert bs.stream_info(gold)["align"] == 8
    o, pool, res = deserialize(out, 280, 1, 2, 512)
    ref = oracle.deserialize(np.frombuffer(gold, np.uint8))
    assert res["status"] == bs.OK and res["dtype"] == (bs.F64 | bs.ALIGN8) and (pool.cpu().numpy()[:512] == ref["pool"][:512]).all()


@pytest.mark.parametrize("opts", SHAPES, ids=lambda o: "default" if o is None else "-".join(f"{k[0]}{v}" for k, v in o.items()))
def test_unpadded_stream_and_round_trip_match_the_oracle(opts):
    for bset in sets():
        up = Uploaded(bset)
        want = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs), align=8)
        total = len(want)
        dset = a8_set(up)
        ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total + 4096, DEV)
        assert bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, bs.current_stream()) == oracle.serialized_size(bset.n_tensors, bset.dim, align=8)
        for cap in (total, total + 4096):          # an exact capacity (the total may be 8 off a multiple of 16) and a loose one
            out, res = serialize(dset, cap, opts)
            assert res["status"] == bs.OK and res["total_bytes"] == total, (bset.name, res)
            got = out.cpu().numpy()
            bad = np.nonzero(got[:total] != want)[0]
            assert bad.size == 0, f"{bset.name}: first mismatch at stream byte {bad[0]} of {total}, opts={opts}"
            assert (got[total:] == 0xCD).all(), "bytes beyond the stream were written"
        ref = oracle.deserialize(want)
        need = oracle.pool_bytes(want)
        o, pool, res = deserialize(out, total, bset.n_tensors, bset.n_blocks, need, opts)
        assert res["status"] == bs.OK and res["pool_bytes"] == need and res["dtype"] & bs.ALIGN8, (bset.name, res)
        assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        h = o.to_host()
        assert h["tensors"].tobytes() == bset.tensors.tobytes() and (h["qn"] == bset.qn).all() and (h["dim"] == bset.dim).all()
        # fixpoint on the device, and the padded stream of the same object is the oracle's padded stream
        o.dtype = bs.F64 | bs.ALIGN8
        again, res = serialize(o, total, opts)
        assert res["status"] == bs.OK and (again.cpu().numpy()[:total] == want).all()
        o.dtype = bs.F64
        want16 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs))
        padded, res = serialize(o, len(want16), opts)
        assert res["status"] == bs.OK and (padded.cpu().numpy()[:len(want16)] == want16).all()


@pytest.mark.parametrize("dtype", [bs.F32, bs.C64, bs.C128], ids=["f32", "c64", "c128"])
def test_other_element_types_unpadded(dtype):
    e = {bs.F32: 4, bs.C64: 8, bs.C128: 16}[dtype]
    for bset in (W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial"),
                 W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)):
        pool, offs = W.fill_pool_host(bset)
        if e == 16:
            big = np.zeros(2 * pool.size + 2, np.float64)
            offs = offs * 2
            for o, n in zip(offs, bset.nelems):
                big[int(o) // 8: int(o) // 8 + 2 * int(n)] = np.repeat(pool[int(o) // 16: int(o) // 16 + int(n)], 2)
            pool = big
        raw = pool.view(np.uint8)
        blocks = [raw[int(o): int(o) + e * int(n)] for o, n in zip(offs, bset.nelems)]
        want = dt.serialize(bset.tensors, bset.qn, bset.dim, blocks, dtype, align=8)
        up = Uploaded(bset, pool, offs)
        for opts in (None, dict(variant=bs.VARIANT_TMA, fuse=1), dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=3, warps=2)):
            out, res = serialize(a8_set(up, dtype), len(want), opts)
            assert res["status"] == bs.OK and res["total_bytes"] == len(want) and res["dtype"] == (dtype | bs.ALIGN8), res
            got = out.cpu().numpy()
            bad = np.nonzero(got[:len(want)] != want)[0]
            assert bad.size == 0, f"first mismatch at stream byte {bad[0]}"
            ref = dt.deserialize(want)
            o, pl, res = deserialize(out, len(want), bset.n_tensors, bset.n_blocks, ref["pool_bytes"], opts)
            assert res["status"] == bs.OK and (pl.cpu().numpy()[:ref["pool_bytes"]] == ref["pool"][:ref["pool_bytes"]]).all()


def test_eight_byte_aligned_sources_ranges_scatter_and_capture():
    bset = W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)
    cs = bs.current_stream()
    up = Uploaded(bset, misalign=8)          # every source 8 off the grid: now the blocks at odd-8 stream offsets are the aligned ones
    want = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs), align=8)
    total = len(want)
    out, res = serialize(a8_set(up), total)
    assert res["status"] == bs.OK and (out.cpu().numpy()[:total] == want).all()
    up = Uploaded(bset)
    dset = a8_set(up)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    # concat(ranges) == the stream: cuts on the 16-byte grid, the last range ends at the total
    for chunk in (4096, 100000 * 16, 1 << 20):
        got = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
        cuts = list(range(0, total, chunk)) + [(total + 15) // 16 * 16]
        for k, (lo, hi) in enumerate(zip(cuts[:-1], cuts[1:])):
            seg = torch.full((hi - lo + 32,), 0x77, dtype=torch.uint8, device=DEV)
            bs.serialize_range(dset.desc, seg.data_ptr(), lo, hi, k == 0, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
            n = min(hi, total) - lo
            assert (seg[n:] == 0x77).all(), "range call wrote beyond its segment"
            got[lo:lo + n] = seg[:n]
        assert ws.read_result()["status"] == bs.OK and (got.cpu().numpy() == want).all()
    # scatter to caller addresses, 16-byte-aligned and 8-byte-aligned destinations
    st = torch.from_numpy(want.copy()).to(DEV)
    for shift in (0, 8):
        dst = torch.full((up.pool.numel() + 64,), 0xEE, dtype=torch.uint8, device=DEV)
        daddr = (np.uint64(dst.data_ptr() + shift) + up.host_offs).astype(np.uint64)
        o = bs.DeviceSet.from_host(np.zeros(bset.n_tensors, W.TENSOR_REC_DTYPE), np.zeros_like(bset.qn), bset.dim, daddr, DEV)
        _, _, res = deserialize(st, total, bset.n_tensors, bset.n_blocks, 0, flags=bs.SCATTER_TO_ADDR, out=o)
        assert res["status"] == bs.OK
        gotp = dst.cpu().numpy()
        expect = np.full_like(gotp, 0xEE)
        src = up.host_pool.view(np.uint8)
        for i in range(bset.n_blocks):
            a, n = int(up.host_offs[i]), int(bset.nelems[i]) * 8
            expect[shift + a: shift + a + n] = src[a:a + n]
        assert (gotp == expect).all()


def test_engine_queue_and_packages_carry_unpadded_streams():
    bset = W.make_config("2", n_ops=52)
    up = Uploaded(bset)
    want = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs), align=8)
    total = len(want)
    dset = a8_set(up)
    cs = bs.current_stream()
    ref = oracle.deserialize(want)
    need = oracle.pool_bytes(want)
    for chunk, n_st in ((65536, 2), (5 * 65536, 1), (1 << 28, 2)):
        eng = bs.Engine(bset.n_tensors, bset.n_blocks, total + 4096, chunk_bytes=chunk, n_staging=n_st)
        host = torch.empty(total + 4096, dtype=torch.uint8, pin_memory=True)
        host.fill_(0x5A)
        for tb in (total, 0):                          # the predicted size, and "compute it"
            st = eng.offload_async(dset.desc, tb, host.data_ptr(), host.numel(), cs).wait()
            assert st["status"] == bs.OK and st["bytes"] == total
            assert (host.numpy()[:total] == want).all() and (host.numpy()[total:] == 0x5A).all()
        out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
        pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
        st = eng.prefetch_async(host.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs).wait()
        torch.cuda.synchronize()
        assert st["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        eng.destroy()
    q = bs.Queue(bset.n_tensors, bset.n_blocks, total, chunk_bytes=4 * 65536)
    host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    q.save(3, dset.desc, total, host.data_ptr(), total, cs)
    q.load(3, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)
    assert q.wait(3)["status"] == bs.OK
    torch.cuda.synchronize()
    assert (host.numpy() == want).all() and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
    q.destroy()
    from oracle import pkg
    hb = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
    for cap in (32768, 4096 + 16):
        n = pkg.count(hb, total, cap)
        slots = torch.full((n * (64 + cap),), 0x5A, dtype=torch.uint8, device=DEV)
        wsp = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV, packages=True)
        bs.package_emit(dset.desc, total, cap, 9, slots.data_ptr(), 64 + cap, n, None, wsp.ptr, wsp.nbytes, wsp.result_ptr, None, cs)
        assert wsp.read_result()["status"] == bs.OK
        assert (slots.cpu().numpy().reshape(n, -1) == pkg.emit_slots(want, cap, 9, 64 + cap, poison=0x5A)).all(), "packages differ"
        pool.fill_(0xEE)
        bs.package_unpack(slots.data_ptr(), 64 + cap, n, 9, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, wsp.ptr, wsp.nbytes,
                          wsp.result_ptr, None, cs)
        assert wsp.read_result()["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


def test_what_is_refused():
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    up = Uploaded(bset)
    want = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs), align=8)
    dset = a8_set(up)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, 1 << 20, DEV)
    out = torch.full((1 << 20,), 0xCD, dtype=torch.uint8, device=DEV)
    with pytest.raises(bs.BsError) as e:          # the LDG variant moves 16-byte units
        bs.serialize(dset.desc, out.data_ptr(), 1 << 20, ws.ptr, ws.nbytes, ws.result_ptr, dict(variant=bs.VARIANT_LDG), bs.current_stream())
    assert e.value.code == bs.ERR_UNSUPPORTED
    st = torch.from_numpy(want.copy()).to(DEV)
    need = oracle.pool_bytes(want)
    o, pool, res = deserialize(st, len(want), bset.n_tensors, bset.n_blocks, need, dict(variant=bs.VARIANT_LDG))
    assert res["status"] == bs.ERR_UNSUPPORTED and (pool == 0xEE).all()
    # a range call with the LDG variant on tables a TMA-variant pass parsed from an unpadded stream: nothing is written
    # (it used to scatter 16-byte units with status OK), and the workspace refuses every later range call too
    o2 = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool2 = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.deserialize(st.data_ptr(), len(want), o2.desc, pool2.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr, None,
                   bs.current_stream())
    assert ws.read_result()["status"] == bs.OK and (pool2.cpu().numpy() == oracle.deserialize(want)["pool"][:need]).all()
    pool2.fill_(0xEE)
    for variant in (dict(variant=bs.VARIANT_LDG, tile_bytes=16384), None):
        bs.deserialize_range(st.data_ptr(), 0, len(want), 0, o2.desc, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, variant, bs.current_stream())
        torch.cuda.synchronize()
        assert (pool2 == 0xEE).all()
    bad_flag = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, up.addr, DEV, dtype=bs.F64 | 0x400)
    with pytest.raises(bs.BsError) as e:
        bs.serialize(bad_flag.desc, out.data_ptr(), 1 << 20, ws.ptr, ws.nbytes, ws.result_ptr, None, bs.current_stream())
    assert e.value.code == bs.ERR_UNSUPPORTED
    lv = W.layered_view(bset)
    ls = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], up.addr, DEV, dtype=bs.F64 | bs.ALIGN8)
    wl = bs.Workspace(0, 0, 1 << 20, DEV, layered=(len(lv["structs"]), lv["dim"].shape[0], bset.n_tensors, bset.n_blocks))
    with pytest.raises(bs.BsError) as e:          # layered sets keep align 16
        bs.layered_serialize(ls.desc, out.data_ptr(), 1 << 20, wl.ptr, wl.nbytes, wl.result_ptr, None, bs.current_stream())
    assert e.value.code == bs.ERR_UNSUPPORTED
    # corrupt unpadded streams: the align word, an offset, the payload size, a truncated stream
    for pos, xor in ((0x1C, 0x18), (0x1C, 4), (64 + 32 * bset.n_tensors + 48 * 3 + 40, 8), (0x38, 8)):
        bad = want.copy()
        bad[pos] ^= xor
        assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
        o, pool, res = deserialize(torch.from_numpy(bad).to(DEV), len(bad), bset.n_tensors, bset.n_blocks, need)
        assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all(), (pos, res)
    o, pool, res = deserialize(st, len(want) - 8, bset.n_tensors, bset.n_blocks, need)
    assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all()
