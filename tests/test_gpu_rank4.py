"""Tensors of rank up to 4 on the GPU (bs.h BS_RANK4, wire format v3; DESIGN.md §19 reading D20) through
the C ABI against oracle/bs_oracle_v3.c.  Bit-exact.  Every test needs a GPU."""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from oracle import v3
from tests.gpu_util import DEV
from tests.util import host_addrs, read_hex_fixture

pytestmark = pytest.mark.gpu

SHAPES = [None, dict(variant=bs.VARIANT_TMA, fuse=1), dict(variant=bs.VARIANT_TMA, fuse=2), dict(variant=bs.VARIANT_LDG),
          dict(variant=bs.VARIANT_LDG, tile_bytes=65536), dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=4, warps=1)]
ELEM = {bs.F64: 8, bs.F32: 4, bs.C128: 16}


def tree_sets():
    return [W.make_tree_set("tree-small", 5), W.make_tree_set("tree", 7, D=40, S=8, n_nodes=4, n_ops=5),
            W.make_tree_set("tree-big", 8, D=96, S=10, n_nodes=6, n_ops=13)]


class Up4:
    def __init__(self, bset, dtype=bs.F64, misalign=0):
        pool, offs = W.fill_pool_host(bset)
        if ELEM[dtype] == 16:
            pool = np.concatenate([pool, pool])      # room to read 16-byte elements; the values are arbitrary bits
        self.bset, self.dtype, self.host_pool, self.host_offs = bset, dtype, pool, offs
        raw = torch.from_numpy(pool.view(np.uint8).copy())
        buf = torch.zeros(raw.numel() + 64, dtype=torch.uint8, device=DEV)
        buf[misalign:misalign + raw.numel()] = raw.to(DEV)
        self.pool = buf
        self.addr = (np.uint64(buf.data_ptr() + misalign) + offs.astype(np.uint64)).astype(np.uint64)
        self.dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, self.addr, DEV, dtype=dtype | bs.RANK4)
        self.want = v3.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs), dtype)


def serialize(dset, capacity, opts=None):
    out = torch.full((max(capacity, 16),), 0xCD, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(dset.n_tensors, dset.n_blocks, max(capacity, 1 << 16), DEV)
    bs.serialize(dset.desc, out.data_ptr(), capacity, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    return out, ws.read_result()


def deserialize(stream_t, nbytes, cap_t, cap_b, pool_bytes, opts=None, flags=bs.LAYOUT_POOL, out=None, rank4=True):
    out = out or bs.DeviceSet.empty(cap_t, cap_b, DEV, fill=0xAB, rank4=rank4)
    pool = torch.full((max(pool_bytes, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(cap_t, cap_b, max(nbytes, 1 << 16), DEV)
    bs.deserialize(stream_t.data_ptr(), nbytes, out.desc, pool.data_ptr(), pool_bytes, flags, ws.ptr, ws.nbytes, ws.result_ptr,
                   opts, bs.current_stream())
    return out, pool, ws.read_result()


def test_golden_v3_stream_from_the_gpu():
    from tests.test_oracle_v3 import GOLD, golden_set
    gold = read_hex_fixture(GOLD)
    tensors, qn, dim, blocks = golden_set()
    raw = np.zeros(3 * 64, np.uint8)
    for k, b in enumerate(blocks):
        raw[64 * k: 64 * k + b.nbytes] = b.view(np.uint8)
    d_pool = torch.from_numpy(raw).to(DEV)
    addr = (np.uint64(d_pool.data_ptr()) + np.arange(3, dtype=np.uint64) * np.uint64(64)).astype(np.uint64)
    dset = bs.DeviceSet.from_host(tensors, qn, dim, addr, DEV, dtype=bs.F64 | bs.RANK4)
    out, res = serialize(dset, 1024)
    assert res["status"] == bs.OK and res["total_bytes"] == 448 and res["header_bytes"] == 384 and res["dtype"] == (bs.F64 | bs.RANK4), res
    got = out.cpu().numpy()
    assert got[:448].tobytes() == gold and (got[448:] == 0xCD).all()
    assert bs.stream_info(gold)["max_rank"] == 4
    o, pool, res = deserialize(out, 448, 2, 3, 768)
    ref = v3.deserialize(np.frombuffer(gold, np.uint8))
    assert res["status"] == bs.OK and res["dtype"] == (bs.F64 | bs.RANK4) and (pool.cpu().numpy()[:768] == ref["pool"][:768]).all()
    h = o.to_host()
    assert h["tensors"].tobytes() == tensors.tobytes() and (h["qn"] == qn).all() and (h["dim"] == dim).all()


@pytest.mark.parametrize("opts", SHAPES, ids=lambda o: "default" if o is None else "-".join(f"{k[0]}{v}" for k, v in o.items()))
def test_order_4_sets_match_the_oracle_and_round_trip(opts):
    for bset in tree_sets():
        up = Up4(bset)
        total = len(up.want)
        ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total + 4096, DEV)
        assert bs.serialized_size(up.dset.desc, ws.ptr, ws.nbytes, bs.current_stream()) == v3.serialized_size(bset.n_tensors, bset.dim)
        out, res = serialize(up.dset, total + 4096, opts)
        assert res["status"] == bs.OK and res["total_bytes"] == total and res["n_blocks"] == bset.n_blocks, (bset.name, res)
        got = out.cpu().numpy()
        bad = np.nonzero(got[:total] != up.want)[0]
        assert bad.size == 0, f"{bset.name}: first mismatch at stream byte {bad[0]} (header {res['header_bytes']}), opts={opts}"
        assert (got[total:] == 0xCD).all()
        ref = v3.deserialize(up.want)
        need = v3.pool_bytes(up.want)
        o, pool, res = deserialize(out, total, bset.n_tensors, bset.n_blocks, need, opts)
        assert res["status"] == bs.OK and res["pool_bytes"] == need and res["dtype"] & bs.RANK4, (bset.name, res)
        assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        h = o.to_host()
        assert h["tensors"].tobytes() == bset.tensors.tobytes() and (h["qn"] == bset.qn).all() and (h["dim"] == bset.dim).all()
        assert ((h["addr"] - np.uint64(pool.data_ptr())) == (ref["addr"] - np.uint64(ref["pool"].ctypes.data))).all()
        o.dtype = bs.F64 | bs.RANK4                      # fixpoint on the device
        again, res = serialize(o, total, opts)
        assert res["status"] == bs.OK and (again.cpu().numpy()[:total] == up.want).all()


@pytest.mark.parametrize("dtype", [bs.F32, bs.C128], ids=["f32", "c128"])
def test_other_element_types_eight_byte_sources_ranges_and_scatter(dtype):
    bset = W.make_tree_set("tree", 7, D=40, S=8, n_nodes=4, n_ops=5)
    cs = bs.current_stream()
    for mis in (0, 8):
        up = Up4(bset, dtype, misalign=mis)
        total = len(up.want)
        out, res = serialize(up.dset, total)
        assert res["status"] == bs.OK and res["dtype"] == (dtype | bs.RANK4) and (out.cpu().numpy()[:total] == up.want).all()
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    got = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    cuts = list(range(0, total, 50000 * 16)) + [total]
    for k, (lo, hi) in enumerate(zip(cuts[:-1], cuts[1:])):
        bs.serialize_range(up.dset.desc, got[lo:].data_ptr(), lo, hi, k == 0, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK and (got.cpu().numpy() == up.want).all()
    # scatter to caller addresses (extents given with four legs)
    e = ELEM[dtype]
    dst = torch.full((up.pool.numel(),), 0xEE, dtype=torch.uint8, device=DEV)
    daddr = (np.uint64(dst.data_ptr()) + up.host_offs).astype(np.uint64)
    o = bs.DeviceSet.from_host(np.zeros(bset.n_tensors, W.TENSOR_REC_DTYPE), np.zeros_like(bset.qn), bset.dim, daddr, DEV, dtype=bs.RANK4)
    _, _, res = deserialize(got, total, bset.n_tensors, bset.n_blocks, 0, flags=bs.SCATTER_TO_ADDR, out=o)
    assert res["status"] == bs.OK
    gotp = dst.cpu().numpy()
    src = up.host_pool.view(np.uint8)
    expect = np.full_like(gotp, 0xEE)
    for i in range(bset.n_blocks):
        a, n = int(up.host_offs[i]), int(bset.nelems[i]) * e
        expect[a:a + n] = src[a:a + n]
    assert (gotp == expect).all()
    wrong = bset.dim.copy()
    wrong[3, 3] += 1
    o = bs.DeviceSet.from_host(np.zeros(bset.n_tensors, W.TENSOR_REC_DTYPE), np.zeros_like(bset.qn), wrong, daddr, DEV, dtype=bs.RANK4)
    dst.fill_(0xEE)
    _, _, res = deserialize(got, total, bset.n_tensors, bset.n_blocks, 0, flags=bs.SCATTER_TO_ADDR, out=o)
    assert res["status"] == bs.ERR_ARG and (dst == 0xEE).all()


def test_engine_queue_and_packages_carry_order_4_sets():
    bset = W.make_tree_set("tree-big", 8, D=96, S=10, n_nodes=6, n_ops=13)
    up = Up4(bset)
    total = len(up.want)
    cs = bs.current_stream()
    ref = v3.deserialize(up.want)
    need = v3.pool_bytes(up.want)
    for chunk, n_st in ((65536, 2), (1 << 28, 2)):
        eng = bs.Engine(bset.n_tensors, bset.n_blocks, total + 4096, chunk_bytes=chunk, n_staging=n_st)
        host = torch.empty(total + 4096, dtype=torch.uint8, pin_memory=True)
        host.fill_(0x5A)
        for tb in (total, 0):
            st = eng.offload_async(up.dset.desc, tb, host.data_ptr(), host.numel(), cs).wait()
            assert st["status"] == bs.OK and st["bytes"] == total
            assert (host.numpy()[:total] == up.want).all() and (host.numpy()[total:] == 0x5A).all()
        out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB, rank4=True)
        pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
        st = eng.prefetch_async(host.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs).wait()
        torch.cuda.synchronize()
        assert st["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        assert (out.to_host()["dim"] == bset.dim).all()
        flat = bs.DeviceSet.empty(bset.n_tensors, 2 * bset.n_blocks, DEV, fill=0xAB)     # three-leg arrays cannot take the stream
        with pytest.raises(bs.BsError) as e:
            eng.prefetch_async(host.data_ptr(), total, flat.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)
        assert e.value.code == bs.ERR_ARG
        eng.destroy()
    q = bs.Queue(bset.n_tensors, bset.n_blocks, total, chunk_bytes=4 * 65536)
    host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB, rank4=True)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    q.save(4, up.dset.desc, total, host.data_ptr(), total, cs)
    q.load(4, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)          # submitted behind the save: counts remembered
    assert q.wait(4)["status"] == bs.OK
    torch.cuda.synchronize()
    assert (host.numpy() == up.want).all() and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
    q.destroy()
    from oracle import pkg
    hb = v3.header_bytes(bset.n_tensors, bset.n_blocks)
    for cap in (32768, 4096 + 16):
        n = pkg.count(hb, total, cap)
        slots = torch.full((n * (64 + cap),), 0x5A, dtype=torch.uint8, device=DEV)
        wsp = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV, packages=True)
        bs.package_emit(up.dset.desc, total, cap, 9, slots.data_ptr(), 64 + cap, n, None, wsp.ptr, wsp.nbytes, wsp.result_ptr, None, cs)
        assert wsp.read_result()["status"] == bs.OK
        got = slots.cpu().numpy().reshape(n, -1)
        # package k = 64-byte header | stream bytes [lo, hi) of the oracle's cut
        for k in range(n):
            lo, hi = pkg.package_range(hb, total, cap, k)
            assert (got[k, 64:64 + hi - lo] == up.want[lo:hi]).all() and (got[k, 64 + hi - lo:] == 0x5A).all(), f"package {k}"
        pool.fill_(0xEE)
        bs.package_unpack(slots.data_ptr(), 64 + cap, n, 9, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, wsp.ptr, wsp.nbytes,
                          wsp.result_ptr, None, cs)
        assert wsp.read_result()["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


def test_what_is_refused():
    bset = W.make_tree_set("fault", 9, D=12, S=4, n_nodes=2, n_ops=3)
    up = Up4(bset)
    total = len(up.want)
    need = v3.pool_bytes(up.want)
    st = torch.from_numpy(up.want.copy()).to(DEV)
    # a v3 stream into three-leg arrays, a v1 stream into four-leg arrays
    o, pool, res = deserialize(st, total, bset.n_tensors, 2 * bset.n_blocks, need, rank4=False)
    assert res["status"] == bs.ERR_ARG and (pool == 0xEE).all()
    flat = W.make_config("1")
    fp, fo = W.fill_pool_host(flat)
    s1 = oracle.serialize(flat.tensors, flat.qn, flat.dim, host_addrs(fp, fo))
    o, pool, res = deserialize(torch.from_numpy(s1.copy()).to(DEV), len(s1), 4, 64, 1 << 16, rank4=True)
    assert res["status"] == bs.ERR_ARG and (pool == 0xEE).all()
    # rank 5; RANK4 | ALIGN8; layered sets
    t = bset.tensors.copy()
    t["rank"][0] = 5
    d = bs.DeviceSet.from_host(t, bset.qn, bset.dim, up.addr, DEV, dtype=bs.RANK4)
    out, res = serialize(d, 1 << 20)
    assert res["status"] == bs.ERR_UNSUPPORTED and (out == 0xCD).all()
    d = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, up.addr, DEV, dtype=bs.RANK4 | bs.ALIGN8)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, 1 << 20, DEV)
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d.desc, st.data_ptr(), 1 << 20, ws.ptr, ws.nbytes, ws.result_ptr, None, bs.current_stream())
    assert e.value.code == bs.ERR_UNSUPPORTED
    # corrupt v3 streams: every kind of field the oracle refuses
    T, B = bset.n_tensors, bset.n_blocks
    b0 = 64 + 32 * T
    r2 = int(np.nonzero(bset.tensors["rank"] == 2)[0][0])
    fb2 = int(bset.tensors["first_block"][r2])
    for name, pos, xor in (("version", 8, 2), ("max_rank", 24, 1), ("align", 28, 0x18), ("header_bytes", 48, 128), ("rank", 64, 1),
                           ("owner", b0 + 48, 1), ("b_reserved", b0 + 52, 1), ("offset_k", b0 + 64 * (B // 2) + 56, 16),
                           ("dim_leg4", b0 + 64 + 44, 1), ("unused_dim_of_rank2", b0 + 64 * fb2 + 40, 2),
                           ("unused_leg4_of_rank2", b0 + 64 * fb2 + 44, 3), ("unused_qn_of_rank2", b0 + 64 * fb2 + 28, 1)):
        bad = up.want.copy()
        bad[pos] ^= xor
        assert v3.validate_stream(bad) == oracle.ERR_CORRUPT, name
        o, pool, res = deserialize(torch.from_numpy(bad).to(DEV), len(bad), T, B, need)
        assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all(), (name, res)
        assert (o.qn == 0xAB).all() and (o.dim == 0xAB).all()
