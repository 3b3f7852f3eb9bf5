"""NEXT-4 on the GPU: element types f32 / c64 / c128 (bs_set_desc.dtype) through the C ABI against
oracle/bs_oracle_dtype.py — bit-exact streams and round trips; the type only changes how many bytes a block has, so f32
blocks exercise pads of 4, 8 and 12 bytes in every kernel variant."""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from oracle import dt
from tests.gpu_util import DEV
from tests.util import read_hex_fixture

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(__file__)
DTYPES = [(dt.F32, "f32"), (dt.C64, "c64"), (dt.C128, "c128"), (dt.F64, "f64")]
VARIANTS = [dict(variant=bs.VARIANT_TMA), dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_LDG, tile_bytes=32768),
            dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=3, warps=2)]


class RawSet:
    """Labels / extents of a workloads set, blocks of seeded random BYTES of the given element type, uploaded."""

    def __init__(self, bset, dtype, seed, misalign=0):
        e = dt.ELEM_BYTES[dtype]
        rng = np.random.default_rng(seed)
        self.bset, self.dtype = bset, dtype
        self.blocks = [rng.integers(0, 256, e * int(n), dtype=np.uint8).tobytes() for n in bset.nelems]
        order = rng.permutation(bset.n_blocks)                    # scattered placement, 512-byte slots
        offs = np.zeros(bset.n_blocks, np.uint64)
        cur = 0
        for i in order:
            offs[i] = cur + misalign
            cur += (len(self.blocks[i]) + misalign + 511) // 512 * 512
        host = np.full(max(cur, 512), 0x33, np.uint8)
        for b, o in zip(self.blocks, offs):
            host[int(o): int(o) + len(b)] = np.frombuffer(b, np.uint8)
        self.pool = torch.from_numpy(host).to(DEV)
        addr = (np.uint64(self.pool.data_ptr()) + offs).astype(np.uint64)
        self.dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, addr, DEV, dtype=dtype)
        self.want = dt.serialize(bset.tensors, bset.qn, bset.dim, self.blocks, dtype)


def small(name="dt", seed=77, **kw):
    a = dict(D=60, S=9, M=2, N0=3, n_ops=9, n_site=1, dims="multinomial")
    a.update(kw)
    return W.make_set(name, seed, **a)


def serialize_on_gpu(rs, opts=None, capacity=None):
    total = len(rs.want) if capacity is None else capacity
    ws = bs.Workspace(rs.bset.n_tensors, rs.bset.n_blocks, max(total, 1 << 16), DEV)
    out = torch.full((total + 64,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.serialize(rs.dset.desc, out.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    return out, ws.read_result(), ws


def deserialize_on_gpu(stream_t, nbytes, bset, need, opts=None):
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((max(need, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, max(nbytes, 1 << 16), DEV)
    bs.deserialize(stream_t.data_ptr(), nbytes, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                   ws.result_ptr, opts, bs.current_stream())
    return out, pool, ws.read_result()


def test_golden_f32_stream_from_the_gpu():
    gold = read_hex_fixture(os.path.join(HERE, "golden", "g4_golden_stream_f32.hex"))
    tensors = np.zeros(1, W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 2, (0, 0), (-1, 1, 0, 0), 9, 0)
    qn = np.array([[[0, 0], [0, 0], [0, 0]], [[1, 1], [1, 1], [0, 0]]], np.int32)
    dim = np.array([[1, 3, 1], [1, 1, 1]], np.uint32)
    host = np.zeros(1024, np.uint8)
    host[0:12] = np.frombuffer(np.array([1.0, 2.0, 3.0], np.float32).tobytes(), np.uint8)
    host[512:516] = np.frombuffer(np.array([-1.0], np.float32).tobytes(), np.uint8)
    host[12:16] = 0x77                                            # what lies behind a block must not reach the stream
    pool = torch.from_numpy(host).to(DEV)
    addr = (np.uint64(pool.data_ptr()) + np.array([0, 512], np.uint64)).astype(np.uint64)
    dset = bs.DeviceSet.from_host(tensors, qn, dim, addr, DEV, dtype=bs.F32)
    for opts in VARIANTS[:2]:
        ws = bs.Workspace(1, 2, 1 << 16, DEV)
        out = torch.full((288,), 0xCD, dtype=torch.uint8, device=DEV)
        bs.serialize(dset.desc, out.data_ptr(), 288, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
        assert ws.read_result()["status"] == bs.OK
        assert bytes(out.cpu().numpy()) == gold
    assert bs.stream_info(gold)["dtype"] == bs.F32


@pytest.mark.parametrize("dtype,name", DTYPES, ids=[n for _, n in DTYPES])
@pytest.mark.parametrize("opts", VARIANTS, ids=lambda o: f"v{o['variant']}t{o.get('tile_bytes', 0)}")
def test_serialize_and_round_trip_match_the_oracle(dtype, name, opts):
    rs = RawSet(small(), dtype, seed=5 + dtype)
    out, res, _ = serialize_on_gpu(rs, opts)
    total = len(rs.want)
    assert res["status"] == bs.OK and res["total_bytes"] == total
    got = out.cpu().numpy()
    assert (got[:total] == rs.want).all(), "stream differs from the oracle's"
    assert (got[total:] == 0xCD).all()
    ref = dt.deserialize(rs.want)
    o, pool, res2 = deserialize_on_gpu(out, total, rs.bset, ref["pool_bytes"], opts)
    assert res2["status"] == bs.OK and res2["pool_bytes"] == ref["pool_bytes"] and res2["dtype"] == dtype
    assert (pool.cpu().numpy()[:ref["pool_bytes"]] == ref["pool"][:ref["pool_bytes"]]).all(), "blocks differ (or gaps were written)"
    h = o.to_host()
    assert h["tensors"].tobytes() == rs.bset.tensors.tobytes() and (h["qn"] == rs.bset.qn).all() and (h["dim"] == rs.bset.dim).all()


@pytest.mark.parametrize("dtype,name", DTYPES[:3], ids=[n for _, n in DTYPES[:3]])
def test_many_tiles_ragged_tails_and_eight_byte_aligned_sources(dtype, name):
    bset = small("dt2", 78, D=400, S=25, n_ops=26, n_site=2)                    # ~MBs: many tiles, thousands of blocks
    for misalign in (0, 8):
        rs = RawSet(bset, dtype, seed=9, misalign=misalign)
        for opts in VARIANTS[:2]:
            out, res, _ = serialize_on_gpu(rs, opts)
            assert res["status"] == bs.OK
            assert (out.cpu().numpy()[:len(rs.want)] == rs.want).all(), (name, misalign, opts)
    ref = dt.deserialize(rs.want)
    o, pool, res2 = deserialize_on_gpu(out, len(rs.want), bset, ref["pool_bytes"])
    assert res2["status"] == bs.OK and (pool.cpu().numpy()[:ref["pool_bytes"]] == ref["pool"][:ref["pool_bytes"]]).all()


@pytest.mark.parametrize("chunk", [16, 4096, 100000 * 16])
def test_concat_of_ranges_is_the_stream_f32(chunk):
    rs = RawSet(small(), dt.F32, seed=3)
    total = len(rs.want)
    ws = bs.Workspace(rs.bset.n_tensors, rs.bset.n_blocks, max(total, 1 << 16), DEV)
    got = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    first = True
    step = chunk if chunk > 16 else 4096 + 16
    for lo in range(0, total, step):
        hi = min(lo + step, total)
        bs.serialize_range(rs.dset.desc, got.data_ptr() + lo, lo, hi, first, ws.ptr, ws.nbytes, ws.result_ptr, None,
                           bs.current_stream())
        first = False
    assert ws.read_result()["status"] == bs.OK and (got.cpu().numpy() == rs.want).all()


def test_engine_and_packages_carry_the_element_type():
    rs = RawSet(small("dt3", 79, D=200, S=15, n_ops=13), dt.F32, seed=11)
    total = len(rs.want)
    ref = dt.deserialize(rs.want)
    need = ref["pool_bytes"]
    eng = bs.Engine(rs.bset.n_tensors, rs.bset.n_blocks, total, chunk_bytes=65536)
    host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
    host.fill_(0xCD)
    assert eng.offload_async(rs.dset.desc, total, host.data_ptr(), total, bs.current_stream()).wait()["status"] == bs.OK
    assert (host.numpy() == rs.want).all()
    out = bs.DeviceSet.empty(rs.bset.n_tensors, rs.bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    t = eng.prefetch_async(host.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, bs.current_stream())
    assert t.wait()["status"] == bs.OK
    torch.cuda.synchronize()
    assert (pool.cpu().numpy() == ref["pool"][:need]).all()
    eng.destroy()
    # packages: the oracle's cut of the oracle's f32 stream
    from oracle import pkg
    cap = 32768
    hb = bs.header_bytes(rs.bset.n_tensors, rs.bset.n_blocks)
    n = pkg.count(hb, total, cap)
    slots = torch.full((n * (64 + cap),), 0x5A, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(rs.bset.n_tensors, rs.bset.n_blocks, total, DEV, packages=True)
    bs.package_emit(rs.dset.desc, total, cap, 9, slots.data_ptr(), 64 + cap, n, None, ws.ptr, ws.nbytes, ws.result_ptr, None,
                    bs.current_stream())
    assert ws.read_result()["status"] == bs.OK
    assert (slots.cpu().numpy().reshape(n, -1) == pkg.emit_slots(rs.want, cap, 9, 64 + cap, poison=0x5A)).all()
    pool.fill_(0xEE)
    bs.package_unpack(slots.data_ptr(), 64 + cap, n, 9, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                      ws.result_ptr, None, bs.current_stream())
    assert ws.read_result()["status"] == bs.OK and (pool.cpu().numpy() == ref["pool"][:need]).all()


def test_bad_element_types_and_nonzero_pad_are_rejected():
    rs = RawSet(small(), dt.F32, seed=2)
    total = len(rs.want)
    d = rs.dset.desc
    d.dtype = 4
    with pytest.raises(bs.BsError) as e:
        bs.serialize(d, 256, total, 256, 1 << 20, 0)
    assert e.value.code == bs.ERR_UNSUPPORTED
    ref = dt.deserialize(rs.want)
    nbytes, stored, offset, P = dt.plan(rs.bset.dim, dt.F32)
    hb = dt.header_bytes(rs.bset.n_tensors, rs.bset.n_blocks)
    cases = [(16, 4)]                                            # the dtype word itself
    for pad in (4, 8, 12):                                       # one byte of pad of a block with that much pad
        i = next(k for k in range(len(nbytes)) if stored[k] - nbytes[k] == pad)
        cases.append((hb + offset[i] + stored[i] - 1, 1))
    for pos, flip in cases:
        bad = rs.want.copy()
        bad[pos] ^= flip
        with pytest.raises(oracle.OracleError):
            dt.deserialize(bad)
        st = torch.from_numpy(bad).to(DEV)
        o, pool, res = deserialize_on_gpu(st, total, rs.bset, ref["pool_bytes"])
        assert res["status"] == bs.ERR_CORRUPT, (pos, res)
        assert (pool.cpu().numpy() == 0xEE).all() and (o.tensors.cpu().numpy() == 0xAB).all()
    # layered sets (wire format v2) carry the same four types (tests/test_gpu_layered.py); anything else is refused at once
    lv = W.layered_view(rs.bset)
    ls = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], np.zeros(rs.bset.n_blocks, np.uint64), DEV)
    ld = ls.desc
    ld.dtype = 4
    with pytest.raises(bs.BsError) as e:
        bs.layered_serialize(ld, 256, 1 << 20, 256, 1 << 24, 0)
    assert e.value.code == bs.ERR_UNSUPPORTED
