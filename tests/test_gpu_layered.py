"""Parity of the CUDA path for wire format v2 (structure-shared layers) with the v2 oracle:
bit-exact, through the C ABI.  Every test needs a GPU."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from oracle import v2
from tests.gpu_util import DEV, Uploaded
from tests.util import host_addrs

pytestmark = pytest.mark.gpu

VARIANTS = [None, dict(variant=bs.VARIANT_LDG, tile_bytes=16384), dict(variant=bs.VARIANT_LDG, tile_bytes=65536, ctas_per_sm=1),
            dict(variant=bs.VARIANT_TMA, tile_bytes=32768), dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=4, warps=1)]


def small_sets():
    return [W.make_config("1"), W.make_config("2"),
            W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial"),
            W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0),
            W.make_set("few-ops", 13, D=64, S=12, M=2, N0=2, n_ops=5, n_site=1, dims="multinomial")]


class LayeredUp:
    """A set uploaded once; its layered descriptor shares the pool and addresses of the flat one."""

    def __init__(self, bset, keep_unused=False, misalign=0):
        self.bset = bset
        self.up = Uploaded(bset, misalign=misalign)
        self.lv = W.layered_view(bset, keep_unused=keep_unused)
        lv = self.lv
        self.dset = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], self.up.addr, DEV)
        self.want = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(self.up.host_pool, self.up.host_offs))
        self.counts = (len(lv["structs"]), lv["dim"].shape[0], len(lv["layers"]), bset.n_blocks)

    def workspace(self, cap):
        return bs.Workspace(0, 0, max(cap, 1 << 16), DEV, layered=self.counts)


def gpu_lserialize(lu, capacity, opts=None, poison=0xCD, dset=None):
    out = torch.full((max(capacity, 16),), poison, dtype=torch.uint8, device=DEV)
    ws = lu.workspace(capacity)
    bs.layered_serialize((dset or lu.dset).desc, out.data_ptr(), capacity, ws.ptr, ws.nbytes, ws.result_ptr, opts,
                         bs.current_stream())
    return out, ws.read_result()


def gpu_ldeserialize(stream_t, nbytes, caps, pool_bytes, flags=bs.LAYOUT_POOL, opts=None, out=None, poison=0xEE):
    if out is None:
        out = bs.DeviceLayeredSet.empty(*caps, DEV, fill=0xAB)
    pool = torch.full((max(pool_bytes, 256),), poison, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(0, 0, max(nbytes, 1 << 16), DEV, layered=caps)
    bs.layered_deserialize(stream_t.data_ptr(), nbytes, out.desc, pool.data_ptr(), pool_bytes, flags, ws.ptr, ws.nbytes,
                           ws.result_ptr, opts, bs.current_stream())
    return out, pool, ws.read_result()


def check_stream(lu, opts=None, slack=4096):
    want = lu.want
    total = len(want)
    got_t, res = gpu_lserialize(lu, total + slack, opts)
    assert res["status"] == bs.OK, res
    hb, tot = v2.serialized_size(lu.lv["structs"], lu.lv["layers"], lu.lv["dim"])
    assert (res["header_bytes"], res["total_bytes"], res["payload_bytes"]) == (hb, tot, tot - hb)
    assert (res["n_structs"], res["n_struct_blocks"], res["n_tensors"], res["n_blocks"]) == lu.counts
    got = got_t.cpu().numpy()
    bad = np.nonzero(got[:total] != want)[0]
    assert bad.size == 0, f"first mismatch at stream byte {bad[0]} (header_bytes={hb}), opts={opts}"
    assert (got[total:] == 0xCD).all(), "bytes beyond the stream were written"
    return got_t


@pytest.mark.parametrize("keep_unused", [False, True])
@pytest.mark.parametrize("bset", small_sets(), ids=lambda s: s.name)
def test_serialize_matches_oracle_byte_for_byte(bset, keep_unused):
    check_stream(LayeredUp(bset, keep_unused))


@pytest.mark.parametrize("opts", VARIANTS, ids=lambda o: "default" if o is None else f"v{o['variant']}-t{o.get('tile_bytes')}")
def test_stream_independent_of_decomposition(opts):
    for bset in (W.make_config("2"), W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2,
                                                dims="lognormal", sigma=1.0)):
        check_stream(LayeredUp(bset), opts)


def test_payload_is_the_v1_payload_and_header_is_smaller():
    bset = W.make_config("2")
    lu = LayeredUp(bset)
    got2 = check_stream(lu).cpu().numpy()[:len(lu.want)]
    want1 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(lu.up.host_pool, lu.up.host_offs))
    h1, h2 = oracle.stream_info(want1)["header_bytes"], v2.stream_info(lu.want)["header_bytes"]
    assert (got2[h2:] == want1[h1:]).all() and h1 > 8 * h2


@pytest.mark.parametrize("bset", small_sets(), ids=lambda s: s.name)
def test_deserialize_matches_oracle_and_round_trips(bset):
    lu = LayeredUp(bset)
    want = lu.want
    ref = v2.deserialize(want)
    na, need = v2.counts(want)
    stream_t = torch.from_numpy(want.copy()).to(DEV)
    out, pool, res = gpu_ldeserialize(stream_t, len(want), lu.counts, need)
    assert res["status"] == bs.OK, res
    assert (res["n_structs"], res["n_struct_blocks"], res["n_tensors"], res["n_blocks"], res["pool_bytes"]) == lu.counts + (need,)
    h = out.to_host(*lu.counts)
    assert h["structs"].tobytes() == ref["structs"].tobytes() and h["layers"].tobytes() == ref["layers"].tobytes()
    assert (h["qn"] == ref["qn"]).all() and (h["dim"] == ref["dim"]).all()
    assert ((h["addr"] - np.uint64(pool.data_ptr())) == (ref["addr"] - np.uint64(ref["pool"].ctypes.data))).all()
    assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
    # fixpoint on the device: serialize(deserialize(S)) == S
    again, res2 = gpu_lserialize(lu, len(want), dset=out)
    assert res2["status"] == bs.OK
    assert (again.cpu().numpy()[:len(want)] == want).all()


@pytest.mark.parametrize("opts", VARIANTS[1:], ids=lambda o: f"v{o['variant']}-t{o.get('tile_bytes')}")
def test_unpack_independent_of_decomposition(opts):
    lu = LayeredUp(W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0))
    ref = v2.deserialize(lu.want)
    na, need = v2.counts(lu.want)
    out, pool, res = gpu_ldeserialize(torch.from_numpy(lu.want.copy()).to(DEV), len(lu.want), lu.counts, need, opts=opts)
    assert res["status"] == bs.OK
    assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


@pytest.mark.parametrize("chunk", [16, 4096, 100000 * 16, 1 << 22])
def test_concat_of_ranges_is_the_stream(chunk):
    lu = LayeredUp(W.make_config("2"))
    want = lu.want
    total = len(want)
    if chunk == 16:
        hb = v2.stream_info(want)["header_bytes"]
        cuts = [0] + list(range(hb - 64, hb + 64, 16)) + [total]
    else:
        cuts = list(range(0, total, chunk)) + [total]
    ws = lu.workspace(total)
    out = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    first = True
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        seg = torch.full((hi - lo + 32,), 0x77, dtype=torch.uint8, device=DEV)
        bs.layered_serialize_range(lu.dset.desc, seg.data_ptr(), lo, hi, first, ws.ptr, ws.nbytes, ws.result_ptr, None,
                                   bs.current_stream())
        first = False
        assert (seg[hi - lo:] == 0x77).all(), "range call wrote beyond its segment"
        out[lo:hi] = seg[:hi - lo]
    assert ws.read_result()["status"] == bs.OK
    assert (out.cpu().numpy() == want).all()


def test_serialized_size_is_exact_prediction():
    for bset in small_sets():
        lu = LayeredUp(bset)
        ws = lu.workspace(1 << 16)          # tile index far too small: the prediction is still exact
        hb, tot = bs.layered_serialized_size(lu.dset.desc, ws.ptr, ws.nbytes, bs.current_stream())
        assert (hb, tot) == v2.serialized_size(lu.lv["structs"], lu.lv["layers"], lu.lv["dim"])


# ---- edge cases ------------------------------------------------------------------------------------------------------------
def _custom_layered(struct_rows, layer_struct, dim, seed=0):
    structs = np.zeros(len(struct_rows), dtype=W.STRUCT_REC_DTYPE)
    for i, r in enumerate(struct_rows):
        structs[i] = r
    layers = np.zeros(len(layer_struct), dtype=W.LAYER_REC_DTYPE)
    layers["structure"] = layer_struct
    layers["tag"] = np.arange(len(layer_struct)) + 5
    dim = np.array(dim, np.uint32).reshape(-1, 3)
    qn = np.zeros((len(dim), 3, 2), np.int32)
    rng = np.random.default_rng(seed)
    ne, offs, pos = [], [], 0
    for s in layer_struct:
        f, n = int(structs["first_block"][s]), int(structs["n_blocks"][s])
        for j in range(f, f + n):
            k = int(dim[j].astype(np.int64).prod())
            ne.append(k)
            offs.append(pos)
            pos += (k * 8 + 511) // 512 * 512
    pool = rng.uniform(-1, 1, max(pos // 8, 1))
    return structs, layers, qn, dim, pool, np.array(offs, np.uint64), np.array(ne, np.int64)


def _roundtrip_custom(structs, layers, qn, dim, pool, offs, opts=None):
    want = v2.serialize(structs, layers, qn, dim, host_addrs(pool, offs))
    d_pool = torch.from_numpy(pool.view(np.uint8).copy()).to(DEV)
    addr = (np.uint64(d_pool.data_ptr()) + offs).astype(np.uint64)
    dset = bs.DeviceLayeredSet.from_host(structs, layers, qn, dim, addr, DEV)
    caps = (len(structs), len(dim), len(layers), len(offs))
    ws = bs.Workspace(0, 0, max(len(want), 1 << 16), DEV, layered=caps)
    out = torch.full((len(want) + 256,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.layered_serialize(dset.desc, out.data_ptr(), len(want) + 256, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    res = ws.read_result()
    assert res["status"] == bs.OK, res
    got = out.cpu().numpy()
    assert (got[:len(want)] == want).all() and (got[len(want):] == 0xCD).all()
    ref = v2.deserialize(want)
    na, need = v2.counts(want)
    o2, p2, r2 = gpu_ldeserialize(out, len(want), caps, need, opts=opts)
    assert r2["status"] == bs.OK, r2
    assert (p2.cpu().numpy()[:need] == ref["pool"][:need]).all()
    return want


def test_empty_set_and_unused_structures():
    z = np.zeros(0, np.uint64)
    want = _roundtrip_custom(np.zeros(0, W.STRUCT_REC_DTYPE), np.zeros(0, W.LAYER_REC_DTYPE), np.zeros((0, 3, 2), np.int32),
                             np.zeros((0, 3), np.uint32), np.zeros(1), z)
    assert len(want) == 128
    # structure 0 has no blocks, structure 1 is used by nobody, zero-extent blocks in structure 2
    rows = [(2, 0, 0, (0, 0), (-1, 1, 0, 0), 0), (2, 0, 2, (0, 0), (-1, 1, 0, 0), 0), (3, 2, 3, (0, 0), (1, 1, -1, 0), 0)]
    dim = [[4, 5, 1], [3, 3, 1], [0, 5, 2], [3, 1, 1], [1, 1, 1]]
    st, ly, qn, dm, pool, offs, ne = _custom_layered(rows, [2, 0, 2, 0, 2], dim)
    _roundtrip_custom(st, ly, qn, dm, pool, offs)


def test_many_tiny_layers_and_one_huge_block():
    # 3000 layers of a 3-block structure of 1x1 / 1x2 / 3x1 blocks: every unit a tail unit, ~200 layers per tile
    rows = [(2, 0, 3, (0, 0), (-1, 1, 0, 0), 0), (2, 3, 2, (0, 0), (-1, 1, 0, 0), 0)]
    dim = [[1, 1, 1], [1, 2, 1], [3, 1, 1], [1500, 1501, 1], [2, 2, 1]]
    layer_struct = [0] * 1500 + [1] + [0] * 1500 + [1]
    st, ly, qn, dm, pool, offs, ne = _custom_layered(rows, layer_struct, dim, seed=3)
    for opts in (None, dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_TMA, tile_bytes=32768)):
        _roundtrip_custom(st, ly, qn, dm, pool, offs, opts)


def test_eight_byte_aligned_sources():
    bset = W.make_set("mis", 13, D=120, S=12, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    lu = LayeredUp(bset, misalign=8)
    assert (lu.up.addr % 16 == 8).all()
    for opts in (None, dict(variant=bs.VARIANT_LDG)):
        check_stream(lu, opts)


def test_scatter_to_caller_addresses():
    bset = W.make_set("scat", 51, D=60, S=10, M=2, N0=3, n_ops=15, n_site=1, dims="multinomial")
    lu = LayeredUp(bset)
    dst = torch.full((lu.up.pool.numel(),), 0xEE, dtype=torch.uint8, device=DEV)
    daddr = (np.uint64(dst.data_ptr()) + lu.up.host_offs).astype(np.uint64)
    lv = lu.lv
    out = bs.DeviceLayeredSet.from_host(np.zeros_like(lv["structs"]), np.zeros_like(lv["layers"]), np.zeros_like(lv["qn"]),
                                        lv["dim"], daddr, DEV)
    st = torch.from_numpy(lu.want.copy()).to(DEV)
    o, pool, res = gpu_ldeserialize(st, len(lu.want), lu.counts, 0, flags=bs.SCATTER_TO_ADDR, out=out)
    assert res["status"] == bs.OK, res
    got = dst.cpu().numpy()
    src = lu.up.host_pool.view(np.uint8)
    expect = np.full_like(got, 0xEE)
    ne = bset.nelems
    for i in range(bset.n_blocks):
        o_, n = int(lu.up.host_offs[i]), int(ne[i]) * 8
        expect[o_:o_ + n] = src[o_:o_ + n]
    assert (got == expect).all()
    h = out.to_host(*lu.counts)
    assert (h["structs"]["layer_bytes"] == v2.deserialize(lu.want)["structs"]["layer_bytes"]).all()
    # extents that differ are an argument error and nothing is written
    wrong = lv["dim"].copy()
    wrong[0, 0] += 1
    out = bs.DeviceLayeredSet.from_host(np.zeros_like(lv["structs"]), np.zeros_like(lv["layers"]), np.zeros_like(lv["qn"]),
                                        wrong, daddr, DEV)
    dst.fill_(0xEE)
    o, pool, res = gpu_ldeserialize(st, len(lu.want), lu.counts, 0, flags=bs.SCATTER_TO_ADDR, out=out)
    assert res["status"] == bs.ERR_ARG and (dst == 0xEE).all()


# ---- deferred errors --------------------------------------------------------------------------------------------------------
def test_capacity_and_descriptor_errors():
    bset = W.make_set("cap", 42, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    lu = LayeredUp(bset)
    out, res = gpu_lserialize(lu, len(lu.want) - 16)
    assert res["status"] == bs.ERR_CAPACITY and res["total_bytes"] == len(lu.want) and (out == 0xCD).all()
    lv = lu.lv
    # a layer naming a structure that does not exist; structures that do not partition; bad rank; misaligned block
    ly = lv["layers"].copy()
    ly["structure"][3] = len(lv["structs"])
    d = bs.DeviceLayeredSet.from_host(lv["structs"], ly, lv["qn"], lv["dim"], lu.up.addr, DEV)
    out, res = gpu_lserialize(lu, 1 << 20, dset=d)
    assert res["status"] == bs.ERR_ARG and (out == 0xCD).all()
    st = lv["structs"].copy()
    st["n_blocks"][0] -= 1
    d = bs.DeviceLayeredSet.from_host(st, lv["layers"], lv["qn"], lv["dim"], lu.up.addr, DEV)
    out, res = gpu_lserialize(lu, 1 << 20, dset=d)
    assert res["status"] == bs.ERR_ARG and (out == 0xCD).all()
    st = lv["structs"].copy()
    st["rank"][1] = 4
    d = bs.DeviceLayeredSet.from_host(st, lv["layers"], lv["qn"], lv["dim"], lu.up.addr, DEV)
    out, res = gpu_lserialize(lu, 1 << 20, dset=d)
    assert res["status"] == bs.ERR_UNSUPPORTED and (out == 0xCD).all()
    a = lu.up.addr.copy()
    a[5] += 4
    d = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], a, DEV)
    out, res = gpu_lserialize(lu, 1 << 20, dset=d)
    assert res["status"] == bs.ERR_ARG and (out == 0xCD).all()
    # addr[] shorter than the number of blocks
    d = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], lu.up.addr[:-1], DEV)
    out, res = gpu_lserialize(lu, 1 << 20, dset=d)
    assert res["status"] == bs.ERR_CAPACITY and (out == 0xCD).all()
    # deserialize: pool / arrays too small
    na, need = v2.counts(lu.want)
    s = torch.from_numpy(lu.want.copy()).to(DEV)
    o, pool, res = gpu_ldeserialize(s, len(lu.want), lu.counts, need - 256)
    assert res["status"] == bs.ERR_CAPACITY and res["pool_bytes"] == need and (pool == 0xEE).all()
    c = lu.counts
    o, pool, res = gpu_ldeserialize(s, len(lu.want), (c[0], c[1] - 1, c[2], c[3]), need)
    assert res["status"] == bs.ERR_CAPACITY and (pool == 0xEE).all()
    o, pool, res = gpu_ldeserialize(s, len(lu.want), (c[0], c[1], c[2], c[3] - 1), need)
    assert res["status"] == bs.ERR_CAPACITY and (pool == 0xEE).all()


def test_corrupt_headers_are_rejected_and_nothing_is_written():
    from tests.test_oracle_v2 import _mutations
    bset = W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    lu = LayeredUp(bset)
    want = lu.want
    na, need = v2.counts(want)
    caps = tuple(x + 1 for x in lu.counts)
    for what, pos in _mutations(want):
        bad = want.copy()
        bad[pos] ^= 0x04 if what == "struct rank" else 0x01
        assert v2.validate_stream(bad) == oracle.ERR_CORRUPT
        out, pool, res = gpu_ldeserialize(torch.from_numpy(bad).to(DEV), len(bad), caps, need + 4096)
        assert res["status"] == bs.ERR_CORRUPT, (what, res)
        assert (pool == 0xEE).all(), f"{what}: pool written despite corrupt header"
        for arr in (out.structs, out.layers, out.qn, out.dim):
            assert (arr == 0xAB).all(), f"{what}: descriptor written despite corrupt header"
    st = torch.from_numpy(want.copy()).to(DEV)
    for n in (len(want) - 16, 48):
        out, pool, res = gpu_ldeserialize(st, n, lu.counts, need)
        assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all()
    # a v1 stream handed to the v2 entry point
    s1 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(lu.up.host_pool, lu.up.host_offs))
    out, pool, res = gpu_ldeserialize(torch.from_numpy(s1.copy()).to(DEV), len(s1), caps, need)
    assert res["status"] == bs.ERR_CORRUPT


# ---- engine -------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("chunk,n_staging", [(65536, 2), (1 << 20, 3), (65536, 1)])
def test_engine_offload_prefetch_round_trip(chunk, n_staging):
    bset = W.make_config("2")
    lu = LayeredUp(bset)
    want = lu.want
    total = len(want)
    c = lu.counts
    eng = bs.Engine(max(c[0], c[2]), max(c[1], c[3]), total, chunk_bytes=chunk, n_staging=n_staging)
    host = torch.full((total,), 0x33, dtype=torch.uint8).pin_memory()
    t = eng.offload_layered_async(lu.dset.desc, total, host.data_ptr(), total, bs.current_stream())
    st = t.wait()
    assert st["status"] == bs.OK and st["bytes"] == total
    assert (host.numpy() == want).all()
    ref = v2.deserialize(want)
    na, need = v2.counts(want)
    out = bs.DeviceLayeredSet.empty(*c, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    t = eng.prefetch_layered_async(host.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, bs.current_stream())
    assert t.wait()["status"] == bs.OK
    torch.cuda.synchronize()
    assert (pool.cpu().numpy() == ref["pool"][:need]).all()
    h = out.to_host(*c)
    assert h["structs"].tobytes() == ref["structs"].tobytes() and h["layers"].tobytes() == ref["layers"].tobytes()
    # a flipped pad byte in a payload chunk is caught by the unpack kernels
    _, structs, layers, blocks, _, _ = __import__("tests.streamreader", fromlist=["x"]).read_stream_v2(want.tobytes())
    hb = v2.stream_info(want)["header_bytes"]
    for ly in layers:
        sr = structs[ly["structure"]]
        odd = [b for b in blocks[sr["first_block"]:sr["first_block"] + sr["n_blocks"]] if (b["dim"][0] * b["dim"][1] * b["dim"][2]) % 2]
        if odd:
            b = odd[0]
            pos = hb + ly["offset"] + b["offset"] + 8 * b["dim"][0] * b["dim"][1] * b["dim"][2] + 2
            break
    host[pos] ^= 1
    t = eng.prefetch_layered_async(host.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, bs.current_stream())
    assert t.wait()["status"] == bs.ERR_CORRUPT
    eng.destroy()


# ---- element types of layered sets (reading E-2) ------------------------------------------
ELEM = {bs.F64: 8, bs.F32: 4, bs.C64: 8, bs.C128: 16}


class TypedLayeredUp:
    """The blocks of a set read as e-byte elements (the first e*n bytes of each block's storage; for 16-byte elements the
    pool is laid out with twice the room).  The oracle and the CUDA path see the same host / device bytes."""

    def __init__(self, bset, dtype, misalign=0):
        e = ELEM[dtype]
        pool, offs = W.fill_pool_host(bset)
        if e == 16:
            big = np.zeros(2 * pool.size + 2, np.float64)
            offs = offs * 2
            for o, n in zip(offs, bset.nelems):
                src = pool[int(o) // 16: int(o) // 16 + int(n)]
                big[int(o) // 8: int(o) // 8 + 2 * int(n)] = np.repeat(src, 2) * np.tile([1.0, -0.5], int(n))
            pool = big
        self.bset, self.dtype, self.e = bset, dtype, e
        self.up = Uploaded(bset, pool, offs, misalign=misalign)
        self.lv = lv = W.layered_view(bset)
        self.dset = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], self.up.addr, DEV, dtype=dtype)
        self.want = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), dtype=dtype)
        self.counts = (len(lv["structs"]), lv["dim"].shape[0], len(lv["layers"]), bset.n_blocks)

    def workspace(self, cap):
        return bs.Workspace(0, 0, max(cap, 1 << 16), DEV, layered=self.counts)


def test_golden_v2_f32_stream_from_the_gpu():
    """The hand-typed G6 bytes (tests/golden/g6_golden_stream_v2_f32.hex) out of the CUDA path, and back."""
    import os
    from tests.test_oracle_v2 import GOLD_F32, golden_set_f32
    from tests.util import read_hex_fixture
    structs, layers, qn, dim, blocks = golden_set_f32()
    raw = np.zeros(4 * 64, np.uint8)
    for k, b in enumerate(blocks):
        raw[64 * k: 64 * k + b.nbytes] = b.view(np.uint8)
    d_pool = torch.from_numpy(raw).to(DEV)
    addr = (np.uint64(d_pool.data_ptr()) + np.arange(4, dtype=np.uint64) * np.uint64(64)).astype(np.uint64)
    dset = bs.DeviceLayeredSet.from_host(structs, layers, qn, dim, addr, DEV, dtype=bs.F32)
    ws = bs.Workspace(0, 0, 1 << 16, DEV, layered=(1, 2, 2, 4))
    out = torch.full((1024,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.layered_serialize(dset.desc, out.data_ptr(), 1024, ws.ptr, ws.nbytes, ws.result_ptr, None, bs.current_stream())
    res = ws.read_result()
    assert res["status"] == bs.OK and res["total_bytes"] == 320 and res["dtype"] == bs.F32
    gold = read_hex_fixture(GOLD_F32)
    assert out.cpu().numpy()[:320].tobytes() == gold and (out.cpu().numpy()[320:] == 0xCD).all()
    assert bs.layered_stream_info(gold)["dtype"] == bs.F32
    o, pool, res = gpu_ldeserialize(out, 320, (1, 2, 2, 4), 1024)
    ref = v2.deserialize(np.frombuffer(gold, np.uint8))
    assert res["status"] == bs.OK and res["dtype"] == bs.F32 and (pool.cpu().numpy()[:1024] == ref["pool"][:1024]).all()


@pytest.mark.parametrize("opts", [None, dict(variant=bs.VARIANT_LDG, tile_bytes=16384), dict(variant=bs.VARIANT_TMA, tile_bytes=32768)],
                         ids=["default", "ldg", "tma32k"])
@pytest.mark.parametrize("dtype", [bs.F32, bs.C64, bs.C128, bs.F64], ids=["f32", "c64", "c128", "f64"])
def test_typed_layered_sets_match_the_oracle_and_round_trip(dtype, opts):
    for bset in (W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial"),
                 W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)):
        lu = TypedLayeredUp(bset, dtype)
        total = len(lu.want)
        got_t, res = gpu_lserialize(lu, total + 4096, opts)
        assert res["status"] == bs.OK and res["total_bytes"] == total and res["dtype"] == dtype, res
        got = got_t.cpu().numpy()
        bad = np.nonzero(got[:total] != lu.want)[0]
        assert bad.size == 0, f"first mismatch at stream byte {bad[0]}"
        assert (got[total:] == 0xCD).all()
        ws = lu.workspace(total)
        assert bs.layered_serialized_size(lu.dset.desc, ws.ptr, ws.nbytes, bs.current_stream()) == \
            v2.serialized_size(lu.lv["structs"], lu.lv["layers"], lu.lv["dim"], dtype)
        ref = v2.deserialize(lu.want)
        na, need = v2.counts(lu.want)
        out, pool, res = gpu_ldeserialize(got_t, total, lu.counts, need, opts=opts)
        assert res["status"] == bs.OK and res["pool_bytes"] == need and res["dtype"] == dtype, res
        assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        h = out.to_host(*lu.counts)
        assert (h["dim"] == lu.lv["dim"]).all() and (h["qn"] == lu.lv["qn"]).all()
        assert (h["structs"]["layer_bytes"] == ref["structs"]["layer_bytes"]).all() and (h["layers"]["offset"] == ref["layers"]["offset"]).all()
        out.dtype = dtype                     # fixpoint: serialize(deserialize(S)) == S
        again = torch.full((total,), 0x11, dtype=torch.uint8, device=DEV)
        bs.layered_serialize(out.desc, again.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
        assert ws.read_result()["status"] == bs.OK and (again.cpu().numpy() == lu.want).all()


def test_typed_layered_sets_eight_byte_sources_ranges_engine_queue_and_packages():
    bset = W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)
    cs = bs.current_stream()
    for dtype in (bs.F32, bs.C128):
        lu = TypedLayeredUp(bset, dtype, misalign=8)          # 8-byte-aligned sources take the slow path (D16)
        total = len(lu.want)
        got_t, res = gpu_lserialize(lu, total)
        assert res["status"] == bs.OK and (got_t.cpu().numpy()[:total] == lu.want).all()
        lu = TypedLayeredUp(bset, dtype)
        ws = lu.workspace(total)
        # concat(ranges) == the stream
        out = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
        cuts = list(range(0, total, 100000 * 16)) + [total]
        for k, (lo, hi) in enumerate(zip(cuts[:-1], cuts[1:])):
            bs.layered_serialize_range(lu.dset.desc, out[lo:].data_ptr(), lo, hi, k == 0, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
        assert ws.read_result()["status"] == bs.OK and (out.cpu().numpy() == lu.want).all()
        # engine + queue: the stream crosses PCIe with its element type; packages of it reassemble
        c = lu.counts
        eng = bs.Engine(max(c[0], c[2]), c[3], total, chunk_bytes=4 * 65536)
        host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
        host.fill_(0x5A)
        assert eng.offload_layered_async(lu.dset.desc, total, host.data_ptr(), total, cs).wait()["status"] == bs.OK
        assert (host.numpy() == lu.want).all()
        ref = v2.deserialize(lu.want)
        na, need = v2.counts(lu.want)
        lout = bs.DeviceLayeredSet.empty(*c, DEV, fill=0xAB)
        pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
        st = eng.prefetch_layered_async(host.data_ptr(), total, lout.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs).wait()
        torch.cuda.synchronize()
        assert st["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        eng.destroy()
        q = bs.Queue(max(c[0], c[2]), c[3], total, chunk_bytes=4 * 65536)
        host.fill_(0x5A)
        pool.fill_(0xEE)
        q.save_layered(5, lu.dset.desc, total, host.data_ptr(), total, cs)
        q.load_layered(5, lout.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)
        assert q.wait(5)["status"] == bs.OK
        torch.cuda.synchronize()
        assert (host.numpy() == lu.want).all() and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
        q.destroy()
        from oracle import pkg
        cap = 32768
        hb = v2.stream_info(lu.want)["header_bytes"]
        n = pkg.count(hb, total, cap)
        slots = torch.full((n * (64 + cap),), 0x5A, dtype=torch.uint8, device=DEV)
        wsp = bs.Workspace(0, 0, total, DEV, layered=c, packages=True)
        bs.layered_package_emit(lu.dset.desc, total, cap, 11, slots.data_ptr(), 64 + cap, n, None, wsp.ptr, wsp.nbytes,
                                wsp.result_ptr, None, cs)
        assert wsp.read_result()["status"] == bs.OK
        assert (slots.cpu().numpy().reshape(n, -1) == pkg.emit_slots(lu.want, cap, 11, 64 + cap, poison=0x5A)).all()
        pool.fill_(0xEE)
        bs.layered_package_unpack(slots.data_ptr(), 64 + cap, n, 11, lout.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, wsp.ptr,
                                  wsp.nbytes, wsp.result_ptr, None, cs)
        assert wsp.read_result()["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


def test_typed_layered_sets_bad_types_and_nonzero_pads_are_rejected():
    bset = W.make_set("few-ops", 13, D=64, S=12, M=2, N0=2, n_ops=5, n_site=1, dims="multinomial")
    lu = TypedLayeredUp(bset, bs.F32)
    d = bs.DeviceLayeredSet.from_host(lu.lv["structs"], lu.lv["layers"], lu.lv["qn"], lu.lv["dim"], lu.up.addr, DEV, dtype=4)
    ws = lu.workspace(1 << 20)
    with pytest.raises(bs.BsError) as e:
        bs.layered_serialize(d.desc, 256, 1 << 20, ws.ptr, ws.nbytes, ws.result_ptr, None, bs.current_stream())
    assert e.value.code == bs.ERR_UNSUPPORTED
    na, need = v2.counts(lu.want)
    bad = lu.want.copy()
    bad[16] = 4                                   # dtype word
    assert v2.validate_stream(bad) == oracle.ERR_CORRUPT
    o, pool, res = gpu_ldeserialize(torch.from_numpy(bad).to(DEV), len(bad), lu.counts, need)
    assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all()
    # a non-zero pad byte of every pad length (4, 8, 12) — direct call and through the engine (checked while unpacking)
    info = v2.stream_info(lu.want)
    plan = v2.plan(lu.lv["structs"], lu.lv["layers"], lu.lv["dim"], bs.F32)
    seen = set()
    for k, srec in enumerate(lu.lv["structs"]):
        layer0 = int(np.nonzero(lu.lv["layers"]["structure"] == k)[0][0])
        for j in range(int(srec["first_block"]), int(srec["first_block"]) + int(srec["n_blocks"])):
            nb = 4 * int(np.prod(lu.lv["dim"][j].astype(np.int64)))
            pad = -nb % 16
            if pad and pad not in seen:
                seen.add(pad)
                bad = lu.want.copy()
                bad[info["header_bytes"] + int(plan["layer_offset"][layer0]) + int(plan["rel_offset"][j]) + nb + pad - 1] = 0x80
                assert v2.validate_stream(bad) == oracle.ERR_CORRUPT
                o, pool, res = gpu_ldeserialize(torch.from_numpy(bad).to(DEV), len(bad), lu.counts, need)
                assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all(), (pad, res)
                c = lu.counts
                eng = bs.Engine(max(c[0], c[2]), c[3], len(bad), chunk_bytes=65536)
                host = torch.empty(len(bad), dtype=torch.uint8, pin_memory=True)
                host.numpy()[:] = bad
                lout = bs.DeviceLayeredSet.empty(*c, DEV, fill=0xAB)
                pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
                st = eng.prefetch_layered_async(host.data_ptr(), len(bad), lout.desc, pool.data_ptr(), need).wait()
                assert st["status"] == bs.ERR_CORRUPT
                eng.destroy()
    assert seen == {4, 8, 12}
