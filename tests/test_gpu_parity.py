"""Parity of the CUDA path (through the C ABI) with the CPU oracle: bit-exact, tolerance 0.
Every test here needs a GPU.  Inputs: seeded synthetic sets (workloads/), never a value from the CUDA path."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from tests.gpu_util import DEV, Uploaded, gpu_deserialize, gpu_serialize
from tests.streamreader import read_stream
from tests.util import host_addrs, oracle_stream

pytestmark = pytest.mark.gpu

VARIANTS = [dict(variant=bs.VARIANT_LDG, tile_bytes=16384), dict(variant=bs.VARIANT_LDG, tile_bytes=32768),
            dict(variant=bs.VARIANT_LDG, tile_bytes=49152), dict(variant=bs.VARIANT_LDG, tile_bytes=65536, ctas_per_sm=1),
            dict(variant=bs.VARIANT_TMA), dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=4, warps=3),
            dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=4, warps=1),
            dict(variant=bs.VARIANT_TMA, tile_bytes=16384), dict(variant=bs.VARIANT_TMA, tile_bytes=32768),
            dict(variant=bs.VARIANT_TMA, tile_bytes=65536), dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=1),
            dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=8, warps=1),
            dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=4),
            dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=3, warps=2),
            # the shape the pack preset switches to on sets of half a GB and more (one ring of 3 x 48 KiB)
            dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=3, warps=1),
            # one fused launch (size / offset pass + movement) against separate launches; default shape and a wide one
            dict(variant=bs.VARIANT_TMA, fuse=1), dict(variant=bs.VARIANT_TMA, fuse=2),
            dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=4, fuse=2),
            dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=4, warps=1, fuse=2),
            # tiles that do not end on a 16 KiB granule of the work partition (the TMA variant takes any multiple of 1 KiB)
            dict(variant=bs.VARIANT_TMA, tile_bytes=40960, stages=3, warps=1), dict(variant=bs.VARIANT_TMA, tile_bytes=24576, stages=4, warps=2),
            dict(variant=bs.VARIANT_TMA, tile_bytes=20480, stages=3, warps=3, fuse=2), dict(variant=bs.VARIANT_TMA, tile_bytes=5120, stages=5, warps=2),
            dict(variant=bs.VARIANT_TMA, tile_bytes=4096, stages=3, warps=1, fuse=2), dict(variant=bs.VARIANT_TMA, tile_bytes=4096, stages=3, warps=1, fuse=1),
            # paced launches (bs_opts.reserved[2]): a fixed target rate with the large-set shape, and pacing switched off
            dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=4, warps=1, pace=6500), dict(variant=bs.VARIANT_TMA, pace=1),
            dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=2, pace=200, fuse=2),
            # round 1's static round-robin deal of the tiles (tune bit 3) and table entries fetched two iterations ahead (bit 12)
            dict(variant=bs.VARIANT_TMA, tune=8), dict(variant=bs.VARIANT_TMA, tile_bytes=32768, stages=5, warps=1, tune=0x1000),
            dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=3, warps=4, tune=0x1008, fuse=2),
            # tiles handed out by the counter (what ranges of 128 MiB and more do; bit 4 forces it on these small sets)
            dict(variant=bs.VARIANT_TMA, tune=0x10), dict(variant=bs.VARIANT_TMA, tune=0x10, fuse=1), dict(variant=bs.VARIANT_TMA, tune=0x10, fuse=2),
            dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=3, warps=1, tune=0x10),
            dict(variant=bs.VARIANT_TMA, tile_bytes=20480, stages=5, warps=2, tune=0x1010), dict(variant=bs.VARIANT_TMA, tile_bytes=16384, stages=8, warps=1, tune=0x10, fuse=2)]


def _vid(o):
    return (f"v{o['variant']}-t{o.get('tile_bytes', 0)}-c{o.get('ctas_per_sm', 0)}-s{o.get('stages', 0)}-w{o.get('warps', 0)}"
            f"-f{o.get('fuse', 0)}" + (f"-p{o['pace']}" if o.get("pace") else "") + (f"-x{o['tune']:x}" if o.get("tune") else ""))


def small_sets():
    return [W.make_config("1"), W.make_config("2"),
            W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial"),
            W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)]


def check_stream(bset, up, opts=None, slack=4096):
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    got_t, res = gpu_serialize(up.dset, total + slack, opts)
    assert res["status"] == bs.OK, res
    hb, tot = oracle.serialized_size(bset.n_tensors, bset.dim)
    assert (res["header_bytes"], res["total_bytes"], res["payload_bytes"]) == (hb, tot, tot - hb)
    got = got_t.cpu().numpy()
    bad = np.nonzero(got[:total] != want)[0]
    assert bad.size == 0, f"first mismatch at stream byte {bad[0]} (header_bytes={hb}), opts={opts}"
    assert (got[total:] == 0xCD).all(), "bytes beyond the stream were written"
    return got_t, want


@pytest.mark.parametrize("bset", small_sets(), ids=lambda s: s.name)
def test_serialize_matches_oracle_byte_for_byte(bset):
    up = Uploaded(bset)
    check_stream(bset, up)


@pytest.mark.parametrize("opts", VARIANTS, ids=_vid)
def test_P6_stream_independent_of_decomposition(opts):
    for bset in (W.make_config("2"), W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2,
                                                dims="lognormal", sigma=1.0)):
        up = Uploaded(bset)
        check_stream(bset, up, opts)


@pytest.mark.parametrize("bset", small_sets(), ids=lambda s: s.name)
def test_deserialize_matches_oracle_and_round_trips(bset):
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    ref = oracle.deserialize(want)                       # pool poisoned 0xEE, as on the GPU side
    stream_t = torch.from_numpy(want.copy()).to(DEV)
    need = oracle.pool_bytes(want)
    out, pool, res = gpu_deserialize(stream_t, len(want), bset.n_tensors, bset.n_blocks, need)
    assert res["status"] == bs.OK, res
    assert (res["n_tensors"], res["n_blocks"], res["pool_bytes"]) == (bset.n_tensors, bset.n_blocks, need)
    h = out.to_host()
    assert h["tensors"].tobytes() == ref["tensors"].tobytes() == bset.tensors.tobytes()
    assert (h["qn"] == ref["qn"]).all() and (h["dim"] == ref["dim"]).all()
    # D14 placement: same pool-relative addresses as the oracle, and byte-identical pools (untouched bytes included)
    assert ((h["addr"] - np.uint64(pool.data_ptr())) == (ref["addr"] - np.uint64(ref["pool"].ctypes.data))).all()
    gp = pool.cpu().numpy()
    assert (gp[:need] == ref["pool"][:need]).all()
    # fixpoint on the device: serialize(deserialize(S)) == S
    again, res2 = gpu_serialize(out, len(want))
    assert res2["status"] == bs.OK
    assert (again.cpu().numpy()[:len(want)] == want).all()


@pytest.mark.parametrize("opts", VARIANTS, ids=_vid)
def test_P6_unpack_independent_of_decomposition(opts):
    bset = W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2, dims="lognormal", sigma=1.0)
    want, _, _ = oracle_stream(bset)
    ref = oracle.deserialize(want)
    need = oracle.pool_bytes(want)
    out, pool, res = gpu_deserialize(torch.from_numpy(want.copy()).to(DEV), len(want), bset.n_tensors, bset.n_blocks,
                                     need, opts=opts)
    assert res["status"] == bs.OK
    assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


@pytest.mark.parametrize("opts", [None, dict(variant=bs.VARIANT_TMA, tune=0x10), dict(variant=bs.VARIANT_TMA, tile_bytes=20480, stages=4, warps=2, tune=0x10)],
                         ids=["default", "counter", "counter-20K"])
@pytest.mark.parametrize("chunk", [16, 4096, 65536, 100000 * 16, 1 << 22])
def test_P6_concat_of_ranges_is_the_stream(chunk, opts):
    bset = W.make_config("2")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    if chunk == 16:      # byte-granular ranges only around the header/payload boundary (keeps the test fast)
        hb = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
        cuts = [0] + list(range(hb - 64, hb + 64, 16)) + [total]
    else:
        cuts = list(range(0, total, chunk)) + [total]
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    out = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    first = True
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        seg = torch.full((hi - lo + 32,), 0x77, dtype=torch.uint8, device=DEV)
        bs.serialize_range(up.dset.desc, seg.data_ptr(), lo, hi, first, ws.ptr, ws.nbytes, ws.result_ptr, opts,
                           bs.current_stream())
        first = False
        assert (seg[hi - lo:] == 0x77).all(), "range call wrote beyond its segment"
        out[lo:hi] = seg[:hi - lo]
    assert ws.read_result()["status"] == bs.OK
    assert (out.cpu().numpy() == want).all()


def test_serialized_size_is_exact_prediction():
    for bset in small_sets():
        up = Uploaded(bset)
        ws = bs.Workspace(bset.n_tensors, bset.n_blocks, 1 << 16, DEV)     # tile index far too small: still exact
        hb, tot = bs.serialized_size(up.dset.desc, ws.ptr, ws.nbytes, bs.current_stream())
        assert (hb, tot) == oracle.serialized_size(bset.n_tensors, bset.dim)


# ---- edge cases ---------------------------------------------------------------------------------------------
def _custom(tensor_rows, dim, data, qn=None):
    tensors = np.zeros(len(tensor_rows), dtype=W.TENSOR_REC_DTYPE)
    for i, r in enumerate(tensor_rows):
        tensors[i] = r
    dim = np.array(dim, np.uint32).reshape(-1, 3)
    B = len(dim)
    qn = np.zeros((B, 3, 2), np.int32) if qn is None else qn
    ne = dim.astype(np.int64).prod(axis=1)
    offs = np.zeros(B, np.uint64)
    sz = (ne * 8 + 511) // 512 * 512
    if B > 1:
        offs[1:] = np.cumsum(sz[:-1])
    pool = np.zeros(max(int(sz.sum()) // 8, 1))
    for i in range(B):
        pool[int(offs[i]) // 8: int(offs[i]) // 8 + int(ne[i])] = data[i]
    bset = W.BlockSparseSet("custom", 0, tensors, qn, dim, offs, pool.nbytes)
    return bset, pool, offs


def test_D11_empty_set():
    bset, pool, offs = _custom([], np.zeros((0, 3)), [])
    up = Uploaded(bset, pool, offs)
    got, want = check_stream(bset, up)
    assert len(want) == 128
    out, p, res = gpu_deserialize(got, 128, 0, 0, 0)
    assert res["status"] == bs.OK and res["n_blocks"] == 0


def test_D11_zero_extent_blocks_and_empty_tensors():
    rows = [(2, 0, 2, (0, 0), (-1, 1, 0, 0), 0, 0), (3, 2, 0, (0, 0), (1, 1, -1, 0), 1, 0),
            (2, 2, 3, (0, 0), (-1, 1, 0, 0), 2, 0)]
    dim = [[0, 5, 1], [3, 1, 1], [2, 0, 1], [0, 0, 1], [1, 1, 1]]
    bset, pool, offs = _custom(rows, dim, [[], [1., 2., 3.], [], [], [4.]])
    up = Uploaded(bset, pool, offs)
    got, want = check_stream(bset, up)
    out, p, res = gpu_deserialize(got, len(want), 3, 5, oracle.pool_bytes(want))
    assert res["status"] == bs.OK
    ref = oracle.deserialize(want)
    assert (p.cpu().numpy()[:len(ref["pool"])] == ref["pool"]).all()
    assert (out.to_host()["dim"] == bset.dim).all()


def test_many_tiny_blocks_per_tile():
    # 1x1 blocks: 16 stored bytes each -> 2048 blocks per 32 KiB tile, every unit is a tail unit
    B = 9000
    rng = np.random.default_rng(1)
    dim = np.ones((B, 3), np.int64)
    dim[::7, 1] = 2
    dim[::11, 0] = 3
    data = [rng.uniform(-1, 1, int(d.prod())) for d in dim]
    bset, pool, offs = _custom([(2, 0, B, (0, 0), (-1, 1, 0, 0), 0, 0)], dim, data)
    up = Uploaded(bset, pool, offs)
    for opts in (None, dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_TMA, tile_bytes=32768)):
        got, want = check_stream(bset, up, opts)
        out, p, res = gpu_deserialize(got, len(want), 1, B, oracle.pool_bytes(want), opts=opts)
        assert res["status"] == bs.OK
        ref = oracle.deserialize(want)
        assert (p.cpu().numpy()[:len(ref["pool"])] == ref["pool"]).all()


def test_one_huge_block_and_neighbours():
    rng = np.random.default_rng(2)
    dim = [[3, 3, 1], [1500, 1501, 1], [5, 1, 7]]           # 18 MB block: thousands of tiles, odd element count
    data = [rng.uniform(-1, 1, int(np.prod(d))) for d in dim]
    bset, pool, offs = _custom([(2, 0, 2, (0, 0), (-1, 1, 0, 0), 0, 0), (3, 2, 1, (0, 0), (1, 1, -1, 0), 1, 0)], dim, data)
    up = Uploaded(bset, pool, offs)
    for opts in (None, dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_TMA, tile_bytes=32768)):
        got, want = check_stream(bset, up, opts)
        out, p, res = gpu_deserialize(got, len(want), 2, 3, oracle.pool_bytes(want), opts=opts)
        ref = oracle.deserialize(want)
        assert res["status"] == bs.OK and (p.cpu().numpy()[:len(ref["pool"])] == ref["pool"]).all()


def test_D16_eight_byte_aligned_sources_take_the_slow_path():
    bset = W.make_set("mis", 13, D=120, S=12, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    up = Uploaded(bset, misalign=8)
    assert (up.addr % 16 == 8).all()
    for opts in (None, dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_TMA, tile_bytes=32768)):
        check_stream(bset, up, opts)
    # and scatter back to 8-byte-aligned destinations
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    dst = torch.full((up.pool.numel(),), 0xEE, dtype=torch.uint8, device=DEV)
    daddr = (np.uint64(dst.data_ptr() + 8) + up.host_offs).astype(np.uint64)
    out = bs.DeviceSet.from_host(np.zeros(bset.n_tensors, W.TENSOR_REC_DTYPE), np.zeros_like(bset.qn), bset.dim, daddr, DEV)
    for opts in (None, dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_TMA, tile_bytes=32768)):
        dst.fill_(0xEE)
        ws = bs.Workspace(bset.n_tensors, bset.n_blocks, len(want), DEV)
        st = torch.from_numpy(want.copy()).to(DEV)
        bs.deserialize(st.data_ptr(), len(want), out.desc, 0, 0, bs.SCATTER_TO_ADDR, ws.ptr, ws.nbytes, ws.result_ptr, opts,
                       bs.current_stream())
        assert ws.read_result()["status"] == bs.OK
        got = dst.cpu().numpy()
        src = up.host_pool.view(np.uint8)
        ne = bset.nelems
        expect = np.full_like(got, 0xEE)
        for i in range(bset.n_blocks):
            o, n = int(up.host_offs[i]), int(ne[i]) * 8
            expect[8 + o: 8 + o + n] = src[o:o + n]
        assert (got == expect).all()
        assert out.to_host()["tensors"].tobytes() == bset.tensors.tobytes()


def test_P11_special_bit_patterns():
    pats = np.array([0x7FF8000000000001, 0xFFF0000000000000, 0x8000000000000000, 0x0000000000000001,
                     0x7FF0000000000000, 0x7FF4DEADBEEF0001, 0x000FFFFFFFFFFFFF], dtype=np.uint64)
    bset, pool, offs = _custom([(2, 0, 1, (0, 0), (-1, 1, 0, 0), 0, 0)], [[1, 7, 1]], [pats.view(np.float64)])
    assert (pool.view(np.uint64)[:7] == pats).all()
    up = Uploaded(bset, pool, offs)
    got, want = check_stream(bset, up)
    out, p, res = gpu_deserialize(got, len(want), 1, 1, 256)
    assert (p.cpu().numpy()[:56].view(np.uint64) == pats).all()


# ---- deferred errors -------------------------------------------------------------------------------------------
def test_capacity_error_reports_required_size_and_writes_nothing():
    bset = W.make_config("1")
    up = Uploaded(bset)
    hb, tot = oracle.serialized_size(1, bset.dim)
    out, res = gpu_serialize(up.dset, tot - 16)
    assert res["status"] == bs.ERR_CAPACITY and res["total_bytes"] == tot
    assert (out == 0xCD).all()


def test_bad_descriptors_are_rejected_on_the_device():
    bset = W.make_config("1")
    up = Uploaded(bset)
    t = bset.tensors.copy()
    t["n_blocks"][0] -= 1
    d = bs.DeviceSet.from_host(t, bset.qn, bset.dim, up.addr, DEV)
    out, res = gpu_serialize(d, 1 << 16)
    assert res["status"] == bs.ERR_ARG and (out == 0xCD).all()
    t = bset.tensors.copy()
    t["rank"][0] = 4
    d = bs.DeviceSet.from_host(t, bset.qn, bset.dim, up.addr, DEV)
    out, res = gpu_serialize(d, 1 << 16)
    assert res["status"] == bs.ERR_UNSUPPORTED and (out == 0xCD).all()
    a = up.addr.copy()
    a[3] += 4
    d = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, a, DEV)
    out, res = gpu_serialize(d, 1 << 16)
    assert res["status"] == bs.ERR_ARG and (out == 0xCD).all()
    # host-side argument errors are immediate
    with pytest.raises(bs.BsError) as e:
        bs.serialize(up.dset.desc, 8, 1 << 16, 0, 0, 0, None, 0)
    assert e.value.code == bs.ERR_ARG


def test_P10_corrupt_headers_are_rejected_and_nothing_is_written():
    from tests.test_oracle_invariants import _mutations
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    want, _, _ = oracle_stream(bset)
    need = oracle.pool_bytes(want)
    cases = [(name, pos, xor, len(want)) for name, pos, xor in _mutations(want, bset)]
    for name, pos, xor, n in cases:
        bad = want.copy()
        bad[pos] ^= xor
        assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
        out, pool, res = gpu_deserialize(torch.from_numpy(bad).to(DEV), n, bset.n_tensors + 1, bset.n_blocks + 1, need + 4096)
        assert res["status"] == bs.ERR_CORRUPT, (name, res)
        assert (pool == 0xEE).all(), f"{name}: pool written despite corrupt header"
        for arr in (out.tensors, out.qn, out.dim, out.addr):
            assert (arr == 0xAB).all(), f"{name}: descriptor written despite corrupt header"
    st = torch.from_numpy(want.copy()).to(DEV)
    for n in (len(want) - 16, 48):
        out, pool, res = gpu_deserialize(st, n, bset.n_tensors, bset.n_blocks, need)
        assert res["status"] == bs.ERR_CORRUPT and (pool == 0xEE).all()


def test_a_payload_without_blocks_is_corrupt():
    """T = 0, B = 0, payload_bytes != 0: no block record carries the offset link check, so the totals must catch it
    ("final sum == payload_bytes").  Oracle first, then every kernel variant and both launch forms."""
    import struct
    for P in (16, 65536 + 32):
        bad = np.zeros(128 + P, np.uint8)
        bad[:64] = np.frombuffer(b"BSPARSE1" + struct.pack("<IIIIIIQQQQ", 1, 0x01020304, 0, 2, 3, 16, 0, 0, 128, P), np.uint8)
        assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
        for opts in (None, dict(variant=bs.VARIANT_TMA, fuse=1), dict(variant=bs.VARIANT_TMA, fuse=2),
                     dict(variant=bs.VARIANT_LDG), dict(variant=bs.VARIANT_LDG, tile_bytes=65536)):
            out, pool, res = gpu_deserialize(torch.from_numpy(bad).to(DEV), len(bad), 4, 64, 4096, opts=opts)
            assert res["status"] == bs.ERR_CORRUPT, (P, opts, res)
            assert (pool == 0xEE).all()
            for arr in (out.tensors, out.qn, out.dim, out.addr):
                assert (arr == 0xAB).all()


@pytest.mark.parametrize("junk", ["ones", "random", "previous-call"])
def test_the_workspace_needs_no_clearing(junk):
    """The size / offset pass synchronises on epoch-tagged words only (bs_scan_phase.cuh) and the movement's tile counter is
    tagged too (bs_move_tma.cu): whatever the workspace holds — all ones, noise, the state of an earlier call on a larger set
    — the stream is the oracle's.  Both launch forms, sets of
    one work item (replicated pass), of a few, and deserialize."""
    sets = [W.make_config("1"), W.make_config("2"),
            W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")]
    ups = [Uploaded(b) for b in sets]
    wants = [oracle_stream(b, u.host_pool, u.host_offs)[0] for b, u in zip(sets, ups)]
    cap_t, cap_b = max(b.n_tensors for b in sets), max(b.n_blocks for b in sets)
    cap = max(len(w) for w in wants) + 4096
    ws = bs.Workspace(cap_t, cap_b, cap, DEV)
    rng = torch.Generator(device=DEV).manual_seed(5)
    cs = bs.current_stream()
    for rnd in range(3):
        for fuse, tune in ((2, 0), (1, 0), (0, 0), (2, 0x10), (1, 0x10)):   # 0x10: tiles handed out by the tagged counter
            for bset, up, want in zip(sets, ups, wants):
                if junk == "ones":
                    ws.buf.fill_(0xFF)
                elif junk == "random":
                    ws.buf.copy_(torch.randint(0, 256, (ws.nbytes,), dtype=torch.uint8, device=DEV, generator=rng))
                total = len(want)
                out = torch.full((cap,), 0xCD, dtype=torch.uint8, device=DEV)
                opts = dict(variant=bs.VARIANT_TMA, fuse=fuse, tune=tune)
                bs.serialize(up.dset.desc, out.data_ptr(), cap, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)
                res = ws.read_result()
                assert res["status"] == bs.OK and res["total_bytes"] == total, (junk, fuse, bset.name, res)
                got = out.cpu().numpy()
                assert (got[:total] == want).all() and (got[total:] == 0xCD).all(), (junk, fuse, bset.name)
                need = oracle.pool_bytes(want)
                dst = bs.DeviceSet.empty(cap_t, cap_b, DEV, fill=0xAB)
                pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
                bs.deserialize(out.data_ptr(), total, dst.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                               ws.result_ptr, opts, cs)
                res = ws.read_result()
                assert res["status"] == bs.OK and res["n_blocks"] == bset.n_blocks, (junk, fuse, bset.name, res)
                assert (pool.cpu().numpy() == oracle.deserialize(want)["pool"][:need]).all()


@pytest.mark.parametrize("opts", [dict(variant=bs.VARIANT_TMA, fuse=2), dict(variant=bs.VARIANT_TMA, fuse=2, tune=0x10),
                                  dict(variant=bs.VARIANT_TMA, fuse=1, tune=0x10)], ids=["fused", "fused-counter", "two-launches-counter"])
def test_fused_calls_on_two_streams_at_once(opts):
    """bs.h: calls are re-entrant.  Two streams each run fused serialize + deserialize calls back to back on their own
    workspaces; the kernels are persistent (one CTA per SM each) and may be co-resident only in part — items are claimed
    from a ticket, so a resident CTA never waits for one that is not (bs_scan_phase.cuh).  Results: the oracle's."""
    bset = W.make_config("2")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total, need = len(want), oracle.pool_bytes(want)
    ref_pool = oracle.deserialize(want)["pool"][:need]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    lanes = []
    for s in streams:
        lanes.append(dict(ws=bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV),
                          out=torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV),
                          dst=bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB),
                          pool=torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)))
    torch.cuda.synchronize()
    for it in range(20):
        for s, ln in zip(streams, lanes):
            bs.serialize(up.dset.desc, ln["out"].data_ptr(), total, ln["ws"].ptr, ln["ws"].nbytes, ln["ws"].result_ptr, opts,
                         s.cuda_stream)
            bs.deserialize(ln["out"].data_ptr(), total, ln["dst"].desc, ln["pool"].data_ptr(), need, bs.LAYOUT_POOL, ln["ws"].ptr,
                           ln["ws"].nbytes, ln["ws"].result_ptr, opts, s.cuda_stream)
    torch.cuda.synchronize()
    for ln in lanes:
        assert ln["ws"].read_result()["status"] == bs.OK
        assert (ln["out"].cpu().numpy() == want).all()
        assert (ln["pool"].cpu().numpy() == ref_pool).all()


@pytest.mark.parametrize("opts", [dict(variant=bs.VARIANT_TMA, tune=0x10), dict(variant=bs.VARIANT_TMA, tile_bytes=49152, stages=3, warps=1, tune=0x1010),
                                  dict(variant=bs.VARIANT_TMA)], ids=_vid)
def test_ranges_of_one_stream_on_two_cuda_streams_share_the_workspace(opts):
    """The segment calls run on the workspace the pass left its tables in, so the halves of one stream issued on two CUDA
    streams use the SAME workspace.  The movement only reads it (round 3: the tile counter of a launch is a pair of the
    library's own ring, not a word of the head — with one shared counter two launches drew tile numbers from the same word
    and skipped tiles with status BS_OK).  Both directions, tiles from the counter: the oracle's bytes every round."""
    bset = W.make_config("2")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total, need = len(want), oracle.pool_bytes(want)
    ref_pool = oracle.deserialize(want)["pool"][:need]
    hb = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
    mid = (hb + (total - hb) // 2) // 16 * 16
    cuts = [(0, mid), (mid, total)]
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    main = torch.cuda.current_stream()
    side = [torch.cuda.Stream(), torch.cuda.Stream()]
    dst = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    for it in range(12):
        out = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
        pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
        # the pass on the main stream, then the two halves side by side
        bs.serialize_range(up.dset.desc, out.data_ptr(), 0, 0, True, ws.ptr, ws.nbytes, ws.result_ptr, opts, main.cuda_stream)
        for s, (lo, hi) in zip(side, cuts):
            s.wait_stream(main)
            bs.serialize_range(up.dset.desc, out.data_ptr() + lo, lo, hi, False, ws.ptr, ws.nbytes, ws.result_ptr, opts, s.cuda_stream)
        for s in side:
            main.wait_stream(s)
        assert ws.read_result()["status"] == bs.OK
        bad = np.nonzero(out.cpu().numpy() != want)[0]
        assert bad.size == 0, f"round {it}: first wrong stream byte {bad[0]} of {total}"
        # the mirror image: bs_deserialize leaves the parsed tables (and fills the pool once); the pool is poisoned again and
        # the two halves are scattered side by side, the first one rebuilding the descriptor arrays as well
        bs.deserialize(out.data_ptr(), total, dst.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr,
                       opts, main.cuda_stream)
        pool.fill_(0xEE)
        for t in (dst.tensors, dst.qn, dst.dim):
            t.fill_(0xAB)
        for s, (lo, hi) in zip(side, cuts):
            s.wait_stream(main)
            bs.deserialize_range(out.data_ptr() + lo, lo, hi, out.data_ptr() if lo == 0 else 0, dst.desc, bs.LAYOUT_POOL, ws.ptr,
                                 ws.nbytes, opts, s.cuda_stream)
        for s in side:
            main.wait_stream(s)
        torch.cuda.synchronize()
        assert ws.read_result()["status"] == bs.OK
        bad = np.nonzero(pool.cpu().numpy() != ref_pool)[0]
        assert bad.size == 0, f"round {it}: first wrong pool byte {bad[0]} of {need}"
        assert bytes(dst.tensors.cpu().numpy()[:32 * bset.n_tensors]) == bset.tensors.tobytes()
        assert (dst.qn.cpu().numpy()[:24 * bset.n_blocks].view(np.int32).reshape(-1, 3, 2) == bset.qn).all()
        assert (dst.dim.cpu().numpy()[:12 * bset.n_blocks].view(np.uint32).reshape(-1, 3) == bset.dim).all()


def test_deserialize_capacity_errors():
    bset = W.make_set("cap", 42, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    want, _, _ = oracle_stream(bset)
    need = oracle.pool_bytes(want)
    st = torch.from_numpy(want.copy()).to(DEV)
    out, pool, res = gpu_deserialize(st, len(want), bset.n_tensors, bset.n_blocks, need - 256)
    assert res["status"] == bs.ERR_CAPACITY and res["pool_bytes"] == need and (pool == 0xEE).all()
    out, pool, res = gpu_deserialize(st, len(want), bset.n_tensors, bset.n_blocks - 1, need)
    assert res["status"] == bs.ERR_CAPACITY and res["n_blocks"] == bset.n_blocks and (pool == 0xEE).all()


def test_scatter_extent_mismatch_is_an_argument_error():
    bset = W.make_set("scat", 51, D=30, S=8, M=2, N0=3, n_ops=5, n_site=0, dims="multinomial")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    wrong = bset.dim.copy()
    wrong[0, 0] += 1
    dst = torch.full((up.pool.numel(),), 0xEE, dtype=torch.uint8, device=DEV)
    daddr = (np.uint64(dst.data_ptr()) + up.host_offs).astype(np.uint64)
    out = bs.DeviceSet.from_host(np.zeros(bset.n_tensors, W.TENSOR_REC_DTYPE), np.zeros_like(bset.qn), wrong, daddr, DEV)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, len(want), DEV)
    st = torch.from_numpy(want.copy()).to(DEV)
    bs.deserialize(st.data_ptr(), len(want), out.desc, 0, 0, bs.SCATTER_TO_ADDR, ws.ptr, ws.nbytes, ws.result_ptr, None,
                   bs.current_stream())
    assert ws.read_result()["status"] == bs.ERR_ARG and (dst == 0xEE).all()


@pytest.mark.parametrize("opts", [None, dict(variant=bs.VARIANT_TMA, tune=0x10), dict(variant=bs.VARIANT_TMA, tune=0x10, fuse=1)],
                         ids=["default", "counter", "counter-two-launches"])
def test_calls_are_capturable_in_a_cuda_graph(opts):
    """The calls only enqueue work (no host synchronisation, no allocation), so a launch-bound loop over small sets can be
    captured once and replayed: the replay must give the oracle's bytes for whatever the blocks hold at replay time.  With
    tiles handed out by the counter (tune 0x10; what large sets do) every replay finds the counter put back by the last one."""
    bset = W.make_config("2", n_ops=26)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    need = oracle.pool_bytes(want)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    stream = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)

    def step(s):
        bs.serialize(up.dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, s)
        bs.deserialize(stream.data_ptr(), total, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                       ws.result_ptr, opts, s)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step(side.cuda_stream)                       # warm-up outside the capture (one-time kernel attributes)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        step(side.cuda_stream)
    # new values in the same blocks, then replay: the graph holds launches, not data
    up.pool.copy_(torch.roll(up.pool, 8))
    rolled = np.roll(up.host_pool.view(np.uint8), 8)
    want2 = oracle.serialize(bset.tensors, bset.qn, bset.dim,
                             (np.uint64(rolled.ctypes.data) + up.host_offs.astype(np.uint64)).astype(np.uint64))
    stream.fill_(0xCD)
    pool.fill_(0xEE)
    for _ in range(3):   # several replays: each must leave the workspace as the next one expects it
        stream.fill_(0xCD)
        pool.fill_(0xEE)
        g.replay()
        torch.cuda.synchronize()
        assert ws.read_result()["status"] == bs.OK
        assert (stream.cpu().numpy() == want2).all(), "graph replay: stream differs from the oracle's"
        assert (pool.cpu().numpy()[:need] == oracle.deserialize(want2)["pool"][:need]).all()
