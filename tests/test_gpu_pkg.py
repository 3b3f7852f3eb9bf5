"""NEXT-2 on the GPU: self-contained packages through the C ABI against oracle/bs_oracle_pkg.c —
bs_package_emit / bs_package_unpack (device slots) and bs_offload_packages_async / bs_prefetch_packages_async (pinned
host slots).  Bit-exact: every slot byte the oracle writes, and nothing else; any order of arrival, foreign slots mixed
in; fault injection on every package-header field."""
import os
import struct

import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from oracle import pkg
from tests.gpu_util import DEV, Uploaded
from tests.util import oracle_stream, read_hex_fixture

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(__file__)
SID = 0x1122334455667788
POISON = 0x5A


def golden_set():
    """The set of the 288-byte golden stream P7, typed out here."""
    tensors = np.zeros(1, W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 2, (1, 1), (-1, 1, 0, 0), 7, 0)
    qn = np.array([[[0, 0], [1, 1], [0, 0]], [[1, -1], [2, 0], [0, 0]]], np.int32)
    dim = np.array([[1, 1, 1], [1, 2, 1]], np.uint32)
    pool = np.zeros(128, np.float64)
    pool[0] = 1.0
    pool[64] = 2.0
    pool[65] = 3.0
    offs = np.array([0, 512], np.uint64)
    return tensors, qn, dim, pool, offs


def upload_raw(tensors, qn, dim, pool, offs):
    d_pool = torch.from_numpy(pool.view(np.uint8).copy()).to(DEV)
    addr = (np.uint64(d_pool.data_ptr()) + offs).astype(np.uint64)
    return d_pool, bs.DeviceSet.from_host(tensors, qn, dim, addr, DEV)


def emit_on_gpu(dset, total, cap, slot_bytes, n_slots, slot_of=None, opts=None, total_arg=None, pkg_ws=True):
    """pkg_ws=False: a plain bs_workspace_bytes workspace (the slot table then comes from a stream-ordered allocation)."""
    slots = torch.full((n_slots * slot_bytes,), POISON, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(dset.n_tensors, dset.n_blocks, max(total, 1 << 16), DEV, packages=pkg_ws)
    bs.package_emit(dset.desc, total if total_arg is None else total_arg, cap, SID, slots.data_ptr(), slot_bytes, n_slots,
                    slot_of, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    return slots, ws.read_result()


def test_golden_package_headers_from_the_gpu():
    gold = read_hex_fixture(os.path.join(HERE, "golden", "g3_package_headers.hex"))
    stream = np.frombuffer(read_hex_fixture(os.path.join(HERE, "golden", "p7_golden_stream.hex")), np.uint8)
    d_pool, dset = upload_raw(*golden_set())
    slots, res = emit_on_gpu(dset, 288, 128, 64 + 128, 3)
    assert res["status"] == bs.OK and res["total_bytes"] == 288 and res["n_packages"] == 3
    got = slots.cpu().numpy().reshape(3, 192)
    assert bytes(got[2, :64]) == gold[0:64] and bytes(got[2, 64:96]) == bytes(stream[256:288])
    assert bytes(got[1, :64]) == gold[128:192] and bytes(got[1, 64:]) == bytes(stream[128:256])
    assert (got[2, 96:] == POISON).all()                      # bytes behind a short package are not written
    slots, res = emit_on_gpu(dset, 288, 16, 64 + 16, 18)
    got = slots.cpu().numpy().reshape(18, 80)
    assert res["n_packages"] == 18
    assert bytes(got[17, :64]) == gold[64:128] and bytes(got[17, 64:]) == bytes(stream[272:288])


CASES = [("1", {}, 4096), ("1", {}, 16), ("2", dict(n_ops=26), 65536), ("2", dict(n_ops=26), 1 << 20),
         ("2", dict(n_ops=26), 48 * 1024 + 16), ("3", dict(n_ops=13, D=600, S=40), 16384)]


@pytest.mark.parametrize("cfg,kw,cap", CASES)
@pytest.mark.parametrize("variant", [bs.VARIANT_TMA, bs.VARIANT_LDG])
def test_emit_matches_the_oracle_slot_for_slot(cfg, kw, cap, variant):
    bset = W.make_config(cfg, **kw)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    hb = bs.header_bytes(bset.n_tensors, bset.n_blocks)
    n = pkg.count(hb, total, cap)
    assert bs.package_count(hb, total, cap) == n
    assert [bs.package_range(hb, total, cap, k) for k in (0, n - 1)] == [pkg.package_range(hb, total, cap, k) for k in (0, n - 1)]
    rng = np.random.default_rng(7)
    n_slots = n + 3
    slot_of = rng.permutation(n_slots)[:n]
    slot_bytes = 64 + cap + 32
    ref = pkg.emit_slots(want, cap, SID, slot_bytes, slot_of=slot_of, n_slots=n_slots, poison=POISON)
    slots, res = emit_on_gpu(up.dset, total, cap, slot_bytes, n_slots, slot_of, opts=dict(variant=variant))
    assert res["status"] == bs.OK and res["total_bytes"] == total and res["n_packages"] == n
    got = slots.cpu().numpy().reshape(n_slots, slot_bytes)
    assert (got == ref).all(), "GPU packages differ from the oracle's"
    assert bytes(pkg.assemble(got, SID)) == bytes(want)        # the paper's property, by the oracle's reassembly


def test_emit_size_zero_means_query_and_a_wrong_prediction_is_an_error():
    bset = W.make_config("1")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    hb = bs.header_bytes(bset.n_tensors, bset.n_blocks)
    n = pkg.count(hb, total, 4096)
    ref = pkg.emit_slots(want, 4096, SID, 64 + 4096, poison=POISON)
    slots, res = emit_on_gpu(up.dset, total, 4096, 64 + 4096, n, total_arg=0)
    assert res["status"] == bs.OK and (slots.cpu().numpy().reshape(n, -1) == ref).all()
    slots, res = emit_on_gpu(up.dset, total, 4096, 64 + 4096, n + 1, total_arg=total + 16)
    assert res["status"] == bs.ERR_ARG and (slots.cpu().numpy() == POISON).all()   # nothing written
    for bad in (dict(cap=4100), dict(slot_bytes=64 + 4096 - 16), dict(n_slots=n - 1), dict(slot_of=[0] * n),
                dict(slot_of=list(range(1, n + 1)))):
        a = dict(cap=4096, slot_bytes=64 + 4096, n_slots=n, slot_of=None)
        a.update(bad)
        with pytest.raises(bs.BsError) as e:
            emit_on_gpu(up.dset, total, a["cap"], a["slot_bytes"], a["n_slots"], a["slot_of"])
        assert e.value.code == (bs.ERR_CAPACITY if "n_slots" in bad else bs.ERR_ARG)


def oracle_slots(want, cap, slot_bytes, seed, extra=2, foreign=True):
    """The oracle's packages in shuffled slots, with poisoned spare slots and (optionally) a foreign stream's packages."""
    hb = int(np.frombuffer(want[48:56].tobytes(), "<u8")[0])
    n = pkg.count(hb, len(want), cap)
    rng = np.random.default_rng(seed)
    n_slots = n + extra + (2 if foreign else 0)
    perm = rng.permutation(n_slots)
    slots = pkg.emit_slots(want, cap, SID, slot_bytes, slot_of=perm[:n], n_slots=n_slots, poison=POISON)
    if foreign:  # "mixed with other packages" (L124): two packages of another serialization call
        other = pkg.emit_slots(want, cap, SID + 1, slot_bytes)
        slots[perm[n]] = other[0]
        slots[perm[n + 1]] = other[-1]
    return slots, perm[:n], n


def unpack_on_gpu(slots_np, bset, want, flags=bs.LAYOUT_POOL, opts=None, sid=SID, pkg_ws=True):
    need = oracle.pool_bytes(want)
    n_slots, slot_bytes = slots_np.shape
    d_slots = torch.from_numpy(slots_np.copy()).to(DEV)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((max(need, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, max(len(want), 1 << 16), DEV, packages=True)
    if not pkg_ws:   # the smallest workspace the call accepts: v1 workspace + the header region, no room for the slot table
        ws.nbytes = bs.workspace_bytes(bset.n_tensors, bset.n_blocks, max(len(want), 1 << 16)) + \
            (bs.header_bytes(bset.n_tensors, bset.n_blocks) + 255) // 256 * 256
    bs.package_unpack(d_slots.data_ptr(), slot_bytes, n_slots, sid, out.desc, pool.data_ptr(), need, flags, ws.ptr, ws.nbytes,
                      ws.result_ptr, opts, bs.current_stream())
    return out, pool, ws.read_result(), need


@pytest.mark.parametrize("cfg,kw,cap", CASES)
@pytest.mark.parametrize("variant", [bs.VARIANT_TMA, bs.VARIANT_LDG])
def test_unpack_from_shuffled_oracle_packages(cfg, kw, cap, variant):
    bset = W.make_config(cfg, **kw)
    want, _, _ = oracle_stream(bset)
    ref = oracle.deserialize(want)
    slots, _, _ = oracle_slots(want, cap, 64 + cap + 16, seed=11)
    out, pool, res, need = unpack_on_gpu(slots, bset, want, opts=dict(variant=variant))
    assert res["status"] == bs.OK and res["n_tensors"] == bset.n_tensors and res["n_blocks"] == bset.n_blocks
    assert res["total_bytes"] == len(want) and res["pool_bytes"] == need
    assert (pool.cpu().numpy()[:need] == ref["pool"][:need]).all(), "blocks differ from the oracle's"
    h = out.to_host()
    assert h["tensors"].tobytes() == bset.tensors.tobytes() and (h["qn"] == bset.qn).all() and (h["dim"] == bset.dim).all()


@pytest.mark.parametrize("tile,cap", [(32768, 65536), (32768, 49152), (65536, 1 << 20), (49152, 49152 * 3)])
@pytest.mark.parametrize("variant", [bs.VARIANT_TMA, bs.VARIANT_LDG])
def test_the_stream_does_not_depend_on_how_packages_map_onto_work_tiles(tile, cap, variant):
    """P6 for packages: limits that are a multiple of the work tile take the one-launch path, the others go package by
    package; both must give the oracle's bytes."""
    bset = W.make_config("2", n_ops=39)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    ref = oracle.deserialize(want)
    hb = bs.header_bytes(bset.n_tensors, bset.n_blocks)
    n = pkg.count(hb, len(want), cap)
    slot_of = np.random.default_rng(1).permutation(n)
    opts = dict(variant=variant, tile_bytes=tile, stages=3, warps=1)
    slots, res = emit_on_gpu(up.dset, len(want), cap, 64 + cap, n, slot_of, opts=opts, pkg_ws=variant == bs.VARIANT_TMA)
    got = slots.cpu().numpy().reshape(n, 64 + cap)
    assert res["status"] == bs.OK
    assert (got == pkg.emit_slots(want, cap, SID, 64 + cap, slot_of=slot_of, poison=POISON)).all()
    out, pool, res2, need = unpack_on_gpu(got, bset, want, opts=opts, pkg_ws=variant == bs.VARIANT_TMA)
    assert res2["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


def test_emit_then_unpack_on_the_device_is_the_identity():
    bset = W.make_config("2", n_ops=39)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    ref = oracle.deserialize(want)
    cap = 256 * 1024
    hb = bs.header_bytes(bset.n_tensors, bset.n_blocks)
    n = pkg.count(hb, len(want), cap)
    slot_of = np.random.default_rng(3).permutation(n)
    slots, res = emit_on_gpu(up.dset, len(want), cap, 64 + cap, n, slot_of)
    assert res["status"] == bs.OK
    out, pool, res2, need = unpack_on_gpu(slots.cpu().numpy().reshape(n, 64 + cap), bset, want)
    assert res2["status"] == bs.OK and (pool.cpu().numpy()[:need] == ref["pool"][:need]).all()


FIELDS = dict(version=(8, "<I"), index=(12, "<I"), count=(16, "<I"), first_block=(20, "<I"), total_bytes=(32, "<Q"),
              lo=(40, "<Q"), nbytes=(48, "<Q"), first_block_offset=(56, "<Q"))


@pytest.mark.parametrize("field", sorted(FIELDS))
@pytest.mark.parametrize("which", ["header_region", "payload"])
def test_unpack_rejects_a_package_that_lies_about_its_place(field, which):
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    want, _, _ = oracle_stream(bset)
    cap = 1024
    slots, slot_of, n = oracle_slots(want, cap, 64 + cap, seed=5, foreign=False)
    hb = int(np.frombuffer(want[48:56].tobytes(), "<u8")[0])
    nh = -(-hb // cap)
    assert nh >= 2 and n - nh >= 3
    k = 1 if which == "header_region" else nh + 1
    off, fmt = FIELDS[field]
    s = int(slot_of[k])
    (v,) = struct.unpack_from(fmt, slots[s].tobytes(), off)
    bump = 16 if field in ("lo", "nbytes", "total_bytes", "first_block_offset") else 1
    slots[s, off:off + struct.calcsize(fmt)] = np.frombuffer(struct.pack(fmt, (v + bump) & (2 ** (8 * struct.calcsize(fmt)) - 1)), np.uint8)
    with pytest.raises(oracle.OracleError):
        if field in ("first_block", "first_block_offset"):
            raise oracle.OracleError(-3, "the oracle's reassembly does not look at these two fields")
        pkg.assemble(slots, SID)
    try:
        out, pool, res, need = unpack_on_gpu(slots, bset, want)
        status = res["status"]
    except bs.BsError as e:       # the host-side plan refused
        status, pool, out = e.code, None, None
    assert status == bs.ERR_CORRUPT
    if pool is not None:          # refused on the device: nothing was written
        assert (pool.cpu().numpy() == 0xEE).all() and (out.tensors.cpu().numpy() == 0xAB).all()


def test_unpack_rejects_missing_and_duplicate_packages_and_a_corrupt_stream_header():
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    want, _, _ = oracle_stream(bset)
    cap = 1024
    slots, slot_of, n = oracle_slots(want, cap, 64 + cap, seed=9, foreign=False)
    missing = slots.copy()
    missing[int(slot_of[n - 2])] = POISON
    dup = slots.copy()
    spare = [s for s in range(slots.shape[0]) if s not in set(slot_of.tolist())][0]
    dup[spare] = slots[int(slot_of[3])]
    for bad in (missing, dup):
        with pytest.raises(oracle.OracleError):
            pkg.assemble(bad, SID)
        with pytest.raises(bs.BsError) as e:
            unpack_on_gpu(bad, bset, want)
        assert e.value.code == bs.ERR_CORRUPT
    with pytest.raises(bs.BsError) as e:                       # no package of this stream id at all
        unpack_on_gpu(slots, bset, want, sid=SID + 5)
    assert e.value.code == bs.ERR_CORRUPT
    # the stream's own header is validated as in bs_deserialize: flip one offset inside a header-region package
    hb = int(np.frombuffer(want[48:56].tobytes(), "<u8")[0])
    bad_stream = want.copy()
    rec = 64 + 32 * bset.n_tensors + 48 * 5 + 40
    bad_stream[rec] ^= 0x10
    with pytest.raises(oracle.OracleError):
        oracle.deserialize(bad_stream)
    bslots = pkg.emit_slots(bad_stream, cap, SID, 64 + cap)
    out, pool, res, need = unpack_on_gpu(bslots, bset, want)
    assert res["status"] == bs.ERR_CORRUPT and (pool.cpu().numpy() == 0xEE).all()


def pinned(n, fill):
    t = torch.empty(max(n, 16), dtype=torch.uint8, pin_memory=True)
    t.fill_(fill)
    return t


@pytest.mark.parametrize("cap,chunk,n_staging", [(65536 - 64, 65536, 2), (200 * 1024, 4 * 65536, 3), (1 << 20, 1 << 24, 1)])
def test_engine_offload_packages_then_prefetch_them_in_any_order(cap, chunk, n_staging):
    bset = W.make_config("2", n_ops=52)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    hb = bs.header_bytes(bset.n_tensors, bset.n_blocks)
    n = pkg.count(hb, total, cap)
    slot_bytes = 64 + cap
    n_slots = n + 2
    slot_of = np.random.default_rng(21).permutation(n_slots)[:n]
    ref_slots = pkg.emit_slots(want, cap, SID, slot_bytes, slot_of=slot_of, n_slots=n_slots, poison=POISON)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total + 4096, chunk_bytes=chunk, n_staging=n_staging)
    host = pinned(n_slots * slot_bytes, POISON)
    t = eng.offload_packages_async(up.dset.desc, total, cap, SID, host.data_ptr(), slot_bytes, n_slots, slot_of,
                                   bs.current_stream())
    st = t.wait()
    assert st["status"] == bs.OK and st["n_chunks"] == n and st["bytes"] == total + 64 * n
    got = host.numpy().reshape(n_slots, slot_bytes)
    assert (got == ref_slots).all(), "host packages differ from the oracle's"

    # the receive side: the slots as they lie (shuffled, two of them foreign poison)
    ref = oracle.deserialize(want)
    need = oracle.pool_bytes(want)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    t2 = eng.prefetch_packages_async(host.data_ptr(), slot_bytes, n_slots, SID, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL,
                                     bs.current_stream())
    snapshot = pool.clone()       # the consumer stream waits on the ticket's event (checkpoint)
    st2 = t2.wait()
    assert st2["status"] == bs.OK, st2
    assert (snapshot.cpu().numpy() == ref["pool"][:need]).all()
    h = out.to_host()
    assert h["tensors"].tobytes() == bset.tensors.tobytes() and (h["qn"] == bset.qn).all() and (h["dim"] == bset.dim).all()

    # a payload package that lies about its first block: refused on the device, nothing written
    k = n - 1
    s = int(slot_of[k])
    bad = pinned(n_slots * slot_bytes, 0)
    bad.copy_(host)
    b = bad.numpy().reshape(n_slots, slot_bytes)
    (fb,) = struct.unpack_from("<I", b[s].tobytes(), 20)
    b[s, 20:24] = np.frombuffer(struct.pack("<I", fb - 1), np.uint8)
    pool.fill_(0xEE)
    t3 = eng.prefetch_packages_async(bad.data_ptr(), slot_bytes, n_slots, SID, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL,
                                     bs.current_stream())
    assert t3.wait()["status"] == bs.ERR_CORRUPT
    torch.cuda.synchronize()
    assert (pool.cpu().numpy() == 0xEE).all()
    with pytest.raises(bs.BsError) as e:
        eng.offload_packages_async(up.dset.desc, total, chunk, SID, host.data_ptr(), 64 + chunk, n_slots, None,
                                   bs.current_stream())
    assert e.value.code in (bs.ERR_CAPACITY, bs.ERR_ARG)
    eng.destroy()


@pytest.mark.parametrize("cap,chunk,n_staging", [(32768, 5 * 65536, 2), (16384, 65536, 3), (49152, 8 * 65536, 1), (32768 + 16, 4 * 65536, 2)])
def test_engine_batches_consecutive_slots_per_staging_buffer(cap, chunk, n_staging):
    """Slots in stream order (no slot map): several packages share a staging buffer, leave in one DMA, and — for limits
    that are a multiple of the work tile — are packed by one launch.  The bytes are the oracle's either way, and the poison
    behind the two short packages (end of the header region, end of the payload) and behind the last slot survives."""
    bset = W.make_config("2", n_ops=39)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    total = len(want)
    hb = bs.header_bytes(bset.n_tensors, bset.n_blocks)
    n = pkg.count(hb, total, cap)
    slot_bytes = 64 + cap
    ref_slots = pkg.emit_slots(want, cap, SID, slot_bytes, n_slots=n + 1, poison=POISON)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total + 4096, chunk_bytes=chunk, n_staging=n_staging)
    host = pinned((n + 1) * slot_bytes, POISON)
    st = eng.offload_packages_async(up.dset.desc, total, cap, SID, host.data_ptr(), slot_bytes, n + 1, None, bs.current_stream()).wait()
    assert st["status"] == bs.OK and st["n_chunks"] == n
    got = host.numpy().reshape(n + 1, slot_bytes)
    assert (got == ref_slots).all(), "host packages differ from the oracle's"
    ref = oracle.deserialize(want)
    need = oracle.pool_bytes(want)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    st2 = eng.prefetch_packages_async(host.data_ptr(), slot_bytes, n + 1, SID, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL,
                                      bs.current_stream()).wait()
    torch.cuda.synchronize()
    assert st2["status"] == bs.OK and (pool.cpu().numpy() == ref["pool"][:need]).all()
    eng.destroy()


# ---- packages of layered sets (wire format v2) ------------------------------------------------------------------------------
@pytest.mark.parametrize("cap", [16384, 65536, 4096 + 16, 1 << 20])
@pytest.mark.parametrize("variant", [bs.VARIANT_TMA, bs.VARIANT_LDG])
def test_layered_packages_match_the_oracle_and_unpack_in_any_order(cap, variant):
    from oracle import v2
    from tests.test_gpu_layered import LayeredUp
    bset = W.make_config("2", n_ops=39)
    lu = LayeredUp(bset)
    want = lu.want
    total = len(want)
    c = lu.counts
    hb = bs.layered_header_bytes(c[0], c[2], c[1])
    n = pkg.count(hb, total, cap)
    slot_bytes = 64 + cap
    slot_of = np.random.default_rng(8).permutation(n + 2)[:n]
    ref_slots = pkg.emit_slots(want, cap, SID, slot_bytes, slot_of=slot_of, n_slots=n + 2, poison=POISON)
    slots = torch.full(((n + 2) * slot_bytes,), POISON, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(0, 0, max(total, 1 << 16), DEV, layered=c, packages=True)
    opts = dict(variant=variant)
    bs.layered_package_emit(lu.dset.desc, total, cap, SID, slots.data_ptr(), slot_bytes, n + 2, slot_of, ws.ptr, ws.nbytes,
                            ws.result_ptr, opts, bs.current_stream())
    res = ws.read_result()
    assert res["status"] == bs.OK and res["total_bytes"] == total and res["n_packages"] == n and res["n_structs"] == c[0]
    got = slots.cpu().numpy().reshape(n + 2, slot_bytes)
    assert (got == ref_slots).all(), "layered packages differ from the oracle's"
    # and back, from the oracle's slots with two foreign packages mixed in
    other = pkg.emit_slots(want, cap, SID + 1, slot_bytes)
    spare = [s for s in range(n + 2) if s not in set(slot_of.tolist())]
    ref_slots[spare[0]] = other[0]
    ref_slots[spare[1]] = other[-1]
    ref = v2.deserialize(want)
    na, need = v2.counts(want)
    out = bs.DeviceLayeredSet.empty(*c, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    d_slots = torch.from_numpy(ref_slots.copy()).to(DEV)
    bs.layered_package_unpack(d_slots.data_ptr(), slot_bytes, n + 2, SID, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr,
                              ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need
    assert (pool.cpu().numpy() == ref["pool"][:need]).all()
    h = out.to_host(*c)
    assert h["structs"].tobytes() == ref["structs"].tobytes() and h["layers"].tobytes() == ref["layers"].tobytes()
    # a payload package that lies about its first block is refused on the device, nothing written
    k = n - 1
    s = int(slot_of[k])
    (fb,) = struct.unpack_from("<I", ref_slots[s].tobytes(), 20)
    ref_slots[s, 20:24] = np.frombuffer(struct.pack("<I", fb + 1), np.uint8)
    pool.fill_(0xEE)
    d_slots = torch.from_numpy(ref_slots.copy()).to(DEV)
    bs.layered_package_unpack(d_slots.data_ptr(), slot_bytes, n + 2, SID, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr,
                              ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    assert ws.read_result()["status"] == bs.ERR_CORRUPT and (pool.cpu().numpy() == 0xEE).all()


@pytest.mark.parametrize("cap,chunk,shuffle", [(32768, 5 * 65536, False), (65536, 4 * 65536 + 65536, True), (4096 + 16, 65536, False)])
def test_engine_layered_packages_round_trip(cap, chunk, shuffle):
    from oracle import v2
    from tests.test_gpu_layered import LayeredUp
    bset = W.make_config("2", n_ops=39)
    lu = LayeredUp(bset)
    want = lu.want
    total = len(want)
    c = lu.counts
    hb = bs.layered_header_bytes(c[0], c[2], c[1])
    n = pkg.count(hb, total, cap)
    slot_bytes = 64 + cap
    slot_of = np.random.default_rng(12).permutation(n + 1)[:n] if shuffle else None
    ref_slots = pkg.emit_slots(want, cap, SID, slot_bytes, slot_of=slot_of, n_slots=n + 1, poison=POISON)
    eng = bs.Engine(max(c[0], c[2]), max(c[1], c[3]), total + 4096, chunk_bytes=chunk, n_staging=2)
    host = pinned((n + 1) * slot_bytes, POISON)
    st = eng.offload_layered_packages_async(lu.dset.desc, total if shuffle else 0, cap, SID, host.data_ptr(), slot_bytes, n + 1,
                                            slot_of, bs.current_stream()).wait()
    assert st["status"] == bs.OK and st["n_chunks"] == n
    assert (host.numpy().reshape(n + 1, slot_bytes) == ref_slots).all(), "host packages differ from the oracle's"
    ref = v2.deserialize(want)
    na, need = v2.counts(want)
    out = bs.DeviceLayeredSet.empty(*c, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    st2 = eng.prefetch_layered_packages_async(host.data_ptr(), slot_bytes, n + 1, SID, out.desc, pool.data_ptr(), need,
                                              bs.LAYOUT_POOL, bs.current_stream()).wait()
    torch.cuda.synchronize()
    assert st2["status"] == bs.OK and (pool.cpu().numpy() == ref["pool"][:need]).all()
    h = out.to_host(*c)
    assert h["structs"].tobytes() == ref["structs"].tobytes() and h["layers"].tobytes() == ref["layers"].tobytes()
    eng.destroy()
