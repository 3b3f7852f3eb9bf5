"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default opts): configs 3 and 4 as their
recipes count (2.2 GB, 7.2 GB) and 3L / 4L, the operator count scaled to the totals BASELINE.json states (11 GB, 42.5 GB;
SURVEY §8(d) R1).  EVERY byte of the stream and of the deserialized pool is compared with the C oracle, which runs
slice-wise over all tensor ranges on a host copy of the seeded source pool (tests/fullsize.py) — never a byte from the CUDA
path.  On top: exact size prediction, the fixpoint serialize(deserialize(S)) == S on the device, chunked offload == the stream."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from tests.fullsize import DeviceReader, HostPool, check_against_oracle
from tests.gpu_util import DEV, Uploaded

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def sampled_tensors(bset, n=10, seed=7):
    per_t = np.add.reduceat(bset.nelems, bset.tensors["first_block"].astype(np.int64))
    rng = np.random.default_rng(seed)
    pick = {0, bset.n_tensors - 1, int(np.argmax(per_t)), int(np.argmin(per_t))}
    pick |= set(int(x) for x in rng.choice(bset.n_tensors, size=n, replace=False))
    return sorted(pick)


def oracle_tensor_payload(bset, t):
    """(first payload offset, bytes) of tensor t from the oracle, block values regenerated on the host."""
    b0 = int(bset.tensors["first_block"][t])
    b1 = b0 + int(bset.tensors["n_blocks"][t])
    pool, offs = W.fill_pool_host(bset, b0, b1, compact=True)
    addr = np.zeros(bset.n_blocks, np.uint64)
    addr[b0:b1] = np.uint64(pool.ctypes.data) + offs
    cap = int(((bset.nelems[b0:b1] * 8 + 15) // 16 * 16).sum())
    first, got = oracle.emit_payload_range(bset.tensors, bset.dim, addr, t, t + 1, cap)
    assert len(got) == cap
    return first, got, pool


def _room_for(cfg, bset):
    """3L / 4L run whenever the box can hold them: source pool + stream + deserialized pool in HBM, the source pool once more
    in host RAM for the oracle."""
    need_dev = int(bset.pool_bytes) + 2 * (bset.data_bytes + 64 * bset.n_blocks + (64 << 20)) + (2 << 30)
    import gc
    gc.collect()
    torch.cuda.empty_cache()   # what earlier tests freed sits in torch's cache, not in the driver's free list
    free_dev, _ = torch.cuda.mem_get_info()
    if need_dev > free_dev:
        pytest.skip(f"config {cfg} needs {need_dev / 1e9:.0f} GB of HBM, {free_dev / 1e9:.0f} GB are free")
    import psutil
    need_host = int(bset.pool_bytes) + (6 << 30)
    if need_host > psutil.virtual_memory().available:
        pytest.skip(f"config {cfg} needs {need_host / 1e9:.0f} GB of host RAM for the oracle's copy of the source pool")


@pytest.mark.parametrize("cfg", ["3", "4", "3L", "4L"])
def test_full_size_serialize_deserialize(cfg):
    bset = W.make_config(cfg)
    _room_for(cfg, bset)
    up = Uploaded(bset, fill="device")
    hp = HostPool(bset, up.pool)
    rd, rd2 = DeviceReader(), DeviceReader()
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    cs = bs.current_stream()
    # exact size prediction before serialization
    assert bs.serialized_size(up.dset.desc, ws.ptr, ws.nbytes, cs) == (hb, total)
    stream = torch.full((total + 4096,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.serialize(up.dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and (res["header_bytes"], res["total_bytes"]) == (hb, total)
    assert bool((stream[total:] == 0xCD).all()), "bytes beyond the stream were written"

    # deserialize: descriptor identical; the pool is compared below, together with the stream
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                   ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need
    host = out.to_host()
    assert host["tensors"].tobytes() == bset.tensors.tobytes()
    assert (host["qn"] == bset.qn).all() and (host["dim"] == bset.dim).all()
    slots = (bset.nelems * 8 + 255) // 256 * 256
    want_addr = opool.data_ptr() + np.concatenate([[0], np.cumsum(slots)[:-1]]).astype(np.uint64)
    assert (host["addr"] == want_addr.astype(np.uint64)).all()          # D14 pool layout

    # 100 % of the stream (header + every payload byte) and 100 % of the pool image (every block, every untouched byte
    # of every align256 slot) against the oracle
    n_payload, n_pool = check_against_oracle(
        bset, hp.addr, header=rd.read(stream, 0, hb).copy(),
        payload_reader=lambda lo, n: rd.read(stream, hb + lo, n),
        pool_reader=lambda lo, n: rd2.read(opool, lo, n), hb=hb, total=total, need=need)
    assert n_payload == total - hb and n_pool == need

    # fixpoint on the device, every byte: serialize(deserialize(S)) == S
    del up.pool, hp                       # 4L: source + stream + pool + second stream would not fit in 180 GB
    up.dset = None
    torch.cuda.empty_cache()
    again = torch.full((total,), 0x11, dtype=torch.uint8, device=DEV)
    bs.serialize(out.desc, again.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK
    assert torch.equal(again, stream[:total]), "serialize(deserialize(S)) != S"


@pytest.mark.parametrize("cfg", ["3", "3L"])
def test_full_size_offload_prefetch_config3(cfg):
    """config 5's data path at full size — config 3 as its recipe counts (2.2 GB, 9 chunks) and at the total BASELINE.json
    states for it (3L: 11 GB, 42 chunks): 256 MiB double-buffered chunks.  The host bytes (concat(chunks), D15) and the
    prefetched pool, every byte, against the ORACLE's stream and pool image — not against bs_serialize."""
    bset = W.make_config(cfg)
    _room_for(cfg, bset)
    import psutil
    if int(bset.pool_bytes) + int(bset.data_bytes) + (8 << 30) > psutil.virtual_memory().available:
        pytest.skip(f"config {cfg}: no host RAM for the pinned stream beside the oracle's copy of the source pool")
    up = Uploaded(bset, fill="device")
    hp = HostPool(bset, up.pool)
    rd = DeviceReader()
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    cs = bs.current_stream()
    host = torch.empty(total + 4096, dtype=torch.uint8, pin_memory=True)
    host.fill_(0x5A)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total)        # defaults: 256 MiB chunks, 2 staging buffers
    st = eng.offload_async(up.dset.desc, total, host.data_ptr(), total, cs).wait()
    assert st["status"] == bs.OK and st["bytes"] == total and st["n_chunks"] == (total + (256 << 20) - 1) // (256 << 20)
    hn = host.numpy()
    assert (hn[total:] == 0x5A).all(), "the engine wrote beyond the stream"
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    st = eng.prefetch_async(host.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs).wait()
    torch.cuda.synchronize()
    assert st["status"] == bs.OK
    check_against_oracle(bset, hp.addr, header=hn[:hb], payload_reader=lambda lo, n: hn[hb + lo: hb + lo + n],
                         pool_reader=lambda lo, n: rd.read(opool, lo, n), hb=hb, total=total, need=need)
    a = out.to_host()
    assert a["tensors"].tobytes() == bset.tensors.tobytes() and (a["qn"] == bset.qn).all() and (a["dim"] == bset.dim).all()
    slots = (bset.nelems * 8 + 255) // 256 * 256
    want_addr = opool.data_ptr() + np.concatenate([[0], np.cumsum(slots)[:-1]]).astype(np.uint64)
    assert (a["addr"] == want_addr.astype(np.uint64)).all()
    eng.destroy()


@pytest.mark.parametrize("cfg", ["3", "4"])
def test_full_size_layered_v2(cfg):
    """Wire format v2 (structure-shared layers) at full size, default launch configuration: the whole header against
    the v2 oracle's plan read by the independent struct reader, EVERY payload byte against the v1 oracle's slice-wise
    payload (pinned relation: identical payload), every pool byte against the oracle's pool image, size prediction,
    device fixpoint."""
    from oracle import v2
    bset = W.make_config(cfg)
    up = Uploaded(bset, fill="device")
    hp = HostPool(bset, up.pool)
    rd, rd2 = DeviceReader(), DeviceReader()
    lv = W.layered_view(bset)
    counts = (len(lv["structs"]), lv["dim"].shape[0], bset.n_tensors, bset.n_blocks)
    dset = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], up.addr, DEV)
    hb, total = v2.serialized_size(lv["structs"], lv["layers"], lv["dim"])
    hb1, total1 = oracle.serialized_size(bset.n_tensors, bset.dim)
    assert total - hb == total1 - hb1 and hb * 20 < hb1
    cs = bs.current_stream()
    ws = bs.Workspace(0, 0, total, DEV, layered=counts)
    assert bs.layered_serialized_size(dset.desc, ws.ptr, ws.nbytes, cs) == (hb, total)
    stream = torch.full((total + 4096,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.layered_serialize(dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and (res["header_bytes"], res["total_bytes"]) == (hb, total)
    assert bool((stream[total:] == 0xCD).all())
    # header: the oracle's plan, written out by the independent struct reader's field list
    from tests.streamreader import read_stream_v2
    plan = v2.plan(lv["structs"], lv["layers"], lv["dim"])
    fixed, structs, layers, blocks, slack, _ = read_stream_v2(stream[:hb].cpu().numpy().tobytes() + b"")
    assert (fixed["n_structs"], fixed["n_struct_blocks"], fixed["n_layers"], fixed["header_bytes"], fixed["payload_bytes"]) == \
        (counts[0], counts[1], counts[2], hb, total - hb)
    assert [s["layer_bytes"] for s in structs] == plan["layer_bytes"].tolist()
    assert [l["offset"] for l in layers] == plan["layer_offset"].tolist()
    assert [l["structure"] for l in layers] == lv["layers"]["structure"].tolist()
    assert [b["offset"] for b in blocks] == plan["rel_offset"].tolist()
    assert [b["dim"] for b in blocks] == [tuple(int(x) for x in d) for d in lv["dim"]]
    assert set(slack) <= {0}
    # deserialize
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceLayeredSet.empty(*counts, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.layered_deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                           ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need and res["n_blocks"] == bset.n_blocks
    h = out.to_host(*counts)
    assert (h["qn"] == lv["qn"]).all() and (h["dim"] == lv["dim"]).all()
    slots = (bset.nelems * 8 + 255) // 256 * 256
    want_addr = opool.data_ptr() + np.concatenate([[0], np.cumsum(slots)[:-1]]).astype(np.uint64)
    assert (h["addr"] == want_addr.astype(np.uint64)).all()
    # every payload byte and every pool byte against the oracle (the v2 payload is the v1 payload of the same tensors)
    check_against_oracle(bset, hp.addr, payload_reader=lambda lo, n: rd.read(stream, hb + lo, n),
                         pool_reader=lambda lo, n: rd2.read(opool, lo, n), hb=hb, total=total, need=need)
    again = torch.full((total,), 0x11, dtype=torch.uint8, device=DEV)
    bs.layered_serialize(out.desc, again.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK
    assert torch.equal(again, stream[:total]), "serialize(deserialize(S)) != S"


def test_full_size_packages_config4():
    """NEXT-2 at full size in the configuration bench.py times: 4 MiB limit (1719 packages), shuffled slots, one launch.
    Every stream byte is read out of the slots with the ORACLE's cut and compared with the oracle's stream."""
    import struct
    from oracle import pkg
    bset = W.make_config("4")
    up = Uploaded(bset, fill="device")
    hp = HostPool(bset, up.pool)
    rd = DeviceReader()
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    cap, sid = 4 << 20, 0xC0FFEE
    n = pkg.count(hb, total, cap)
    slot_bytes = 64 + cap
    slot_of = np.random.default_rng(4).permutation(n)
    slots = torch.full((n * slot_bytes,), 0x5A, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV, packages=True)
    cs = bs.current_stream()
    bs.package_emit(up.dset.desc, total, cap, sid, slots.data_ptr(), slot_bytes, n, slot_of, ws.ptr, ws.nbytes, ws.result_ptr,
                    None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["n_packages"] == n and res["total_bytes"] == total
    gather = torch.empty(512 << 20, dtype=torch.uint8, device=DEV)

    def stream_range(lo, nbytes):
        """Stream bytes [lo, lo+nbytes) out of the slots, located with the ORACLE's cut."""
        nonlocal gather
        if nbytes > gather.numel():
            gather = torch.empty(int(nbytes * 1.25), dtype=torch.uint8, device=DEV)
        nh = -(-hb // cap)
        pos = 0
        while pos < nbytes:
            k = lo // cap if lo < hb else nh + (lo - hb) // cap
            plo, phi = pkg.package_range(hb, total, cap, k)
            take = min(nbytes - pos, phi - lo)
            base = int(slot_of[k]) * slot_bytes + 64 + (lo - plo)
            gather[pos: pos + take].copy_(slots[base: base + take])      # plain device copy of a located range
            lo += take
            pos += take
        return rd.read(gather, 0, nbytes)

    check_against_oracle(bset, hp.addr, header=stream_range(0, hb).copy(),
                         payload_reader=lambda lo, m: stream_range(hb + lo, m), hb=hb, total=total)
    # package headers: the oracle's cut; first_block by numpy.searchsorted over the oracle's offsets
    want_h = oracle.emit_header(bset.tensors, bset.qn, bset.dim)
    offs = np.frombuffer(want_h[64 + 32 * bset.n_tensors: 64 + 32 * bset.n_tensors + 48 * bset.n_blocks].tobytes(),
                         dtype=np.dtype([("x", "V40"), ("off", "<u8")]))["off"]
    for k in [0, 1, n - 1] + [int(x) for x in np.random.default_rng(5).integers(0, n, 24)]:
        lo, hi = pkg.package_range(hb, total, cap, k)
        raw = slots[int(slot_of[k]) * slot_bytes: int(slot_of[k]) * slot_bytes + 64].cpu().numpy().tobytes()
        magic, ver, idx, cnt, fb, psid, ptot, plo, pnb, intra = struct.unpack("<8sIIIIQQQQQ", raw)
        assert (magic, ver, idx, cnt, psid, ptot, plo, pnb) == (b"BSPKG001", 1, k, n, sid, total, lo, hi - lo)
        if lo < hb:
            assert fb == 0xFFFFFFFF and intra == 0
        else:
            i = int(np.searchsorted(offs, lo - hb, side="right")) - 1
            assert fb == i and intra == lo - hb - int(offs[i])
    for k in range(0, n, max(1, n // 40)):   # bytes behind a short package stay untouched
        lo, hi = pkg.package_range(hb, total, cap, k)
        tail = slots[int(slot_of[k]) * slot_bytes + 64 + (hi - lo): (int(slot_of[k]) + 1) * slot_bytes]
        assert bool((tail == 0x5A).all())
    # and back: one-launch unpack from the shuffled slots; every pool byte against the oracle
    del gather
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.package_unpack(slots.data_ptr(), slot_bytes, n, sid, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                      ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need
    host = out.to_host()
    assert host["tensors"].tobytes() == bset.tensors.tobytes() and (host["qn"] == bset.qn).all() and (host["dim"] == bset.dim).all()
    check_against_oracle(bset, hp.addr, pool_reader=lambda lo, m: rd.read(opool, lo, m), need=need)


def test_full_size_queue_config3():
    """NEXT-3 at full size: the bench's e2e pattern — save a set while the stream saved before it is loaded back.  The saved
    host bytes and the loaded pool, every byte, against the oracle."""
    bset = W.make_config("3")
    up = Uploaded(bset, fill="device")
    hp = HostPool(bset, up.pool)
    rd = DeviceReader()
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    cs = bs.current_stream()
    q = bs.Queue(bset.n_tensors, bset.n_blocks, total)                 # defaults: 256 MiB chunks, 2 staging buffers per lane
    hosts = [torch.empty(total, dtype=torch.uint8, pin_memory=True) for _ in range(2)]
    for h in hosts:
        h.fill_(0x5A)
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    q.save(0, up.dset.desc, total, hosts[0].data_ptr(), total, cs)
    q.save(1, up.dset.desc, total, hosts[1].data_ptr(), total, cs)    # runs behind save 0 in the save lane ...
    q.load(0, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)   # ... while the load lane brings key 0 back
    for k in (0, 1):
        st = q.wait(k)
        assert st["status"] == bs.OK and st["save"]["bytes"] == total
    torch.cuda.synchronize()
    h0 = hosts[0].numpy()
    check_against_oracle(bset, hp.addr, header=h0[:hb], payload_reader=lambda lo, n: h0[hb + lo: hb + lo + n],
                         pool_reader=lambda lo, n: rd.read(opool, lo, n), hb=hb, total=total, need=need)
    assert torch.equal(hosts[0], hosts[1])
    host = out.to_host()
    assert host["tensors"].tobytes() == bset.tensors.tobytes() and (host["dim"] == bset.dim).all() and (host["qn"] == bset.qn).all()
    st = q.stats()
    assert st["host_bytes_live"] == 2 * total and st["device_bytes"] < 2 * (2 * (256 << 20)) + (256 << 20)
    q.destroy()


# ---- the SURVEY §8(f) NEXT-4 variants at sizes that reach the launch shape large sets select for themselves -----------------
# (round 3; the align-8 movers, wire format v3 and the other element types had met their oracles only on sets of
# <= 77 MB, i.e. with the static deal of the tiles and the small ring shape).  DEFAULT opts on >= 1 GB: one ring of
# 3 x 48 KiB, tiles from the counter, table two iterations ahead, stream offsets beyond 2^32 for align 8.  The oracle
# serializes the whole set at once from a host copy of the seeded source pool; every stream byte and every byte of the
# deserialized pool image is compared.
def _variant_case(name):
    from oracle import dt, v3
    if name == "align8":          # config 3: 2.2 GB, 447 k blocks of ~5 KB, about half of them 8 off the 16-byte grid
        bset = W.make_config("3")
        return bset, bs.F64 | bs.ALIGN8, 8, False, lambda addr, blocks: oracle.serialize(bset.tensors, bset.qn, bset.dim, addr, align=8), \
            lambda s: (oracle.pool_bytes(s), oracle.deserialize(s)["pool"])
    if name == "rank4":           # order-4 tree nodes + operators: 1.4 GB, 3394 blocks (wire format v3)
        bset = W.make_tree_set("tree-1.4GB", 8, D=600, S=12, n_nodes=6, n_ops=13)
        return bset, bs.F64 | bs.RANK4, 8, True, lambda addr, blocks: v3.serialize(bset.tensors, bset.qn, bset.dim, addr), \
            lambda s: (v3.pool_bytes(s), v3.deserialize(s)["pool"])
    if name == "f32":             # config 4's sectors with 450 operators read as f32: 1.1 GB (the independent numpy oracle)
        bset = W.make_config("4", n_ops=450)
        def deser32(s):
            r = dt.deserialize(s)
            return r["pool_bytes"], np.asarray(r["pool"])
        return bset, bs.F32, 4, False, lambda addr, blocks: dt.serialize(bset.tensors, bset.qn, bset.dim, blocks(), dt.F32), deser32
    raise KeyError(name)


@pytest.mark.parametrize("name", ["align8", "rank4", "f32"])
def test_full_size_variants_with_default_opts(name):
    from oracle import dt
    from workloads.device import fill_pool_device
    bset, dtype, e, rank4, ser, deser = _variant_case(name)
    _room_for(name, bset)
    d_pool, d_addr = fill_pool_device(bset, DEV)
    hp = HostPool(bset, d_pool)                       # host copy of the seeded pool, spot-checked against the host generator
    blocks = lambda: [hp.pool[int(o): int(o) + e * int(k)] for o, k in zip(bset.pool_off, bset.nelems)]
    want = ser(hp.addr, blocks)
    total = len(want)
    assert total >= (1 << 30) and total - bs.header_bytes(bset.n_tensors, bset.n_blocks) >= (512 << 20), "must reach the large shape"
    dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, d_addr, DEV, dtype=dtype)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    cs = bs.current_stream()
    hb = bs.header_bytes_rank4(bset.n_tensors, bset.n_blocks) if rank4 else bs.header_bytes(bset.n_tensors, bset.n_blocks)
    assert bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs) == (hb, total)
    stream = torch.full((total + 4096,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.serialize(dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["total_bytes"] == total and res["dtype"] == dtype, res
    got = stream.cpu().numpy()
    assert (got[total:] == 0xCD).all(), "bytes beyond the stream were written"
    from tests.fullsize import equal_bytes, first_difference
    assert equal_bytes(got[:total], want), f"{name}: stream differs first at byte {first_difference(got[:total], want)} (header {hb})"
    del got
    need = int(((bset.nelems * e + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB, rank4=rank4)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need, res
    host = out.to_host()
    assert host["tensors"].tobytes() == bset.tensors.tobytes() and (host["qn"] == bset.qn).all() and (host["dim"] == bset.dim).all()
    gpool = opool.cpu().numpy()
    n_ref, ref = deser(want)
    assert n_ref == need
    ref = np.frombuffer(ref, np.uint8) if not isinstance(ref, np.ndarray) else ref
    assert equal_bytes(gpool, ref[:need]), f"{name}: pool image differs first at byte {first_difference(gpool, ref[:need])}"
