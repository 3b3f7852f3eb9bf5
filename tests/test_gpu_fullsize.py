"""Parity at BASELINE.json's full sizes (configs 3 and 4), in the launch configuration bench.py times (default opts).
The oracle cannot hold these streams in seconds, so it is run slice-wise: the whole header, and the payload of sampled
tensors whose values it regenerates from the counter-based generator (never a byte from the CUDA path).  Properties that
hold at any size cover the rest: exact size prediction, the fixpoint serialize(deserialize(S)) == S on the device, and
chunked offload == the stream."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
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


import os

# 3L / 4L (operator count scaled to BASELINE.json's stated totals, 11 GB / 43 GB streams) need
# ~3x their size in HBM and minutes of host-side generation: opt in with BS_TEST_LARGE=1
_CFGS = ["3", "4"] + (["3L", "4L"] if os.environ.get("BS_TEST_LARGE") == "1" else [])


@pytest.mark.parametrize("cfg", _CFGS)
def test_full_size_serialize_deserialize(cfg):
    bset = W.make_config(cfg)
    up = Uploaded(bset, fill="device")
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
    # the whole header against the oracle's
    want_h = oracle.emit_header(bset.tensors, bset.qn, bset.dim)
    got_h = stream[:hb].cpu().numpy()
    bad = np.nonzero(got_h != want_h)[0]
    assert bad.size == 0, f"header differs first at byte {bad[0]}"
    # sampled tensors' payload against the oracle's
    for t in sampled_tensors(bset):
        first, want, _ = oracle_tensor_payload(bset, t)
        got = stream[hb + first: hb + first + len(want)].cpu().numpy()
        bad = np.nonzero(got != want)[0]
        assert bad.size == 0, f"tensor {t}: payload differs first at payload byte {first + bad[0]}"

    # deserialize: descriptor identical, sampled blocks bit-identical to the regenerated values
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
    for t in sampled_tensors(bset, n=6, seed=9):
        b0 = int(bset.tensors["first_block"][t])
        b1 = b0 + int(bset.tensors["n_blocks"][t])
        pool, offs = W.fill_pool_host(bset, b0, b1, compact=True)
        for i in range(b0, b1):
            n = int(bset.nelems[i])
            o = int(host["addr"][i]) - opool.data_ptr()
            got = opool[o: o + 8 * n].cpu().numpy().view(np.uint64)
            want = pool.view(np.uint64)[int(offs[i - b0]) // 8: int(offs[i - b0]) // 8 + n]
            assert (got == want).all(), f"block {i} of tensor {t} differs after the round trip"
            # the rest of the align256 slot is untouched: unpack writes exactly nbytes per block, never the stream's pad
            gap = opool[o + 8 * n: o + int(slots[i])].cpu().numpy()
            assert (gap == 0xEE).all(), f"block {i}: bytes past the end of the block were written"
    # fixpoint on the device, every byte: serialize(deserialize(S)) == S
    del up.pool, got                      # 4L: source + stream + pool + second stream would not fit in 180 GB
    up.dset = None
    torch.cuda.empty_cache()
    again = torch.full((total,), 0x11, dtype=torch.uint8, device=DEV)
    bs.serialize(out.desc, again.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK
    assert torch.equal(again, stream[:total]), "serialize(deserialize(S)) != S"


def test_full_size_offload_prefetch_config3():
    """config 5's data path at full size: 256 MiB double-buffered chunks; concat(chunks) == the bs_serialize stream."""
    bset = W.make_config("3")
    up = Uploaded(bset, fill="device")
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, total, DEV)
    cs = bs.current_stream()
    stream = torch.empty(total, dtype=torch.uint8, device=DEV)
    bs.serialize(up.dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK
    host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
    host.fill_(0x5A)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total)        # defaults: 256 MiB chunks, 2 staging buffers
    st = eng.offload_async(up.dset.desc, total, host.data_ptr(), total, cs).wait()
    assert st["status"] == bs.OK and st["bytes"] == total and st["n_chunks"] == (total + (256 << 20) - 1) // (256 << 20)
    assert torch.equal(host, stream.cpu()), "concat(chunks) != stream"
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    st = eng.prefetch_async(host.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs).wait()
    torch.cuda.synchronize()
    assert st["status"] == bs.OK
    ref_out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    ref_pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.deserialize(stream.data_ptr(), total, ref_out.desc, ref_pool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                   ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK
    assert torch.equal(opool, ref_pool)
    a, b = out.to_host(), ref_out.to_host()
    assert a["tensors"].tobytes() == b["tensors"].tobytes() and (a["qn"] == b["qn"]).all() and (a["dim"] == b["dim"]).all()
    assert ((a["addr"] - np.uint64(opool.data_ptr())) == (b["addr"] - np.uint64(ref_pool.data_ptr()))).all()
    eng.destroy()


@pytest.mark.parametrize("cfg", ["3", "4"])
def test_full_size_layered_v2(cfg):
    """Wire format v2 (structure-shared layers) at full size, default launch configuration: the whole header against
    the v2 oracle's (its payload part is skipped by giving the oracle a capacity check only), the payload against the
    v1 stream of the same tensors (pinned relation: identical payload), size prediction, device fixpoint."""
    from oracle import v2
    bset = W.make_config(cfg)
    up = Uploaded(bset, fill="device")
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
    # payload: sampled tensors against the v1 oracle's slice-wise payload (same bytes, same payload offsets)
    for t in sampled_tensors(bset, n=6):
        first, want, _ = oracle_tensor_payload(bset, t)
        got = stream[hb + first: hb + first + len(want)].cpu().numpy()
        assert (got == want).all(), f"layer {t}: payload differs"
    # and, every byte, against the v1 CUDA stream's payload
    ws1 = bs.Workspace(bset.n_tensors, bset.n_blocks, total1, DEV)
    s1 = torch.empty(total1, dtype=torch.uint8, device=DEV)
    bs.serialize(up.dset.desc, s1.data_ptr(), total1, ws1.ptr, ws1.nbytes, ws1.result_ptr, None, cs)
    assert ws1.read_result()["status"] == bs.OK
    assert torch.equal(s1[hb1:], stream[hb:total])
    del s1, ws1
    # deserialize + fixpoint on the device
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
    again = torch.full((total,), 0x11, dtype=torch.uint8, device=DEV)
    bs.layered_serialize(out.desc, again.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, None, cs)
    assert ws.read_result()["status"] == bs.OK
    assert torch.equal(again, stream[:total]), "serialize(deserialize(S)) != S"


def check_blocks_against_generator(bset, host_desc, opool, tensors):
    """Sampled tensors' blocks in a BS_LAYOUT_POOL pool against values regenerated on the host (never the CUDA path's)."""
    for t in tensors:
        b0 = int(bset.tensors["first_block"][t])
        b1 = b0 + int(bset.tensors["n_blocks"][t])
        pool, offs = W.fill_pool_host(bset, b0, b1, compact=True)
        for i in range(b0, b1):
            n = int(bset.nelems[i])
            o = int(host_desc["addr"][i]) - opool.data_ptr()
            got = opool[o: o + 8 * n].cpu().numpy().view(np.uint64)
            want = pool.view(np.uint64)[int(offs[i - b0]) // 8: int(offs[i - b0]) // 8 + n]
            assert (got == want).all(), f"block {i} of tensor {t} differs"


def test_full_size_packages_config4():
    """NEXT-2 at full size in the configuration bench.py times: 4 MiB limit (1719 packages), shuffled slots, one launch."""
    import struct
    from oracle import pkg
    bset = W.make_config("4")
    up = Uploaded(bset, fill="device")
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

    def stream_range(lo, nbytes):
        """Stream bytes [lo, lo+nbytes) out of the slots, located with the ORACLE's cut."""
        parts = []
        nh = -(-hb // cap)
        while nbytes:
            k = lo // cap if lo < hb else nh + (lo - hb) // cap
            plo, phi = pkg.package_range(hb, total, cap, k)
            take = min(nbytes, phi - lo)
            base = int(slot_of[k]) * slot_bytes + 64 + (lo - plo)
            parts.append(slots[base: base + take].cpu().numpy())
            lo += take
            nbytes -= take
        return np.concatenate(parts)

    want_h = oracle.emit_header(bset.tensors, bset.qn, bset.dim)
    assert (stream_range(0, hb) == want_h).all(), "header region of the packages differs from the oracle's header"
    for t in sampled_tensors(bset, n=6):
        first, want, _ = oracle_tensor_payload(bset, t)
        assert (stream_range(hb + first, len(want)) == want).all(), f"tensor {t}: payload in the packages differs"
    # package headers: the oracle's cut; first_block by numpy.searchsorted over the oracle's offsets
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
    # and back: one-launch unpack from the shuffled slots
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
    opool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    bs.package_unpack(slots.data_ptr(), slot_bytes, n, sid, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                      ws.result_ptr, None, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need
    host = out.to_host()
    assert host["tensors"].tobytes() == bset.tensors.tobytes() and (host["qn"] == bset.qn).all() and (host["dim"] == bset.dim).all()
    check_blocks_against_generator(bset, host, opool, sampled_tensors(bset, n=5, seed=3))


def test_full_size_queue_config3():
    """NEXT-3 at full size: the bench's e2e pattern — save a set while the stream saved before it is loaded back."""
    bset = W.make_config("3")
    up = Uploaded(bset, fill="device")
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
    want_h = oracle.emit_header(bset.tensors, bset.qn, bset.dim)
    for h in hosts:
        assert (h[:hb].numpy() == want_h).all()
        for t in sampled_tensors(bset, n=4):
            first, want, _ = oracle_tensor_payload(bset, t)
            assert (h[hb + first: hb + first + len(want)].numpy() == want).all(), f"tensor {t}: saved payload differs"
    assert torch.equal(hosts[0], hosts[1])
    host = out.to_host()
    assert host["tensors"].tobytes() == bset.tensors.tobytes() and (host["dim"] == bset.dim).all()
    check_blocks_against_generator(bset, host, opool, sampled_tensors(bset, n=5, seed=3))
    st = q.stats()
    assert st["host_bytes_live"] == 2 * total and st["device_bytes"] < 2 * (2 * (256 << 20)) + (256 << 20)
    q.destroy()
