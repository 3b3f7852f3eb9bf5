"""NEXT-3 on the GPU: the save / load queue with checkpoints through the C ABI against the sequential
definition oracle.QueueModel — whatever overlaps in time on the device, a caller sees per-key program order."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from tests.gpu_util import DEV, Uploaded
from tests.util import host_addrs, oracle_stream

pytestmark = pytest.mark.gpu


def pinned(n, fill=0xCD):
    t = torch.empty(max(n, 16), dtype=torch.uint8, pin_memory=True)
    t.fill_(fill)
    return t


class Loaded:
    def __init__(self, bset, need):
        self.out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, DEV, fill=0xAB)
        self.pool = torch.full((max(need, 256),), 0xEE, dtype=torch.uint8, device=DEV)
        self.need = need


def test_save_two_keys_and_load_them_back_while_saving_a_third():
    sets = [W.make_config("2", n_ops=26 + 13 * i) for i in range(3)]
    ups = [Uploaded(b) for b in sets]
    model = oracle.QueueModel()
    want = [model.save(k, b.tensors, b.qn, b.dim, host_addrs(u.host_pool, u.host_offs)) for k, (b, u) in enumerate(zip(sets, ups))]
    cap = max(len(w) for w in want)
    q = bs.Queue(max(b.n_tensors for b in sets), max(b.n_blocks for b in sets), cap, chunk_bytes=4 * 65536, n_staging=2)
    hosts = [pinned(len(w) + 256) for w in want]
    cs = bs.current_stream()
    q.save(0, ups[0].dset.desc, len(want[0]), hosts[0].data_ptr(), hosts[0].numel(), cs)
    q.save(1, ups[1].dset.desc, len(want[1]), hosts[1].data_ptr(), hosts[1].numel(), cs)
    # loads are submitted at once, behind the saves they depend on; the save of key 2 runs in the other lane meanwhile
    ld = [Loaded(sets[k], oracle.pool_bytes(want[k])) for k in range(2)]
    q.load(0, ld[0].out.desc, ld[0].pool.data_ptr(), ld[0].need, bs.LAYOUT_POOL, cs)
    q.save(2, ups[2].dset.desc, 0, hosts[2].data_ptr(), hosts[2].numel(), cs)      # size 0: predicted by the call
    q.load(1, ld[1].out.desc, ld[1].pool.data_ptr(), ld[1].need, bs.LAYOUT_POOL, cs)
    snap = [l.pool.clone() for l in ld]     # enqueued on the consumer stream: sees the data (checkpoint, no host wait)
    for k in range(3):
        st = q.wait(k)
        assert st["status"] == bs.OK, st
        assert st["save"]["bytes"] == len(want[k])
        assert (hosts[k].numpy()[:len(want[k])] == want[k]).all(), f"stream of key {k} differs from the oracle's"
        assert (hosts[k].numpy()[len(want[k]):] == 0xCD).all()
    for k in range(2):
        ref = model.load(k)
        assert (snap[k].cpu().numpy()[:ld[k].need] == ref["pool"][:ld[k].need]).all()
        h = ld[k].out.to_host()
        assert h["tensors"].tobytes() == sets[k].tensors.tobytes() and (h["qn"] == sets[k].qn).all() and (h["dim"] == sets[k].dim).all()
    got, ref = q.stats(), model.stats()
    for f in ("saves", "loads", "bytes_saved", "bytes_loaded", "host_bytes_live", "host_bytes_peak", "keys_live"):
        assert got[f] == ref[f], (f, got, ref)
    assert got["in_flight"] == 0 and got["max_in_flight"] >= 1      # how many overlap is timing, not semantics
    assert got["device_bytes"] < 2 * (2 * 4 * 65536) + (8 << 20)     # 2 lanes x 2 staging chunks + O(B): fixed, small
    q.destroy()


def test_a_seeded_sequence_of_saves_overwrites_loads_and_forgets_matches_the_model():
    rng = np.random.default_rng(17)
    model = oracle.QueueModel()
    q = bs.Queue(64, 4096, 4 << 20, chunk_bytes=65536, n_staging=2)
    cs = bs.current_stream()
    hosts = {k: pinned(4 << 20) for k in range(4)}
    keep = []          # device sets must stay alive until their save completed
    pending = []       # (Loaded, reference pool, bset)
    cur = {}           # the set each live key holds
    for step in range(48):
        key = int(rng.integers(0, 4))
        r = rng.random()
        if r < 0.5 or key not in model.store:
            bset = W.make_set(f"q{step}", 300 + step, D=int(rng.integers(40, 160)), S=9, M=2, N0=3,
                              n_ops=int(rng.integers(1, 14)), n_site=int(rng.integers(0, 2)), dims="multinomial")
            up = Uploaded(bset)
            keep.append(up)
            s = model.save(key, bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs))
            q.save(key, up.dset.desc, len(s) if step % 3 else 0, hosts[key].data_ptr(), hosts[key].numel(), cs)
            cur[key] = bset
        elif r < 0.9:
            ref = model.load(key)
            bset = cur[key]
            ld = Loaded(bset, oracle.pool_bytes(model.store[key]))
            q.load(key, ld.out.desc, ld.pool.data_ptr(), ld.need, bs.LAYOUT_POOL, cs)
            pending.append((ld, ref, bset))
        else:
            model.forget(key)
            q.forget(key)
            with pytest.raises(bs.BsError) as e:
                q.load(key, keep[-1].dset.desc, 256, 0, bs.LAYOUT_POOL, cs)
            assert e.value.code == bs.ERR_ARG
    q.drain()
    for ld, ref, bset in pending:     # every load saw the LAST save of its key that preceded it in program order
        assert (ld.pool.cpu().numpy()[:ld.need] == ref["pool"][:ld.need]).all()
        h = ld.out.to_host()
        assert h["tensors"].tobytes() == bset.tensors.tobytes() and (h["dim"] == bset.dim).all()
    for key, s in model.store.items():
        assert q.wait(key)["status"] == bs.OK
        assert (hosts[key].numpy()[:len(s)] == s).all()
    got, ref = q.stats(), model.stats()
    for f in ("saves", "loads", "bytes_saved", "bytes_loaded", "host_bytes_live", "host_bytes_peak", "keys_live"):
        assert got[f] == ref[f], (f, got, ref)
    q.destroy()


def test_checkpoint_lets_the_producer_overwrite_its_blocks_without_a_host_wait():
    bset = W.make_config("2", n_ops=39)
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    q = bs.Queue(bset.n_tensors, bset.n_blocks, len(want), chunk_bytes=65536, n_staging=2)
    host = pinned(len(want))
    cs = bs.current_stream()
    q.save(5, up.dset.desc, len(want), host.data_ptr(), host.numel(), cs)
    q.checkpoint(5, cs)
    up.pool.fill_(0x77)            # on the producer stream, behind the checkpoint: must not leak into the saved stream
    assert q.wait(5)["status"] == bs.OK
    assert (host.numpy()[:len(want)] == want).all()
    with pytest.raises(bs.BsError):
        q.checkpoint(6, cs)
    q.destroy()


def test_adopted_streams_deferred_errors_and_overwrite_behind_a_running_load():
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    up = Uploaded(bset)
    want, _, _ = oracle_stream(bset, up.host_pool, up.host_offs)
    model = oracle.QueueModel()
    q = bs.Queue(bset.n_tensors, bset.n_blocks, len(want) + 64, chunk_bytes=65536)
    cs = bs.current_stream()
    good = pinned(len(want))
    good.numpy()[:] = want
    model.adopt(1, want)
    q.adopt(1, good.data_ptr(), len(want))
    ld = Loaded(bset, oracle.pool_bytes(want))
    q.load(1, ld.out.desc, ld.pool.data_ptr(), ld.need, bs.LAYOUT_POOL, cs)
    # overwrite key 1 while its load may still be running: the save waits for the load (the host buffer is being read)
    bset2 = W.make_set("fault2", 43, D=40, S=9, M=2, N0=3, n_ops=11, n_site=1, dims="multinomial")
    up2 = Uploaded(bset2)
    s2 = model.save(1, bset2.tensors, bset2.qn, bset2.dim, host_addrs(up2.host_pool, up2.host_offs))
    assert len(s2) <= good.numel()
    first = oracle.deserialize(want)
    q.save(1, up2.dset.desc, len(s2), good.data_ptr(), good.numel(), cs)
    assert q.wait(1)["status"] == bs.OK
    assert (ld.pool.cpu().numpy()[:ld.need] == first["pool"][:ld.need]).all()      # the load saw the FIRST stream
    assert (good.numpy()[:len(s2)] == s2).all()                                     # the buffer holds the SECOND now
    # a corrupt adopted stream: deferred BS_ERR_CORRUPT, nothing written
    bad = pinned(len(want))
    bad.numpy()[:] = want
    bad.numpy()[64 + 32 * bset.n_tensors + 48 * 3 + 40] ^= 0x10
    q.adopt(2, bad.data_ptr(), len(want))
    ld2 = Loaded(bset, oracle.pool_bytes(want))
    q.load(2, ld2.out.desc, ld2.pool.data_ptr(), ld2.need, bs.LAYOUT_POOL, cs)
    assert q.wait(2)["status"] == bs.ERR_CORRUPT
    assert (ld2.pool.cpu().numpy() == 0xEE).all()
    # a save whose size prediction is wrong: deferred BS_ERR_ARG; a load behind it is refused on the device
    h3 = pinned(len(want) + 64)
    q.save(3, up.dset.desc, len(want) + 16, h3.data_ptr(), h3.numel(), cs)
    ld3 = Loaded(bset, oracle.pool_bytes(want))
    q.load(3, ld3.out.desc, ld3.pool.data_ptr(), ld3.need, bs.LAYOUT_POOL, cs)
    st = q.wait(3)
    assert st["status"] == bs.ERR_ARG and st["load"]["status"] == bs.ERR_CORRUPT
    assert (ld3.pool.cpu().numpy() == 0xEE).all()
    q.destroy()


def test_layered_sets_and_other_element_types_go_through_the_queue():
    from oracle import dt, v2
    from tests.test_gpu_dtype import RawSet
    from tests.test_gpu_layered import LayeredUp
    bset = W.make_config("2", n_ops=39)
    lu = LayeredUp(bset)
    model = oracle.QueueModel()
    lv = lu.lv if hasattr(lu, "lv") else W.layered_view(bset)
    want = model.save_layered(1, lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(lu.up.host_pool, lu.up.host_offs))
    assert bytes(want) == bytes(lu.want)
    c = lu.counts
    rs = RawSet(W.make_set("dtq", 81, D=120, S=11, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial"), dt.F32, seed=4)
    q = bs.Queue(max(c[0], c[2], rs.bset.n_tensors), max(c[1], c[3], rs.bset.n_blocks), max(len(want), len(rs.want)),
                 chunk_bytes=2 * 65536)
    cs = bs.current_stream()
    h1, h2 = pinned(len(want)), pinned(len(rs.want))
    q.save_layered(1, lu.dset.desc, 0, h1.data_ptr(), h1.numel(), cs)             # size predicted by the call
    q.save(2, rs.dset.desc, len(rs.want), h2.data_ptr(), h2.numel(), cs)
    na, need = v2.counts(want)
    out = bs.DeviceLayeredSet.empty(*c, DEV, fill=0xAB)
    pool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    q.load_layered(1, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)        # behind its save: counts remembered by the queue
    ref32 = dt.deserialize(rs.want)
    out2 = bs.DeviceSet.empty(rs.bset.n_tensors, rs.bset.n_blocks, DEV, fill=0xAB)
    pool2 = torch.full((ref32["pool_bytes"],), 0xEE, dtype=torch.uint8, device=DEV)
    q.load(2, out2.desc, pool2.data_ptr(), ref32["pool_bytes"], bs.LAYOUT_POOL, cs)
    assert q.wait(1)["status"] == bs.OK and q.wait(2)["status"] == bs.OK
    torch.cuda.synchronize()
    assert (h1.numpy() == want).all() and (h2.numpy() == rs.want).all()
    ref = model.load_layered(1)
    assert (pool.cpu().numpy() == ref["pool"][:need]).all()
    h = out.to_host(*c)
    assert h["structs"].tobytes() == ref["structs"].tobytes() and h["layers"].tobytes() == ref["layers"].tobytes()
    assert (pool2.cpu().numpy() == ref32["pool"][:ref32["pool_bytes"]]).all()
    # a key holds a stream of one format
    with pytest.raises(oracle.OracleError):
        model.load(1)
    with pytest.raises(bs.BsError) as e:
        q.load(1, out2.desc, pool2.data_ptr(), ref32["pool_bytes"], bs.LAYOUT_POOL, cs)
    assert e.value.code == bs.ERR_ARG
    with pytest.raises(bs.BsError) as e:
        q.load_layered(2, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)
    assert e.value.code == bs.ERR_ARG
    # an adopted v2 stream is recognised by its version word
    q.adopt(5, h1.data_ptr(), len(want))
    pool.fill_(0xEE)
    q.load_layered(5, out.desc, pool.data_ptr(), need, bs.LAYOUT_POOL, cs)
    assert q.wait(5)["status"] == bs.OK
    torch.cuda.synchronize()
    assert (pool.cpu().numpy() == ref["pool"][:need]).all()
    q.destroy()


def test_storage_tier_spill_forget_fill_load(tmp_path):
    """PAPER L85 / L90: the stream goes on to a file behind the save (one host IO thread), the host buffer is given back,
    and the block comes back file -> pinned host -> device, bit-exact against the oracle's model."""
    bset = W.make_config("2", n_ops=52)
    up = Uploaded(bset)
    model = oracle.QueueModel()
    want = model.save(1, bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs))
    total = len(want)
    q = bs.Queue(bset.n_tensors, bset.n_blocks, total, chunk_bytes=4 * 65536)
    cs = bs.current_stream()
    h1 = pinned(total)
    path = str(tmp_path / "block1.bs")
    ref_path = str(tmp_path / "ref.bs")
    q.save(1, up.dset.desc, total, h1.data_ptr(), total, cs)
    q.spill(1, path)                                   # submitted at once: the IO thread waits for the save itself
    io = q.io_wait(1)
    assert io["status"] == bs.OK and io["bytes"] == total
    model.spill(1, ref_path)
    assert open(path, "rb").read() == open(ref_path, "rb").read() == want.tobytes()
    q.forget(1)
    model.forget(1)
    h1.fill_(0)                                        # the host buffer is the caller's again
    h2 = pinned(total + 4096)
    q.fill(9, path, h2.data_ptr(), h2.numel())
    model.fill(9, ref_path)
    ld = Loaded(bset, oracle.pool_bytes(want))
    q.load(9, ld.out.desc, ld.pool.data_ptr(), ld.need, bs.LAYOUT_POOL, cs)   # blocks the host until the file is in
    assert q.wait(9)["status"] == bs.OK
    torch.cuda.synchronize()
    ref = model.load(9)
    assert (ld.pool.cpu().numpy()[:ld.need] == ref["pool"][:ld.need]).all()
    assert (h2.numpy()[:total] == want).all() and (h2.numpy()[total:] == 0xCD).all()
    st = q.stats()
    assert st["bytes_spilled"] == total == model.bytes_spilled and st["bytes_filled"] == total == model.bytes_filled
    assert st["host_bytes_live"] == model.stats()["host_bytes_live"] == total
    # errors: a missing file, a file larger than the buffer, a truncated file (the device refuses the stream)
    with pytest.raises(bs.BsError) as e:
        q.fill(3, str(tmp_path / "missing.bs"), h1.data_ptr(), h1.numel())
    assert e.value.code == bs.ERR_IO
    with pytest.raises(bs.BsError) as e:
        q.fill(3, path, h1.data_ptr(), total - 16)
    assert e.value.code == bs.ERR_CAPACITY
    short = str(tmp_path / "short.bs")
    open(short, "wb").write(want.tobytes()[: total - 4096])
    q.fill(3, short, h1.data_ptr(), h1.numel())
    ld3 = Loaded(bset, oracle.pool_bytes(want))
    with pytest.raises(bs.BsError) as e:          # the header says more bytes than the file holds: refused at once
        q.load(3, ld3.out.desc, ld3.pool.data_ptr(), ld3.need, bs.LAYOUT_POOL, cs)
    assert e.value.code == bs.ERR_CORRUPT and (ld3.pool.cpu().numpy() == 0xEE).all()
    q.spill(9, str(tmp_path / "no_such_dir" / "x.bs"))
    assert q.io_wait(9)["status"] == bs.ERR_IO
    q.destroy()


def test_a_save_over_a_filled_key_forgets_the_fill(tmp_path):
    """Per-key program order across the storage tier: fill -> save -> load returns the SAVED object, also when the fill
    failed or held the other wire format; and a spill behind a failed save fails instead of writing stale bytes."""
    bset = W.make_config("2", n_ops=26)
    up = Uploaded(bset)
    model = oracle.QueueModel()
    want = model.save(1, bset.tensors, bset.qn, bset.dim, host_addrs(up.host_pool, up.host_offs))
    total = len(want)
    q = bs.Queue(bset.n_tensors, bset.n_blocks, total + 4096, chunk_bytes=4 * 65536)
    cs = bs.current_stream()
    ref = model.load(1)
    need = oracle.pool_bytes(want)
    # (1) a fill that fails (truncated to less than a header's worth of payload ... the read itself fails: a directory)
    h = pinned(total + 4096)
    bad_path = str(tmp_path / "short.bs")
    open(bad_path, "wb").write(want.tobytes()[:4096])
    q.fill(7, bad_path, h.data_ptr(), h.numel())
    ld = Loaded(bset, need)
    with pytest.raises(bs.BsError):                       # 4096 bytes of a longer stream: refused
        q.load(7, ld.out.desc, ld.pool.data_ptr(), ld.need, bs.LAYOUT_POOL, cs)
    q.save(7, up.dset.desc, total, h.data_ptr(), h.numel(), cs)    # the key is saved over: the fill no longer counts
    q.load(7, ld.out.desc, ld.pool.data_ptr(), ld.need, bs.LAYOUT_POOL, cs)
    assert q.wait(7)["status"] == bs.OK
    torch.cuda.synchronize()
    assert (h.numpy()[:total] == want).all()
    assert (ld.pool.cpu().numpy()[:need] == ref["pool"][:need]).all()
    # (2) fill (v1 file) -> save_layered -> load_layered: the key holds the layered stream now
    from oracle import v2
    lv = W.layered_view(bset)
    counts = (len(lv["structs"]), lv["dim"].shape[0], bset.n_tensors, bset.n_blocks)
    lset = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], up.addr, DEV)
    want2 = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(up.host_pool, up.host_offs))
    ql = bs.Queue(max(bset.n_tensors, counts[0]), bset.n_blocks, total + 4096, chunk_bytes=4 * 65536)
    good_path = str(tmp_path / "v1.bs")
    open(good_path, "wb").write(want.tobytes())
    h2 = pinned(total + 4096)
    ql.fill(3, good_path, h2.data_ptr(), h2.numel())
    ql.save_layered(3, lset.desc, len(want2), h2.data_ptr(), h2.numel(), cs)
    lout = bs.DeviceLayeredSet.empty(*counts, DEV, fill=0xAB)
    lpool = torch.full((need,), 0xEE, dtype=torch.uint8, device=DEV)
    ql.load_layered(3, lout.desc, lpool.data_ptr(), need, bs.LAYOUT_POOL, cs)
    assert ql.wait(3)["status"] == bs.OK
    torch.cuda.synchronize()
    assert (h2.numpy()[:len(want2)] == want2).all()
    assert (lpool.cpu().numpy()[:need] == ref["pool"][:need]).all()
    ql.destroy()
    # (3) a save that fails on the device (wrong size prediction): its spill must fail too, and write no file contents
    h3 = pinned(total + 4096)
    q.save(8, up.dset.desc, total, h3.data_ptr(), h3.numel(), cs)          # a good stream first, so the staging buffers hold one
    assert q.wait(8)["status"] == bs.OK
    q.save(8, up.dset.desc, total + 16, h3.data_ptr(), h3.numel(), cs)
    out_path = str(tmp_path / "failed.bs")
    q.spill(8, out_path)
    assert q.io_wait(8)["status"] == bs.ERR_ARG
    assert q.wait(8)["status"] == bs.ERR_ARG
    import os
    assert not os.path.exists(out_path) or os.path.getsize(out_path) == 0
    q.destroy()
