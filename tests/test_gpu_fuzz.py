"""Seeded random sets through the C ABI against the oracles: free-form descriptors (empty tensors, zero extents, ranks 2 and
3, every element type, 8- and 16-byte-aligned sources, sizes from bytes to megabytes) that the paper-shaped generator never
makes.  Everything is compared bit for bit; the launch shape, the chunking and the package limit are drawn too."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_04676_b200 as bs
import workloads as W
from oracle import dt, pkg
from tests.gpu_util import DEV

pytestmark = pytest.mark.gpu
EXTENTS = [0, 1, 1, 2, 3, 5, 8, 17, 64, 127, 300]


def random_set(rng):
    T = int(rng.integers(0, 7))
    tensors = np.zeros(T, W.TENSOR_REC_DTYPE)
    qn, dim = [], []
    for t in range(T):
        rank = int(rng.choice([2, 3]))
        nb = int(rng.integers(0, 9))
        tensors[t] = (rank, len(dim), nb, tuple(int(x) for x in rng.integers(-2, 3, 2)), (-1, 1, 0 if rank == 2 else -1, 0),
                      int(rng.integers(0, 1 << 31)), 0)
        for _ in range(nb):
            d = [int(rng.choice(EXTENTS)), int(rng.choice(EXTENTS)), int(rng.choice(EXTENTS)) if rank == 3 else 1]
            if rng.random() < 0.1:
                d[int(rng.integers(0, 2))] = int(rng.integers(500, 1500))       # now and then a block of megabytes
            q = rng.integers(-5, 6, (3, 2)).astype(np.int32)
            if rank == 2:
                q[2] = 0
            qn.append(q)
            dim.append(d)
    qn = np.array(qn, np.int32).reshape(-1, 3, 2)
    dim = np.array(dim, np.uint32).reshape(-1, 3)
    return tensors, qn, dim


def upload(rng, tensors, qn, dim, dtype):
    return upload_host(rng, tensors, qn, dim, dtype)[:3]


def upload_host(rng, tensors, qn, dim, dtype, flags=0):
    """As upload (same draws in the same order), any number of legs; also returns the host image and the block offsets in it.
    `flags` (bs.ALIGN8 / bs.RANK4) go into the device descriptor's dtype word."""
    e = dt.ELEM_BYTES[dtype]
    sizes = [e * int(np.prod([int(x) for x in d])) for d in dim]
    blocks = [rng.integers(0, 256, n, dtype=np.uint8).tobytes() for n in sizes]
    cur = 0
    order = list(rng.permutation(len(blocks))) if blocks else []
    offs = np.zeros(len(blocks), np.uint64)
    for i in order:
        mis = 8 if rng.random() < 0.3 else 0                                       # D16: 8-byte-aligned sources take the slow path
        offs[i] = cur + mis
        cur += (sizes[i] + mis + 255) // 256 * 256 + 256
    host = np.full(max(cur, 256), 0x33, np.uint8)
    for b, o in zip(blocks, offs):
        host[int(o): int(o) + len(b)] = np.frombuffer(b, np.uint8)
    pool = torch.from_numpy(host).to(DEV)
    addr = (np.uint64(pool.data_ptr()) + offs).astype(np.uint64)
    dset = bs.DeviceSet.from_host(tensors, qn, dim, addr, DEV, dtype=dtype | flags)
    return pool, dset, blocks, host, offs


def wide_opts(rng):
    """A random TMA launch shape the library accepts (bs.h bs_opts; check_opts in bs_api.cu)."""
    while True:
        tile = int(rng.integers(4, 65)) * 1024
        stages = int(rng.integers(3, 9))
        warps = int(rng.integers(1, 6))
        if warps * (stages * tile + 2048) <= 224 * 1024:
            break
    tune = int(rng.choice([0, 8, 0x10, 0x1000, 0x1010, 0x1008, 0x20, 0x30]))
    if rng.random() < 0.3:
        tune |= int(rng.integers(1, 4)) << 8            # fewer tiles loading beside the one being stored
    return dict(variant=bs.VARIANT_TMA, tile_bytes=tile, stages=stages, warps=warps, tune=tune, fuse=int(rng.integers(0, 3)),
                pace=int(rng.choice([0, 0, 300, 6500, 20000])))


@pytest.mark.parametrize("seed", range(24))
def test_random_sets_round_trip_bit_exact(seed):
    rng = np.random.default_rng(1000 + seed)
    tensors, qn, dim = random_set(rng)
    dtype = int(rng.integers(0, 4))
    pool, dset, blocks = upload(rng, tensors, qn, dim, dtype)
    want = dt.serialize(tensors, qn, dim, blocks, dtype)
    if dtype == dt.F64 and len(blocks):        # the C oracle is a second opinion where it applies
        hp = np.frombuffer(b"".join(b.ljust((len(b) + 15) // 16 * 16 + 16, b"\0") for b in blocks), np.uint8).copy()
        ho = np.concatenate([[0], np.cumsum([(len(b) + 15) // 16 * 16 + 16 for b in blocks])[:-1]]).astype(np.uint64)
        assert bytes(oracle.serialize(tensors, qn, dim, (np.uint64(hp.ctypes.data) + ho).astype(np.uint64))) == bytes(want)
    total = len(want)
    T, B = len(tensors), len(blocks)
    variant = int(rng.choice([bs.VARIANT_TMA, bs.VARIANT_LDG]))
    opts = dict(variant=variant, tile_bytes=int(rng.choice([16384, 32768])), stages=3, warps=int(rng.integers(1, 3)))
    ws = bs.Workspace(T, B, max(total, 1 << 16), DEV, packages=True)
    cs = bs.current_stream()
    assert bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs) == (dt.header_bytes(T, B), total)      # L106
    out = torch.full((total + 32,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.serialize(dset.desc, out.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)
    assert ws.read_result()["status"] == bs.OK
    got = out.cpu().numpy()
    assert (got[:total] == want).all() and (got[total:] == 0xCD).all(), f"seed {seed}: stream differs"
    # concat of ranges with a random chunk == the stream (D15)
    chunk = int(rng.integers(1, 40)) * 16 * int(rng.choice([1, 64, 4096]))
    rng_out = torch.full((total,), 0xCD, dtype=torch.uint8, device=DEV)
    for lo in range(0, total, chunk):
        bs.serialize_range(dset.desc, rng_out.data_ptr() + lo, lo, min(lo + chunk, total), lo == 0, ws.ptr, ws.nbytes, ws.result_ptr,
                           opts, cs)
    assert (rng_out.cpu().numpy() == want).all(), f"seed {seed}: concat of ranges differs (chunk {chunk})"
    # deserialize
    ref = dt.deserialize(want)
    need = ref["pool_bytes"]
    o = bs.DeviceSet.empty(T, B, DEV, fill=0xAB)
    opool = torch.full((max(need, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    bs.deserialize(out.data_ptr(), total, o.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need and res["dtype"] == dtype and (res["n_tensors"], res["n_blocks"]) == (T, B)
    assert (opool.cpu().numpy()[:need] == ref["pool"][:need]).all(), f"seed {seed}: blocks differ"
    h = o.to_host()
    assert h["tensors"].tobytes() == tensors.tobytes() and (h["qn"] == qn).all() and (h["dim"] == dim).all()
    # packages at a random limit, shuffled slots, and back
    cap = int(rng.choice([16, 4096, 16384, 32768, 49152 + 16]))
    if cap == 16 and total > 65536:
        cap = 4096                              # keep the number of packages (two launches each) bounded
    n = pkg.count(dt.header_bytes(T, B), total, cap)
    slot_of = rng.permutation(n + 1)[:n]
    slots = torch.full(((n + 1) * (64 + cap),), 0x5A, dtype=torch.uint8, device=DEV)
    bs.package_emit(dset.desc, total, cap, 77, slots.data_ptr(), 64 + cap, n + 1, slot_of, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)
    assert ws.read_result()["status"] == bs.OK
    ref_slots = pkg.emit_slots(want, cap, 77, 64 + cap, slot_of=slot_of, n_slots=n + 1, poison=0x5A)
    assert (slots.cpu().numpy().reshape(n + 1, -1) == ref_slots).all(), f"seed {seed}: packages differ (limit {cap})"
    opool.fill_(0xEE)
    bs.package_unpack(slots.data_ptr(), 64 + cap, n + 1, 77, o.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                      ws.result_ptr, opts, cs)
    assert ws.read_result()["status"] == bs.OK
    assert (opool.cpu().numpy()[:need] == ref["pool"][:need]).all(), f"seed {seed}: blocks differ after the package round trip"
    # the same set through launch shapes of the whole space round 2 opened: tiles of any multiple of 1 KiB, 3-8 stages, the
    # tile counter forced or forbidden, the table fetched further ahead, a pace, one launch or two (own generator: the
    # draws above stay what they were)
    rng_o = np.random.default_rng(7000 + seed)
    for _ in range(3):
        wide = wide_opts(rng_o)
        out.fill_(0xCD)
        bs.serialize(dset.desc, out.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, wide, cs)
        assert ws.read_result()["status"] == bs.OK, wide
        got = out.cpu().numpy()
        assert (got[:total] == want).all() and (got[total:] == 0xCD).all(), f"seed {seed}: stream differs with {wide}"
        chunk = int(rng_o.integers(1, 40)) * 16 * int(rng_o.choice([64, 4096]))
        rng_out.fill_(0xCD)
        for lo in range(0, total, chunk):
            bs.serialize_range(dset.desc, rng_out.data_ptr() + lo, lo, min(lo + chunk, total), lo == 0, ws.ptr, ws.nbytes,
                               ws.result_ptr, wide, cs)
        assert (rng_out.cpu().numpy() == want).all(), f"seed {seed}: concat of ranges differs (chunk {chunk}) with {wide}"
        opool.fill_(0xEE)
        bs.deserialize(out.data_ptr(), total, o.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr, wide, cs)
        assert ws.read_result()["status"] == bs.OK, wide
        assert (opool.cpu().numpy()[:need] == ref["pool"][:need]).all(), f"seed {seed}: blocks differ with {wide}"


def random_set4(rng):
    """Free-form set of ranks 2, 3 and 4 with four legs per block (BS_RANK4; unused legs: extent 1, labels 0)."""
    T = int(rng.integers(0, 7))
    tensors = np.zeros(T, W.TENSOR_REC_DTYPE)
    qn, dim = [], []
    for t in range(T):
        rank = int(rng.choice([2, 3, 4]))
        nb = int(rng.integers(0, 9))
        sign = (1, 1, 1, -1) if rank == 4 else ((-1, 1, -1, 0) if rank == 3 else (-1, 1, 0, 0))
        tensors[t] = (rank, len(dim), nb, tuple(int(x) for x in rng.integers(-2, 3, 2)), sign, int(rng.integers(0, 1 << 31)), 0)
        for _ in range(nb):
            d = [int(rng.choice(EXTENTS)) if k < rank else 1 for k in range(4)]
            if rank == 4:
                d[2] = int(rng.choice(EXTENTS[:6]))                              # keep order-4 blocks below a few MB
                d[3] = int(rng.choice(EXTENTS[:9]))
            if rng.random() < 0.1:
                d[int(rng.integers(0, 2))] = int(rng.integers(500, 1500)) if rank < 4 else 40
            q = rng.integers(-5, 6, (4, 2)).astype(np.int32)
            q[rank:] = 0
            qn.append(q)
            dim.append(d)
    return tensors, np.array(qn, np.int32).reshape(-1, 4, 2), np.array(dim, np.uint32).reshape(-1, 4)


@pytest.mark.parametrize("seed", range(16))
def test_random_unpadded_and_rank4_sets_through_random_launch_shapes(seed):
    """BS_ALIGN8 (even seeds) and BS_RANK4 (odd seeds) sets through the default shape and three drawn from the whole space
    (wide_opts: tile counter forced or forbidden, table further ahead, one launch or two, tiles of any multiple of 1 KiB) —
    the variants' own movers had only met fixed shapes.  Stream, concat of ranges, round trip: bit for bit."""
    from oracle import v3
    rng = np.random.default_rng(9000 + seed)
    rank4 = bool(seed & 1)
    dtype = int(rng.integers(0, 4))
    if rank4:
        tensors, qn, dim = random_set4(rng)
        pool, dset, blocks, host, offs = upload_host(rng, tensors, qn, dim, dtype, bs.RANK4)
        want = v3.serialize(tensors, qn, dim, (np.uint64(host.ctypes.data) + offs).astype(np.uint64), dtype=dtype)
        ref_pool, need = v3.deserialize(want)["pool"], v3.pool_bytes(want)
        hb = v3.header_bytes(len(tensors), len(blocks))
    else:
        tensors, qn, dim = random_set(rng)
        pool, dset, blocks, host, offs = upload_host(rng, tensors, qn, dim, dtype, bs.ALIGN8)
        want = dt.serialize(tensors, qn, dim, blocks, dtype, align=8)
        ref = dt.deserialize(want)
        ref_pool, need = ref["pool"], ref["pool_bytes"]
        hb = dt.header_bytes(len(tensors), len(blocks))
        if dtype == dt.F64 and len(blocks):    # the C oracle as a second opinion
            assert bytes(oracle.serialize(tensors, qn, dim, (np.uint64(host.ctypes.data) + offs).astype(np.uint64), align=8)) == bytes(want)
    total, T, B = len(want), len(tensors), len(blocks)
    ws = bs.Workspace(T, B, max(total, 1 << 16), DEV)
    cs = bs.current_stream()
    assert bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs) == (hb, total)
    out = torch.full((total + 32,), 0xCD, dtype=torch.uint8, device=DEV)
    rng_out = torch.full((total + 32,), 0xCD, dtype=torch.uint8, device=DEV)
    o = bs.DeviceSet.empty(T, B, DEV, fill=0xAB, rank4=rank4)
    opool = torch.full((max(need, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    for shape in [None] + [wide_opts(rng) for _ in range(3)]:
        out.fill_(0xCD)
        bs.serialize(dset.desc, out.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, shape, cs)
        res = ws.read_result()
        assert res["status"] == bs.OK and res["total_bytes"] == total, (shape, res)
        got = out.cpu().numpy()
        assert (got[:total] == want).all() and (got[total:] == 0xCD).all(), f"seed {seed}: stream differs with {shape}"
        chunk = int(rng.integers(1, 40)) * 16 * int(rng.choice([64, 4096]))
        rng_out.fill_(0xCD)
        for lo in range(0, total, chunk):      # hi is a multiple of 16 and clipped to the total (a multiple of 8 when unpadded)
            bs.serialize_range(dset.desc, rng_out.data_ptr() + lo, lo, lo + chunk, lo == 0, ws.ptr, ws.nbytes, ws.result_ptr, shape, cs)
        got = rng_out.cpu().numpy()
        assert (got[:total] == want).all() and (got[total:] == 0xCD).all(), f"seed {seed}: concat of ranges differs (chunk {chunk}) with {shape}"
        opool.fill_(0xEE)
        bs.deserialize(out.data_ptr(), total, o.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr, shape, cs)
        res = ws.read_result()
        assert res["status"] == bs.OK and res["pool_bytes"] == need and (res["n_tensors"], res["n_blocks"]) == (T, B), (shape, res)
        assert (opool.cpu().numpy()[:need] == ref_pool[:need]).all(), f"seed {seed}: blocks differ with {shape}"
        h = o.to_host()
        assert h["tensors"].tobytes() == tensors.tobytes() and (h["qn"] == qn).all() and (h["dim"] == dim).all()


def random_layered(rng):
    """Free-form layered set: C structures (some empty, some unused), T layers naming them in any order."""
    C = int(rng.integers(1, 6))
    structs = np.zeros(C, W.STRUCT_REC_DTYPE)
    qn, dim = [], []
    for c in range(C):
        rank = int(rng.choice([2, 3]))
        nb = int(rng.integers(0, 7))
        structs[c] = (rank, len(dim), nb, tuple(int(x) for x in rng.integers(-2, 3, 2)), (-1, 1, 0 if rank == 2 else -1, 0), 0)
        for _ in range(nb):
            d = [int(rng.choice(EXTENTS)), int(rng.choice(EXTENTS)), int(rng.choice(EXTENTS[:8])) if rank == 3 else 1]
            q = rng.integers(-5, 6, (3, 2)).astype(np.int32)
            if rank == 2:
                q[2] = 0
            qn.append(q)
            dim.append(d)
    T = int(rng.integers(0, 12))
    layers = np.zeros(T, W.LAYER_REC_DTYPE)
    for t in range(T):
        layers[t] = (int(rng.integers(0, C)), int(rng.integers(0, 1 << 31)), 0)
    return structs, layers, np.array(qn, np.int32).reshape(-1, 3, 2), np.array(dim, np.uint32).reshape(-1, 3)


@pytest.mark.parametrize("seed", range(16))
def test_random_layered_sets_round_trip_bit_exact(seed):
    from oracle import v2
    rng = np.random.default_rng(5000 + seed)
    structs, layers, qn, dim = random_layered(rng)
    sizes = []                                   # blocks layer by layer, in the order of the layer's structure
    for ly in layers:
        s = structs[int(ly["structure"])]
        for j in range(int(s["first_block"]), int(s["first_block"]) + int(s["n_blocks"])):
            sizes.append(8 * int(dim[j, 0]) * int(dim[j, 1]) * int(dim[j, 2]))
    B = len(sizes)
    offs = np.zeros(B, np.uint64)
    cur = 0
    for i in (rng.permutation(B) if B else []):
        mis = 8 if rng.random() < 0.3 else 0
        offs[i] = cur + mis
        cur += (sizes[i] + mis + 255) // 256 * 256 + 256
    host = rng.integers(0, 256, max(cur, 256), dtype=np.uint8)
    want = v2.serialize(structs, layers, qn, dim, (np.uint64(host.ctypes.data) + offs).astype(np.uint64))
    pool = torch.from_numpy(host).to(DEV)
    addr = (np.uint64(pool.data_ptr()) + offs).astype(np.uint64)
    dset = bs.DeviceLayeredSet.from_host(structs, layers, qn, dim, addr, DEV)
    counts = (len(structs), dim.shape[0], len(layers), B)
    total = len(want)
    opts = dict(variant=int(rng.choice([bs.VARIANT_TMA, bs.VARIANT_LDG])), tile_bytes=int(rng.choice([16384, 32768])), stages=3,
                warps=int(rng.integers(1, 3)))
    ws = bs.Workspace(0, 0, max(total, 1 << 16), DEV, layered=counts)
    cs = bs.current_stream()
    assert bs.layered_serialized_size(dset.desc, ws.ptr, ws.nbytes, cs) == v2.serialized_size(structs, layers, dim)
    out = torch.full((total + 32,), 0xCD, dtype=torch.uint8, device=DEV)
    bs.layered_serialize(dset.desc, out.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)
    assert ws.read_result()["status"] == bs.OK
    got = out.cpu().numpy()
    assert (got[:total] == want).all() and (got[total:] == 0xCD).all(), f"seed {seed}: v2 stream differs"
    ref = v2.deserialize(want)
    na, need = v2.counts(want)
    assert na == B
    o = bs.DeviceLayeredSet.empty(*counts, DEV, fill=0xAB)
    opool = torch.full((max(need, 256),), 0xEE, dtype=torch.uint8, device=DEV)
    bs.layered_deserialize(out.data_ptr(), total, o.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr,
                           opts, cs)
    res = ws.read_result()
    assert res["status"] == bs.OK and res["pool_bytes"] == need
    assert (opool.cpu().numpy()[:need] == ref["pool"][:need]).all(), f"seed {seed}: blocks differ"
    h = o.to_host(*counts)
    assert h["structs"].tobytes() == ref["structs"].tobytes() and h["layers"].tobytes() == ref["layers"].tobytes()
    assert (h["qn"] == qn).all() and (h["dim"] == dim).all()
