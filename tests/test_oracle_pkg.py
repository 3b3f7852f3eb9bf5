"""Pins of the package oracle (oracle/bs_oracle_pkg.c — self-contained packages):
hand-typed golden headers, a numpy restatement of the cut, numpy.searchsorted for first_block over offsets read by the
independent struct reader, the paper's property (any order of arrival reassembles the stream), fault injection."""
import os
import struct

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import pkg
from tests.streamreader import read_stream
from tests.util import oracle_stream, read_hex_fixture

HERE = os.path.dirname(__file__)
SID = 0x1122334455667788


def read_pkg_header(b):
    magic, version, index, count, first_block, sid, total, lo, nbytes, intra = struct.unpack_from("<8sIIIIQQQQQ", bytes(b), 0)
    return dict(magic=magic, version=version, index=index, count=count, first_block=first_block, stream_id=sid,
                total_bytes=total, lo=lo, nbytes=nbytes, first_block_offset=intra)


def test_golden_package_headers():
    gold = read_hex_fixture(os.path.join(HERE, "golden", "g3_package_headers.hex"))
    assert len(gold) == 192
    stream = np.frombuffer(read_hex_fixture(os.path.join(HERE, "golden", "p7_golden_stream.hex")), np.uint8)
    a = pkg.emit(stream, 128, SID, 2)
    b = pkg.emit(stream, 16, SID, 17)
    c = pkg.emit(stream, 128, SID, 1)
    assert bytes(a[:64]) == gold[0:64] and bytes(a[64:]) == bytes(stream[256:288])
    assert bytes(b[:64]) == gold[64:128] and bytes(b[64:]) == bytes(stream[272:288])
    assert bytes(c[:64]) == gold[128:192] and bytes(c[64:]) == bytes(stream[128:256])
    assert read_pkg_header(gold[0:64]) == dict(magic=b"BSPKG001", version=1, index=2, count=3, first_block=0, stream_id=SID,
                                               total_bytes=288, lo=256, nbytes=32, first_block_offset=0)
    assert read_pkg_header(gold[64:128])["first_block"] == 1 and read_pkg_header(gold[128:192])["first_block"] == pkg.NO_BLOCK


@pytest.mark.parametrize("hb,total,cap", [(256, 288, 128), (256, 288, 16), (128, 128, 64), (1152, 100000, 4096),
                                          (4096, 4096 + 3 * 4096, 4096), (384, 384 + 4096 + 16, 4096)])
def test_cut_is_the_stated_function(hb, total, cap):
    nh, npay = -(-hb // cap), -(-(total - hb) // cap)
    assert pkg.count(hb, total, cap) == nh + npay
    ranges = [pkg.package_range(hb, total, cap, k) for k in range(nh + npay)]
    want = [(k * cap, min((k + 1) * cap, hb)) for k in range(nh)] + \
           [(hb + k * cap, min(hb + (k + 1) * cap, total)) for k in range(npay)]
    assert ranges == want
    # a partition of [0, total) in index order; no package straddles the header / payload boundary
    assert ranges[0][0] == 0 and ranges[-1][1] == total
    assert all(a[1] == b[0] for a, b in zip(ranges[:-1], ranges[1:]))
    assert all(hi <= hb or lo >= hb for lo, hi in ranges) and all(0 < hi - lo <= cap for lo, hi in ranges)
    with pytest.raises(oracle.OracleError):
        pkg.package_range(hb, total, cap, nh + npay)
    assert pkg.count(hb, total, cap + 8) == 0          # the limit must be a multiple of 16


@pytest.mark.parametrize("cap", [16, 4096, 65536, 1 << 20])
def test_first_block_against_searchsorted_and_bytes(cap):
    bset = W.make_set("lognormal", 12, D=200, S=30, M=4, N0=3, n_ops=26, n_site=1, dims="lognormal", sigma=1.0)
    stream, _, _ = oracle_stream(bset)
    fixed, _, blocks, _, _ = read_stream(stream.tobytes())
    hb, total = fixed["header_bytes"], len(stream)
    offs = np.array([b["offset"] for b in blocks], dtype=np.int64)
    n = pkg.count(hb, total, cap)
    idxs = range(n) if n <= 400 else list(range(0, n, max(1, n // 300))) + [n - 1]
    for k in idxs:
        p = pkg.emit(stream, cap, SID, k)
        h = read_pkg_header(p[:64])
        lo, hi = pkg.package_range(hb, total, cap, k)
        assert (h["index"], h["count"], h["lo"], h["nbytes"], h["total_bytes"], h["stream_id"]) == (k, n, lo, hi - lo, total, SID)
        assert bytes(p[64:]) == bytes(stream[lo:hi])
        if lo < hb:
            assert h["first_block"] == pkg.NO_BLOCK and h["first_block_offset"] == 0
        else:
            i = int(np.searchsorted(offs, lo - hb, side="right")) - 1      # largest i with offset_i <= lo - hb
            assert h["first_block"] == i and h["first_block_offset"] == lo - hb - int(offs[i])


def test_zero_size_blocks_share_an_offset_the_last_one_holds_the_byte():
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 4, (0, 0), (-1, 1, 0, 0), 0, 0)
    dim = np.array([[2, 2, 1], [0, 3, 1], [0, 1, 1], [1, 2, 1]], np.uint32)       # offsets 0, 32, 32, 32
    data = [np.arange(4.0), np.zeros(0), np.zeros(0), np.arange(2.0)]
    addr = np.array([d.ctypes.data if d.size else 0 for d in data], dtype=np.uint64)
    s = oracle.serialize(tensors, np.zeros((4, 3, 2), np.int32), dim, addr)
    hb = oracle.stream_info(s)["header_bytes"]
    n = pkg.count(hb, len(s), 16)
    heads = [read_pkg_header(pkg.emit(s, 16, 1, k)[:64]) for k in range(n)]
    pay = [h for h in heads if h["lo"] >= hb]
    assert [(h["first_block"], h["first_block_offset"]) for h in pay] == [(0, 0), (0, 16), (3, 0)]


@pytest.mark.parametrize("cap", [16, 1024, 65536])
def test_packages_reassemble_in_any_order(cap):
    bset = W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    stream, _, _ = oracle_stream(bset)
    hb = oracle.stream_info(stream)["header_bytes"]
    n = pkg.count(hb, len(stream), cap)
    rng = np.random.default_rng(cap)
    n_slots = n + 5
    perm = rng.permutation(n_slots)[:n]                         # shuffled arrival, five slots stay empty
    slots = pkg.emit_slots(stream, cap, SID, 64 + cap, slot_of=perm, n_slots=n_slots, poison=0x5A)
    # packages of another serialization call mixed in (L124): different stream_id, skipped
    other = pkg.emit(stream, cap, SID + 1, 0)
    free = sorted(set(range(n_slots)) - set(int(x) for x in perm))
    slots[free[0], : other.size] = other
    got = pkg.assemble(slots, SID)
    assert got.size == len(stream) and (got == stream).all()
    assert oracle.validate_stream(got) == oracle.OK


def test_assemble_fault_injection():
    bset = W.make_config("1")
    stream, _, _ = oracle_stream(bset)
    cap = 4096
    slots = pkg.emit_slots(stream, cap, SID, 64 + cap)
    n = slots.shape[0]
    assert n >= 3 and (pkg.assemble(slots, SID) == stream).all()
    def bad(mut):
        s = slots.copy()
        mut(s)
        with pytest.raises(oracle.OracleError) as e:
            pkg.assemble(s, SID)
        assert e.value.code == oracle.ERR_CORRUPT
    bad(lambda s: s.__setitem__((1, 8), 2))                     # version
    bad(lambda s: s.__setitem__((1, 12), 0))                    # duplicate index 0, index 1 missing
    bad(lambda s: s.__setitem__((1, 16), n + 1))                # count disagrees
    bad(lambda s: s.__setitem__((1, 32), s[1, 32] ^ 0x10))      # total_bytes disagrees
    bad(lambda s: s.__setitem__((2, 40), s[2, 40] ^ 0x10))      # lo: ranges no longer tile the stream
    bad(lambda s: s.__setitem__((2, 48), s[2, 48] ^ 0x10))      # nbytes
    bad(lambda s: s.__setitem__((0, 0), 0x58))                  # a package lost (magic destroyed)
    with pytest.raises(oracle.OracleError) as e:
        pkg.assemble(slots, SID + 7)                            # no package of that call at all
    assert e.value.code == oracle.ERR_CORRUPT
    with pytest.raises(oracle.OracleError) as e:
        pkg.assemble(slots, SID, capacity=len(stream) - 1)
    assert e.value.code == oracle.ERR_CAPACITY and e.value.required == len(stream)


# ---- packages of wire-format-v2 streams (layered sets): blocks counted in the order of the descriptor's addr[] ----------
def test_golden_package_headers_of_the_v2_golden_stream():
    gold = read_hex_fixture(os.path.join(HERE, "golden", "g5_package_headers_v2.hex"))
    assert len(gold) == 192
    stream = np.frombuffer(read_hex_fixture(os.path.join(HERE, "golden", "g2_golden_stream_v2.hex")), np.uint8)
    a, b, c = pkg.emit(stream, 128, SID, 2), pkg.emit(stream, 16, SID, 19), pkg.emit(stream, 128, SID, 1)
    assert bytes(a[:64]) == gold[0:64] and bytes(a[64:]) == bytes(stream[256:320])
    assert bytes(b[:64]) == gold[64:128] and bytes(b[64:]) == bytes(stream[304:320])
    assert bytes(c[:64]) == gold[128:192] and bytes(c[64:]) == bytes(stream[128:256])
    assert read_pkg_header(pkg.emit(stream, 16, SID, 18))["first_block"] == 2


@pytest.mark.parametrize("cap", [16, 4096, 65536])
def test_first_block_of_v2_packages_against_searchsorted_and_reassembly(cap):
    from oracle import v2
    from tests.streamreader import read_stream_v2
    bset = W.make_config("1") if cap == 16 else W.make_config("2", n_ops=26)     # keep the number of packages bounded
    lv = W.layered_view(bset)
    pool, offs = W.fill_pool_host(bset)
    from tests.util import host_addrs
    s = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs))
    fixed, structs, layers, blocks, _, _ = read_stream_v2(s.tobytes())          # the independent reader
    starts = []
    for ly in layers:
        sr = structs[ly["structure"]]
        starts += [ly["offset"] + b["offset"] for b in blocks[sr["first_block"]: sr["first_block"] + sr["n_blocks"]]]
    starts = np.array(starts, np.uint64)
    assert (np.diff(starts.astype(np.int64)) >= 0).all() and len(starts) == bset.n_blocks
    hb = fixed["header_bytes"]
    n = pkg.count(hb, len(s), cap)
    for k in sorted(set([0, n - 1] + [int(x) for x in np.random.default_rng(cap).integers(0, n, 40)])):
        h = read_pkg_header(pkg.emit(s, cap, SID, k))
        lo, hi = pkg.package_range(hb, len(s), cap, k)
        assert (h["lo"], h["nbytes"], h["total_bytes"], h["count"]) == (lo, hi - lo, len(s), n)
        if lo < hb:
            assert h["first_block"] == pkg.NO_BLOCK and h["first_block_offset"] == 0
        else:
            i = int(np.searchsorted(starts, lo - hb, side="right")) - 1
            assert h["first_block"] == i and h["first_block_offset"] == lo - hb - int(starts[i])
    slots = pkg.emit_slots(s, cap, SID, 64 + cap, slot_of=np.random.default_rng(3).permutation(n))
    assert bytes(pkg.assemble(slots, SID)) == bytes(s)
