"""Pins of reading D19 — wire format v1 with align = 8, the unpadded stream (oracle/bs_oracle.c `_al` entry points and
oracle/bs_oracle_dtype.py; BASELINE.json north_star: "offsets equal to the exclusive prefix
sum of the block byte sizes").  None of them retypes the oracle's loops: hand-typed golden bytes, the independent struct
reader, numpy.cumsum on the UNPADDED sizes, plain concatenation of the blocks, two independently written oracles."""
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import dt
from tests.streamreader import block_doubles, read_stream
from tests.test_oracle_golden import GOLD as GOLD16
from tests.test_oracle_golden import golden_set
from tests.util import host_addrs, read_hex_fixture, sha256

GOLD = os.path.join(os.path.dirname(__file__), "golden", "g7_golden_stream_align8.hex")
GOLD_SHA = "d881b02837d099c282f4b4c8d950b5257dca371c920c21305a6a3ff1d9edc41f"


def sets():
    yield W.make_config("1")
    yield W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    yield W.make_set("lognormal", 12, D=200, S=30, M=4, N0=3, n_ops=40, n_site=1, dims="lognormal", sigma=1.0)


def test_G7_fixture_oracle_and_reader():
    raw = read_hex_fixture(GOLD)
    assert len(raw) == 280 and sha256(raw) == GOLD_SHA
    # exactly three fields differ from the align-16 golden P7: align, payload_bytes, offset of block 1 (and the pad is gone)
    p7 = read_hex_fixture(GOLD16)
    diff = [i for i in range(256) if raw[i] != p7[i]]
    assert diff == [0x1C, 0x38, 0xB8]
    tensors, qn, dim, blocks = golden_set()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = oracle.serialize(tensors, qn, dim, addr, align=8)
    assert bytes(s) == raw
    assert oracle.serialized_size(1, dim, align=8) == (256, 280)
    fixed, tr, br, slack, payload = read_stream(raw)
    assert fixed["align"] == 8 and fixed["payload_bytes"] == 24 and [b["offset"] for b in br] == [0, 8]
    assert block_doubles(payload, br[0]) == (1.0,) and block_doubles(payload, br[1]) == (2.0, 3.0)
    # back: the same object as from the padded stream
    arr = np.frombuffer(raw, np.uint8)
    assert oracle.validate_stream(arr) == oracle.OK and oracle.stream_info(arr)["align"] == 8
    a, b = oracle.deserialize(arr), oracle.deserialize(np.frombuffer(p7, np.uint8))
    assert a["tensors"].tobytes() == b["tensors"].tobytes() and (a["qn"] == b["qn"]).all() and (a["dim"] == b["dim"]).all()
    assert (a["pool"] == b["pool"]).all()
    assert oracle.pool_bytes(arr) == 512


@pytest.mark.parametrize("bset", list(sets()), ids=lambda s: s.name)
def test_offsets_are_the_prefix_sum_of_the_block_byte_sizes_and_the_payload_is_the_concatenation(bset):
    pool, offs = W.fill_pool_host(bset)
    addr = host_addrs(pool, offs)
    s = oracle.serialize(bset.tensors, bset.qn, bset.dim, addr, align=8)
    nbytes, stored, offset, P = oracle.plan(bset.dim, align=8)
    raw8 = (bset.nelems * np.uint64(8)).astype(np.uint64)
    assert (nbytes == raw8).all() and (stored == raw8).all()                       # fp64: no pad byte at all
    assert offset.tolist() == np.concatenate([[0], np.cumsum(raw8)])[:-1].tolist()   # the literal north_star invariant
    assert P == int(raw8.sum())
    hb = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
    assert oracle.serialized_size(bset.n_tensors, bset.dim, align=8) == (hb, hb + P) and len(s) == hb + P
    # the independent reader: offsets in the stream are those; the payload is the blocks back to back
    fixed, _, br, slack, payload = read_stream(s.tobytes())
    assert fixed["align"] == 8 and [b["offset"] for b in br] == offset.tolist() and set(slack) <= {0}
    rawpool = pool.view(np.uint8)
    cat = b"".join(rawpool[int(o): int(o) + int(n)].tobytes() for o, n in zip(offs, raw8))
    assert payload == cat
    # it is shorter than the padded stream by 8 bytes per odd-sized block, and the same header but for three kinds of fields
    s16 = oracle.serialize(bset.tensors, bset.qn, bset.dim, addr)
    assert len(s16) - len(s) == 8 * int((bset.nelems % 2 == 1).sum())
    # slice-wise emit (O-5) agrees with the whole stream
    if bset.n_tensors >= 2:
        t0, t1 = 1, bset.n_tensors
        b0 = int(bset.tensors["first_block"][t0])
        first, got = oracle.emit_payload_range(bset.tensors, bset.dim, addr, t0, t1, P, align=8)
        assert first == int(offset[b0]) and (got == s[hb + first:]).all()
    assert (oracle.emit_header(bset.tensors, bset.qn, bset.dim, align=8) == s[:hb]).all()
    # round trip and fixpoint
    out = oracle.deserialize(s)
    ref = oracle.deserialize(s16)
    assert (out["pool"] == ref["pool"]).all() and out["tensors"].tobytes() == bset.tensors.tobytes()
    again = oracle.serialize(out["tensors"], out["qn"], out["dim"], out["addr"], align=8)
    assert (again == s).all()


@pytest.mark.parametrize("dtype", [0, 1, 2, 3])
@pytest.mark.parametrize("bset", list(sets()), ids=lambda s: s.name)
def test_two_independent_oracles_agree_at_align_8(bset, dtype):
    """bs_oracle_dtype.py (numpy / struct, written independently) at align 8: byte-equal to the C oracle for f64; for the
    other element types offsets against numpy.cumsum of align_up(e*n, 8), round trip, fixpoint."""
    e = {0: 8, 1: 4, 2: 8, 3: 16}[dtype]
    pool, offs = W.fill_pool_host(bset)
    if e == 16:
        big = np.zeros(2 * pool.size + 2, np.float64)
        offs = offs * 2
        for o, n in zip(offs, bset.nelems):
            src = pool[int(o) // 16: int(o) // 16 + int(n)]
            big[int(o) // 8: int(o) // 8 + 2 * int(n)] = np.repeat(src, 2)
        pool = big
    raw = pool.view(np.uint8)
    blocks = [raw[int(o): int(o) + e * int(n)] for o, n in zip(offs, bset.nelems)]
    s = dt.serialize(bset.tensors, bset.qn, bset.dim, blocks, dtype, align=8)
    if dtype == 0:
        c = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs), align=8)
        assert (s == c).all()
    nb = np.uint64(e) * bset.nelems
    st = (nb + np.uint64(7)) // np.uint64(8) * np.uint64(8)
    fixed, _, br, _, payload = read_stream(s.tobytes())
    assert fixed["align"] == 8 and fixed["dtype"] == dtype
    assert [b["offset"] for b in br] == np.concatenate([[0], np.cumsum(st)])[:-1].tolist() and len(payload) == int(st.sum())
    if dtype == 1:
        assert set(int(x) for x in (st - nb)) <= {0, 4} and 4 in set(int(x) for x in (st - nb))
    else:
        assert (st == nb).all()
    out = dt.deserialize(s)
    assert out["align"] == 8 and all(bytes(a) == bytes(b) for a, b in zip(out["blocks"], blocks))
    assert (dt.serialize(bset.tensors, bset.qn, bset.dim, out["blocks"], dtype, align=8) == s).all()


def test_fault_injection_and_bad_alignments():
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    pool, offs = W.fill_pool_host(bset)
    addr = host_addrs(pool, offs)
    s = oracle.serialize(bset.tensors, bset.qn, bset.dim, addr, align=8)
    assert oracle.validate_stream(s) == oracle.OK
    for al in (0, 4, 12, 32):
        with pytest.raises(oracle.OracleError) as e:
            oracle.serialize(bset.tensors, bset.qn, bset.dim, addr, align=al)
        assert e.value.code == oracle.ERR_UNSUPPORTED
        bad = s.copy()
        bad[0x1C] = al
        assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
    # an align-8 stream relabelled 16 (and the other way round) breaks the offset chain
    bad = s.copy()
    bad[0x1C] = 16
    assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
    s16 = oracle.serialize(bset.tensors, bset.qn, bset.dim, addr)
    bad = s16.copy()
    bad[0x1C] = 8
    assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
    # every block offset, the payload size, a truncated stream
    hb = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
    for i in (0, 1, bset.n_blocks // 2, bset.n_blocks - 1):
        bad = s.copy()
        bad[64 + 32 * bset.n_tensors + 48 * i + 40] ^= 8
        assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
    bad = s.copy()
    bad[0x38] ^= 8
    assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT
    assert oracle.validate_stream(s[:-8]) == oracle.ERR_CORRUPT
    with pytest.raises(oracle.OracleError):
        dt.deserialize(s[:-8])
