"""Pins of the element-type oracle (oracle/bs_oracle_dtype.py — SURVEY §8(f) NEXT-4): a hand-typed f32 golden stream, the
separately pinned C oracle for f64 (an independent implementation), c128 / c64 against f64 streams they must coincide
with, round trip, fault injection."""
import os
import struct

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import dt
from tests.util import host_addrs, read_hex_fixture

HERE = os.path.dirname(__file__)


def golden_f32_set():
    tensors = np.zeros(1, W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 2, (0, 0), (-1, 1, 0, 0), 9, 0)
    qn = np.array([[[0, 0], [0, 0], [0, 0]], [[1, 1], [1, 1], [0, 0]]], np.int32)
    dim = np.array([[1, 3, 1], [1, 1, 1]], np.uint32)
    blocks = [np.array([1.0, 2.0, 3.0], np.float32).tobytes(), np.array([-1.0], np.float32).tobytes()]
    return tensors, qn, dim, blocks


def test_golden_f32_stream():
    gold = read_hex_fixture(os.path.join(HERE, "golden", "g4_golden_stream_f32.hex"))
    assert len(gold) == 288
    t, qn, dim, blocks = golden_f32_set()
    got = dt.serialize(t, qn, dim, blocks, dt.F32)
    assert bytes(got) == gold
    back = dt.deserialize(np.frombuffer(gold, np.uint8))
    assert back["dtype"] == dt.F32 and back["blocks"] == blocks and (back["dim"] == dim).all() and (back["qn"] == qn).all()
    assert list(back["pool_off"]) == [0, 256] and back["pool_bytes"] == 512          # align256 slots (D14)
    assert np.frombuffer(back["pool"][:12].tobytes(), np.float32).tolist() == [1.0, 2.0, 3.0]
    assert (back["pool"][12:256] == 0xEE).all()                                       # exactly nbytes are written


def blocks_of(bset, pool, offs, scale=1):
    out = []
    for i in range(bset.n_blocks):
        o = int(offs[i])
        out.append(pool.view(np.uint8)[o: o + 8 * scale * int(bset.nelems[i]) // scale].tobytes())
    return out


@pytest.mark.parametrize("cfg,kw", [("1", {}), ("2", dict(n_ops=13)), ("3", dict(n_ops=13, D=300, S=30))])
def test_f64_equals_the_c_oracle_byte_for_byte(cfg, kw):
    bset = W.make_config(cfg, **kw)
    pool, offs = W.fill_pool_host(bset)
    want = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs))
    got = dt.serialize(bset.tensors, bset.qn, bset.dim, blocks_of(bset, pool, offs), dt.F64)
    assert bytes(got) == bytes(want)
    a, b = dt.deserialize(want), oracle.deserialize(want)
    assert (a["pool"][:a["pool_bytes"]] == b["pool"][:a["pool_bytes"]]).all() and a["pool_bytes"] == oracle.pool_bytes(want)
    assert (a["qn"] == b["qn"]).all() and (a["dim"] == b["dim"]).all() and a["tensors"] == b["tensors"].tobytes()


def test_c64_is_the_f64_stream_but_for_the_dtype_word_and_c128_payload_is_f64_with_a_doubled_extent():
    bset = W.make_config("2", n_ops=13)
    pool, offs = W.fill_pool_host(bset)
    blocks = blocks_of(bset, pool, offs)
    f64 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs))
    c64 = dt.serialize(bset.tensors, bset.qn, bset.dim, blocks, dt.C64)
    diff = np.nonzero(c64 != f64)[0]
    assert list(diff) == [16] and c64[16] == 2
    # c128: the same bytes seen as half as many 16-byte elements: dims with an even last extent only
    keep = [i for i in range(bset.n_blocks) if (int(bset.dim[i, 1]) * int(bset.dim[i, 2])) % 2 == 0 and bset.dim[i, 2] == 1][:40]
    t = np.zeros(1, W.TENSOR_REC_DTYPE)
    t[0] = (2, 0, len(keep), (0, 0), (-1, 1, 0, 0), 0, 0)
    d64 = bset.dim[keep].copy()
    d128 = d64.copy()
    d128[:, 1] //= 2
    sub = [blocks[i] for i in keep]
    subpool = np.frombuffer(b"".join(b.ljust((len(b) + 511) // 512 * 512, b"\0") for b in sub), np.uint8).copy()
    suboffs = np.concatenate([[0], np.cumsum([(len(b) + 511) // 512 * 512 for b in sub])[:-1]]).astype(np.uint64)
    f = oracle.serialize(t, bset.qn[keep], d64, host_addrs(subpool, suboffs))
    c = dt.serialize(t, bset.qn[keep], d128, sub, dt.C128)
    hb = oracle.header_bytes(1, len(keep))
    assert bytes(c[hb:]) == bytes(f[hb:]) and len(c) == len(f)
    assert all(len(b) % 16 == 0 for b in sub)                          # c128 blocks never carry pad


@pytest.mark.parametrize("dtype", [dt.F32, dt.C64, dt.C128])
def test_round_trip_and_sizes(dtype):
    rng = np.random.default_rng(40 + dtype)
    e = dt.ELEM_BYTES[dtype]
    bset = W.make_set("dt", 77, D=30, S=7, M=2, N0=2, n_ops=6, n_site=1, dims="multinomial")
    blocks = [rng.integers(0, 256, e * int(n), dtype=np.uint8).tobytes() for n in bset.nelems]
    s = dt.serialize(bset.tensors, bset.qn, bset.dim, blocks, dtype)
    nbytes, stored, offset, P = dt.plan(bset.dim, dtype)
    assert stored == [(b + 15) // 16 * 16 for b in nbytes] and nbytes == [e * int(n) for n in bset.nelems]
    assert offset == list(np.concatenate([[0], np.cumsum(stored)[:-1]]))           # numpy.cumsum: the textbook routine
    assert len(s) == dt.header_bytes(bset.n_tensors, bset.n_blocks) + P
    if dtype == dt.F32:
        assert {st - nb for st, nb in zip(stored, nbytes)} == {0, 4, 8, 12}      # every pad length occurs in this set
    back = dt.deserialize(s)
    assert back["blocks"] == blocks and back["dtype"] == dtype
    assert bytes(dt.serialize(bset.tensors, back["qn"], back["dim"], back["blocks"], dtype)) == bytes(s)   # fixpoint


def test_fault_injection():
    t, qn, dim, blocks = golden_f32_set()
    s = dt.serialize(t, qn, dim, blocks, dt.F32)
    for pos, what in [(16, "dtype"), (0x10c, "pad of block 0"), (0x114, "pad of block 1"), (0xb8, "offset"), (0x7c, "dim"),
                      (56, "payload_bytes"), (0xc0, "slack")]:
        bad = s.copy()
        bad[pos] ^= 0x04
        with pytest.raises(oracle.OracleError) as e:
            dt.deserialize(bad)
        assert e.value.code == oracle.ERR_CORRUPT, what
    with pytest.raises(oracle.OracleError):
        dt.serialize(t, qn, dim, blocks, 7)
    with pytest.raises(oracle.OracleError):
        dt.serialize(t, qn, dim, [blocks[0], blocks[1] + b"\0"], dt.F32)
