"""P7 — the oracle against a hand-typed 288-byte stream (tests/golden/p7_golden_stream.hex) and against an
independent struct-based reader.  Pins the byte format: field order, widths, endianness, header rounding to
128, block rounding to 16, zero padding.  (DESIGN.md "Wire format v1".)"""
import os

import numpy as np

import oracle
import workloads as W
from tests.streamreader import block_doubles, read_stream
from tests.util import read_hex_fixture, sha256

GOLD = os.path.join(os.path.dirname(__file__), "golden", "p7_golden_stream.hex")
GOLD_SHA = "81013cb579c05d6d1f68efd6a8d00029d8edc3525195282cc437daecc932a639"


def golden_set():
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 2, (1, 1), (-1, 1, 0, 0), 7, 0)
    qn = np.array([[[0, 0], [1, 1], [0, 0]], [[1, -1], [2, 0], [0, 0]]], dtype=np.int32)
    dim = np.array([[1, 1, 1], [1, 2, 1]], dtype=np.uint32)
    b0 = np.array([1.0])
    b1 = np.array([2.0, 3.0])
    return tensors, qn, dim, [b0, b1]


def test_fixture_is_the_cited_one():
    raw = read_hex_fixture(GOLD)
    assert len(raw) == 288
    assert sha256(raw) == GOLD_SHA


def test_oracle_reproduces_golden_bytes():
    tensors, qn, dim, blocks = golden_set()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = oracle.serialize(tensors, qn, dim, addr)
    assert bytes(s) == read_hex_fixture(GOLD)
    assert oracle.serialized_size(1, dim) == (256, 288)


def test_independent_reader_sees_the_stated_fields():
    fixed, tensors, blocks, slack, payload = read_stream(read_hex_fixture(GOLD))
    assert fixed == dict(magic=b"BSPARSE1", version=1, endian_tag=0x01020304, dtype=0, n_qn=2, max_rank=3, align=16,
                         n_tensors=1, n_blocks=2, header_bytes=256, payload_bytes=32)
    assert tensors == [dict(rank=2, first_block=0, n_blocks=2, dq=(1, 1), sign=(-1, 1, 0, 0), tag=7, reserved=0)]
    assert blocks[0] == dict(qn=((0, 0), (1, 1), (0, 0)), dim=(1, 1, 1), tensor=0, offset=0)
    assert blocks[1] == dict(qn=((1, -1), (2, 0), (0, 0)), dim=(1, 2, 1), tensor=0, offset=16)
    assert slack == bytes(64) and len(payload) == 32
    assert block_doubles(payload, blocks[0]) == (1.0,)
    assert block_doubles(payload, blocks[1]) == (2.0, 3.0)
    assert payload[8:16] == bytes(8)            # pad after the odd-sized block


def test_oracle_deserializes_golden():
    raw = np.frombuffer(read_hex_fixture(GOLD), dtype=np.uint8)
    assert oracle.validate_stream(raw) == oracle.OK
    out = oracle.deserialize(raw)
    tensors, qn, dim, blocks = golden_set()
    assert out["tensors"].tobytes() == tensors.tobytes()
    assert (out["qn"] == qn).all() and (out["dim"] == dim).all()
    base = out["pool"].ctypes.data
    assert [int(a) - base for a in out["addr"]] == [0, 256]            # D14: 256-byte pool slots
    assert out["pool"][0:8].view(np.float64)[0] == 1.0
    assert tuple(out["pool"][256:272].view(np.float64)) == (2.0, 3.0)
    assert (out["pool"][8:256] == 0xEE).all()                           # nothing beyond nbytes is touched
