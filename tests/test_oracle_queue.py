"""Pins of the queue model (oracle/bs_oracle_queue.py — SURVEY §8(f) NEXT-3): a hand-traced sequence over
the golden stream P7, the accounting against sums typed by hand, errors."""
import os

import numpy as np
import pytest

import oracle
import workloads as W
from tests.util import host_addrs, read_hex_fixture

HERE = os.path.dirname(__file__)


def golden_set(values=(1.0, 2.0, 3.0)):
    """The set of the 288-byte golden stream P7, typed out here."""
    tensors = np.zeros(1, W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 2, (1, 1), (-1, 1, 0, 0), 7, 0)
    qn = np.array([[[0, 0], [1, 1], [0, 0]], [[1, -1], [2, 0], [0, 0]]], np.int32)
    dim = np.array([[1, 1, 1], [1, 2, 1]], np.uint32)
    pool = np.zeros(128, np.float64)
    pool[0], pool[64], pool[65] = values
    return tensors, qn, dim, pool, np.array([0, 512], np.uint64)


def test_hand_traced_sequence_over_the_golden_stream():
    gold = read_hex_fixture(os.path.join(HERE, "golden", "p7_golden_stream.hex"))
    q = oracle.QueueModel()
    t, qn, dim, pool, offs = golden_set()
    addr = host_addrs(pool.view(np.uint8), offs)
    s = q.save(7, t, qn, dim, addr)
    assert bytes(s) == gold                                   # what the store holds is the v1 stream
    pool[0] = 99.0                                            # the source changes AFTER the save: the store must not
    got = q.load(7)
    assert got["pool"].view(np.float64)[0] == 1.0             # block 0 at pool offset 0
    assert list(got["pool"].view(np.float64)[32:34]) == [2.0, 3.0]   # block 1 at align256(8) = 256 bytes
    assert q.stats() == dict(saves=1, loads=1, bytes_saved=288, bytes_loaded=288, host_bytes_live=288, host_bytes_peak=288,
                             keys_live=1)
    # a second key, then key 7 saved again with the changed source: the load sees the LAST save (program order)
    t2, qn2, dim2, pool2, offs2 = golden_set((4.0, 5.0, 6.0))
    q.save(8, t2, qn2, dim2, host_addrs(pool2.view(np.uint8), offs2))
    q.save(7, t, qn, dim, addr)
    assert q.load(7)["pool"].view(np.float64)[0] == 99.0 and q.load(8)["pool"].view(np.float64)[0] == 4.0
    assert q.stats() == dict(saves=3, loads=3, bytes_saved=864, bytes_loaded=864, host_bytes_live=576, host_bytes_peak=576,
                             keys_live=2)
    q.forget(8)
    assert q.stats()["host_bytes_live"] == 288 and q.stats()["host_bytes_peak"] == 576 and q.stats()["keys_live"] == 1
    with pytest.raises(oracle.OracleError) as e:
        q.load(8)
    assert e.value.code == oracle.ERR_ARG
    with pytest.raises(oracle.OracleError):
        q.forget(8)


def test_adopted_streams_and_corruption():
    gold = np.frombuffer(read_hex_fixture(os.path.join(HERE, "golden", "p7_golden_stream.hex")), np.uint8)
    q = oracle.QueueModel()
    q.adopt(1, gold)
    assert q.stats()["host_bytes_live"] == 288 and q.stats()["saves"] == 0
    assert q.load(1)["pool"].view(np.float64)[0] == 1.0
    bad = gold.copy()
    bad[0xB8] ^= 0x10                                         # block 1's offset field
    q.adopt(2, bad)
    with pytest.raises(oracle.OracleError) as e:
        q.load(2)
    assert e.value.code == oracle.ERR_CORRUPT
    assert q.stats()["loads"] == 1                            # a refused load is not counted


def test_a_longer_seeded_sequence_keeps_per_key_program_order():
    rng = np.random.default_rng(5)
    q = oracle.QueueModel()
    last = {}
    live = 0
    peak = 0
    for step in range(40):
        key = int(rng.integers(0, 4))
        if rng.random() < 0.6 or key not in last:
            bset = W.make_set(f"q{step}", 100 + step, D=24, S=6, M=2, N0=2, n_ops=int(rng.integers(1, 5)), n_site=0,
                              dims="multinomial")
            pool, offs = W.fill_pool_host(bset)
            s = q.save(key, bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs))
            last[key] = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs))
            assert bytes(s) == bytes(last[key])
        else:
            got = q.load(key)
            assert (got["pool"] == oracle.deserialize(last[key])["pool"]).all()
        live = sum(len(v) for v in last.values())
        peak = max(peak, live)
        assert q.stats()["host_bytes_live"] == live and q.stats()["host_bytes_peak"] == peak


def test_layered_streams_share_the_store_but_not_the_load_call():
    """A key holds a stream of one wire format; the G2 golden v2 stream is what a layered save stores."""
    from oracle import v2
    from tests.test_oracle_v2 import GOLD, golden_set as golden_v2
    gold = read_hex_fixture(GOLD)
    q = oracle.QueueModel()
    structs, layers, qn, dim, blocks = golden_v2()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = q.save_layered(3, structs, layers, qn, dim, addr)
    assert bytes(s) == gold and q.stats()["host_bytes_live"] == len(gold) and q.stats()["saves"] == 1
    got = q.load_layered(3)
    assert (got["pool"] == v2.deserialize(np.frombuffer(gold, np.uint8))["pool"]).all()
    with pytest.raises(oracle.OracleError) as e:
        q.load(3)
    assert e.value.code == oracle.ERR_ARG
    t, qn1, dim1, pool, offs = golden_set()
    q.save(3, t, qn1, dim1, host_addrs(pool.view(np.uint8), offs))      # the key changes format with the save
    with pytest.raises(oracle.OracleError):
        q.load_layered(3)
    assert q.load(3)["pool"].view(np.float64)[0] == 1.0 and q.stats()["loads"] == 2


def test_spill_and_fill_are_the_stream_bytes_in_a_file(tmp_path):
    """PAPER L85 step (2): the file holds exactly the serialized bytes; reading it back is an adopted stream."""
    gold = read_hex_fixture(os.path.join(HERE, "golden", "p7_golden_stream.hex"))
    q = oracle.QueueModel()
    t, qn, dim, pool, offs = golden_set()
    q.save(7, t, qn, dim, host_addrs(pool.view(np.uint8), offs))
    path = str(tmp_path / "block7.bs")
    assert q.spill(7, path) == 288 and open(path, "rb").read() == gold
    q.forget(7)
    assert q.stats()["host_bytes_live"] == 0
    assert q.fill(9, path) == 288 and q.stats()["host_bytes_live"] == 288
    assert list(q.load(9)["pool"].view(np.float64)[32:34]) == [2.0, 3.0]
    assert (q.bytes_spilled, q.bytes_filled) == (288, 288)
    with pytest.raises(oracle.OracleError) as e:
        q.fill(1, str(tmp_path / "missing.bs"))
    assert e.value.code == -6
    with pytest.raises(oracle.OracleError):
        q.spill(1, path)
