"""Pins of the v3 oracle (oracle/bs_oracle_v3.c — wire format v3, tensors of rank up to 4; DESIGN.md
§19 reading D20).  None of them retypes the oracle's loops: hand-typed golden bytes, an independent struct reader,
numpy.cumsum, the (separately pinned) v1 oracle on sets of rank <= 3, dense brute force on order-4 arrays."""
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import v3
from tests.streamreader import read_stream, read_stream_v3
from tests.util import host_addrs, read_hex_fixture, sha256

GOLD = os.path.join(os.path.dirname(__file__), "golden", "g8_golden_stream_v3.hex")
GOLD_SHA = "29fca8ec04cbed08c417867f23924ceeb02e5fef3d7e5cf109af2725c6a814a1"


def golden_set():
    tensors = np.zeros(2, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (4, 0, 2, (0, 0), (1, 1, 1, -1), 5, 0)
    tensors[1] = (2, 2, 1, (1, 1), (-1, 1, 0, 0), 7, 0)
    qn = np.array([[[0, 0], [1, 1], [1, -1], [2, 0]], [[1, 1], [0, 0], [0, 0], [1, 1]], [[0, 0], [1, 1], [0, 0], [0, 0]]], np.int32)
    dim = np.array([[1, 1, 1, 2], [1, 1, 1, 1], [1, 3, 1, 1]], np.uint32)
    blocks = [np.array([1.0, 2.0]), np.array([3.0]), np.array([4.0, 5.0, 6.0])]
    return tensors, qn, dim, blocks


def tree_sets():
    yield W.make_tree_set("tree-small", 5)
    yield W.make_tree_set("tree-ops-only", 6, n_nodes=0, n_ops=9)
    yield W.make_tree_set("tree", 7, D=40, S=8, n_nodes=4, n_ops=5)


def stream_of(bset, dtype=0):
    pool, offs = W.fill_pool_host(bset)
    return v3.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs), dtype), pool, offs


def test_G8_fixture_oracle_and_reader():
    raw = read_hex_fixture(GOLD)
    assert len(raw) == 448 and sha256(raw) == GOLD_SHA
    tensors, qn, dim, blocks = golden_set()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = v3.serialize(tensors, qn, dim, addr)
    assert bytes(s) == raw
    assert v3.serialized_size(2, dim) == (384, 448) and v3.header_bytes(2, 3) == 384
    fixed, tr, br, slack, payload = read_stream_v3(raw)
    assert fixed == dict(magic=b"BSPARSE1", version=3, endian_tag=0x01020304, dtype=0, n_qn=2, max_rank=4, align=16,
                         n_tensors=2, n_blocks=3, header_bytes=384, payload_bytes=64)
    assert tr == [dict(rank=4, first_block=0, n_blocks=2, dq=(0, 0), sign=(1, 1, 1, -1), tag=5, reserved=0),
                  dict(rank=2, first_block=2, n_blocks=1, dq=(1, 1), sign=(-1, 1, 0, 0), tag=7, reserved=0)]
    assert [b["offset"] for b in br] == [0, 16, 32] and [b["tensor"] for b in br] == [0, 0, 1]
    assert br[0]["qn"] == ((0, 0), (1, 1), (1, -1), (2, 0)) and br[0]["dim"] == (1, 1, 1, 2)
    assert br[2]["qn"] == ((0, 0), (1, 1), (0, 0), (0, 0)) and br[2]["dim"] == (1, 3, 1, 1)
    assert slack == bytes(64)
    assert np.frombuffer(payload, np.float64).tolist() == [1, 2, 3, 0, 4, 5, 6, 0]
    arr = np.frombuffer(raw, np.uint8)
    assert v3.validate_stream(arr) == oracle.OK
    out = v3.deserialize(arr)
    assert out["tensors"].tobytes() == tensors.tobytes() and (out["qn"] == qn).all() and (out["dim"] == dim).all()
    base = out["pool"].ctypes.data
    assert [int(a) - base for a in out["addr"]] == [0, 256, 512] and v3.pool_bytes(arr) == 768
    assert out["pool"][512:536].view(np.float64).tolist() == [4, 5, 6] and (out["pool"][536:768] == 0xEE).all()
    assert v3.validate_set(tensors, qn) == 0


@pytest.mark.parametrize("dtype", [0, 1, 3])
@pytest.mark.parametrize("bset", list(tree_sets()), ids=lambda s: s.name)
def test_offsets_sizes_round_trip_and_fixpoint(bset, dtype):
    e = {0: 8, 1: 4, 3: 16}[dtype]
    pool, offs = W.fill_pool_host(bset)
    if e == 16:
        pool = np.concatenate([pool, pool])           # room to read 16-byte elements (values are arbitrary bits)
    s = v3.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs), dtype)
    nb = np.uint64(e) * bset.nelems
    st = (nb + np.uint64(15)) // np.uint64(16) * np.uint64(16)
    nbytes, stored, offset, P = v3.plan(bset.dim, dtype)
    assert (nbytes == nb).all() and (stored == st).all() and P == int(st.sum())
    assert offset.tolist() == np.concatenate([[0], np.cumsum(st)])[:-1].tolist()
    hb = (64 + 32 * bset.n_tensors + 64 * bset.n_blocks + 127) // 128 * 128
    assert v3.serialized_size(bset.n_tensors, bset.dim, dtype) == (hb, hb + P) and len(s) == hb + P
    fixed, tr, br, slack, payload = read_stream_v3(s.tobytes())
    assert fixed["dtype"] == dtype and [b["offset"] for b in br] == offset.tolist() and set(slack) <= {0}
    t_of_b = np.repeat(np.arange(bset.n_tensors), bset.tensors["n_blocks"])
    assert [b["tensor"] for b in br] == t_of_b.tolist()
    raw = pool.view(np.uint8)
    for i in (0, bset.n_blocks // 2, bset.n_blocks - 1):
        o = int(offset[i])
        assert payload[o: o + int(nb[i])] == raw[int(offs[i]): int(offs[i]) + int(nb[i])].tobytes()
        assert payload[o + int(nb[i]): o + int(st[i])] == bytes(int(st[i] - nb[i]))
    out = v3.deserialize(s)
    assert out["tensors"].tobytes() == bset.tensors.tobytes() and (out["qn"] == bset.qn).all() and (out["dim"] == bset.dim).all()
    slots = (nb + np.uint64(255)) // np.uint64(256) * np.uint64(256)
    base = out["pool"].ctypes.data
    assert (out["addr"] - np.uint64(base)).tolist() == np.concatenate([[0], np.cumsum(slots)])[:-1].tolist()
    again = v3.serialize(out["tensors"], out["qn"], out["dim"], out["addr"], dtype)
    assert (again == s).all()
    # conservation of every stored block, read from the stream alone (D10 with four legs)
    for b in br[:: max(1, len(br) // 200)]:
        t = tr[b["tensor"]]
        for c in range(2):
            assert sum(t["sign"][k] * b["qn"][k][c] for k in range(4)) == t["dq"][c]
    assert v3.validate_set(bset.tensors, bset.qn) == 0


def test_rank_le_3_sets_have_the_v1_payload():
    """A set without order-4 tensors, written with a fourth leg of extent 1: its v3 payload is byte for byte the payload of
    the separately pinned v1 oracle, and the block offsets agree."""
    for bset in (W.make_config("1"), W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")):
        pool, offs = W.fill_pool_host(bset)
        addr = host_addrs(pool, offs)
        s1 = oracle.serialize(bset.tensors, bset.qn, bset.dim, addr)
        qn4 = np.zeros((bset.n_blocks, 4, 2), np.int32)
        dim4 = np.ones((bset.n_blocks, 4), np.uint32)
        qn4[:, :3], dim4[:, :3] = bset.qn, bset.dim
        s3 = v3.serialize(bset.tensors, qn4, dim4, addr)
        i1, i3 = oracle.stream_info(s1), v3.stream_info(s3)
        assert i1["payload_bytes"] == i3["payload_bytes"]
        assert (s1[i1["header_bytes"]:] == s3[i3["header_bytes"]:]).all()
        _, _, b1, _, _ = read_stream(s1.tobytes())
        _, _, b3, _, _ = read_stream_v3(s3.tobytes())
        assert [b["offset"] for b in b1] == [b["offset"] for b in b3]
        assert all(x["qn"] == y["qn"][:3] and x["dim"] == y["dim"][:3] and y["dim"][3] == 1 and y["qn"][3] == (0, 0) for x, y in zip(b1, b3))


def test_dense_reconstruction_of_order_4_arrays():
    """P5 with four indices: a dense order-4 array, non-zero only where label_a + label_b + q_s = label_c; cut the blocks out
    of it, serialize, deserialize, scatter the blocks back by their sector offsets, compare with the dense original bitwise."""
    rng = np.random.default_rng(3)
    la = [(0, 0), (1, 1), (1, -1)]
    ls = [(0, 0), (1, 1), (1, -1), (2, 0)]
    lc = [(0, 0), (1, 1), (1, -1), (2, 0), (2, 2), (3, 1), (3, -1), (4, 0)]
    da, db, dc = [2, 1, 3], [1, 2, 2], [1, 2, 1, 3, 1, 2, 1, 2]
    oa, ob, oc = np.concatenate([[0], np.cumsum(da)]), np.concatenate([[0], np.cumsum(db)]), np.concatenate([[0], np.cumsum(dc)])
    dense = np.zeros((sum(da), sum(db), 4, sum(dc)))
    qn, dim, blocks, where = [], [], [], []
    for a, qa in enumerate(la):
        for b, qb in enumerate(la):
            for sg, qs in enumerate(ls):
                tot = (qa[0] + qb[0] + qs[0], qa[1] + qb[1] + qs[1])
                if tot in lc:
                    c = lc.index(tot)
                    blk = rng.uniform(-1, 1, (da[a], db[b], 1, dc[c]))
                    dense[oa[a]:oa[a + 1], ob[b]:ob[b + 1], sg:sg + 1, oc[c]:oc[c + 1]] = blk
                    qn.append([qa, qb, qs, tot])
                    dim.append([da[a], db[b], 1, dc[c]])
                    blocks.append(np.ascontiguousarray(blk))
                    where.append((a, b, sg, c))
    B = len(blocks)
    assert B > 20
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (4, 0, B, (0, 0), (1, 1, 1, -1), 1, 0)
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = v3.serialize(tensors, np.array(qn, np.int32), np.array(dim, np.uint32), addr)
    out = v3.deserialize(s)
    back = np.zeros_like(dense)
    base = out["pool"].ctypes.data
    for i, (a, b, sg, c) in enumerate(where):
        d = out["dim"][i]
        n = int(np.prod(d.astype(np.int64)))
        o = int(out["addr"][i]) - base
        vals = out["pool"][o: o + 8 * n].view(np.float64).reshape([int(x) for x in d])     # row-major, last index fastest (D4)
        # the labels in the stream say where the block goes
        q = out["qn"][i]
        assert (tuple(q[0]), tuple(q[1]), tuple(q[2]), tuple(q[3])) == (la[a], la[b], ls[sg], lc[c])
        back[oa[a]:oa[a + 1], ob[b]:ob[b + 1], sg:sg + 1, oc[c]:oc[c + 1]] = vals
    assert back.tobytes() == dense.tobytes()


def test_fault_injection_every_validated_field():
    bset = W.make_tree_set("fault", 9, D=12, S=4, n_nodes=2, n_ops=3)
    s, _, _ = stream_of(bset)
    assert v3.validate_stream(s) == oracle.OK
    T, B = bset.n_tensors, bset.n_blocks
    hb = v3.header_bytes(T, B)
    t0, b0 = 64, 64 + 32 * T
    r2 = int(np.nonzero(bset.tensors["rank"] == 2)[0][0])
    fb2 = int(bset.tensors["first_block"][r2])
    muts = [("magic", 0, 1), ("version", 8, 2), ("endian", 12, 1), ("dtype", 16, 4), ("n_qn", 20, 1), ("max_rank", 24, 1),
            ("align", 28, 8), ("n_tensors", 32, 1), ("n_blocks", 40, 1), ("header_bytes", 48, 128), ("payload_bytes", 56, 16),
            ("rank", t0, 1), ("rank5", t0 + 32, 7), ("first_block", t0 + 32 + 4, 1), ("n_blocks_t", t0 + 8, 1), ("t_reserved", t0 + 28, 1),
            ("owner", b0 + 48, 1), ("b_reserved", b0 + 52, 1), ("offset0", b0 + 56, 16), ("offset_k", b0 + 64 * (B // 2) + 56, 16),
            ("dim_leg4", b0 + 64 * 1 + 44, 1), ("unused_dim_of_rank2", b0 + 64 * fb2 + 40, 2), ("unused_qn_of_rank2", b0 + 64 * fb2 + 24, 1),
            ("unused_leg4_of_rank2", b0 + 64 * fb2 + 44, 3)]
    if b0 + 64 * B < hb:
        muts.append(("slack", hb - 1, 1))
    odd = np.nonzero(bset.nelems % 2 == 1)[0]
    if len(odd):
        _, _, off, _ = v3.plan(bset.dim)
        muts.append(("pad", hb + int(off[odd[0]]) + 8 * int(bset.nelems[odd[0]]), 1))
    for name, pos, xor in muts:
        bad = s.copy()
        bad[pos] ^= xor
        assert v3.validate_stream(bad) == oracle.ERR_CORRUPT, name
        with pytest.raises(oracle.OracleError):
            v3.deserialize(bad)
    assert v3.validate_stream(s[:-16]) == oracle.ERR_CORRUPT and v3.validate_stream(s[:48]) == oracle.ERR_CORRUPT
    # descriptors: rank 5, a hole in the partition, an unknown element type
    t = bset.tensors.copy()
    t["rank"][0] = 5
    pool, offs = W.fill_pool_host(bset)
    with pytest.raises(oracle.OracleError) as e:
        v3.serialize(t, bset.qn, bset.dim, host_addrs(pool, offs))
    assert e.value.code == oracle.ERR_UNSUPPORTED
    t = bset.tensors.copy()
    t["n_blocks"][0] -= 1
    with pytest.raises(oracle.OracleError) as e:
        v3.serialize(t, bset.qn, bset.dim, host_addrs(pool, offs))
    assert e.value.code == oracle.ERR_ARG
    with pytest.raises(oracle.OracleError) as e:
        v3.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs), dtype=4)
    assert e.value.code == oracle.ERR_UNSUPPORTED
    # a flipped label breaks conservation (helper, not the serializer: D12)
    q = bset.qn.copy()
    q[1, 3, 0] += 1
    assert v3.validate_set(bset.tensors, q) == 1


def test_empty_and_zero_extent():
    tensors = np.zeros(0, dtype=W.TENSOR_REC_DTYPE)
    s = v3.serialize(tensors, np.zeros((0, 4, 2), np.int32), np.zeros((0, 4), np.uint32), np.zeros(0, np.uint64))
    assert len(s) == 128 and v3.validate_stream(s) == oracle.OK
    tensors = np.zeros(2, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (4, 0, 2, (0, 0), (1, 1, 1, -1), 0, 0)
    tensors[1] = (3, 2, 0, (0, 0), (1, 1, -1, 0), 1, 0)
    dim = np.array([[2, 0, 1, 3], [1, 1, 1, 1]], np.uint32)
    b = [np.zeros(0), np.array([7.0])]
    s = v3.serialize(tensors, np.zeros((2, 4, 2), np.int32), dim, np.array([x.ctypes.data for x in b], np.uint64))
    _, _, br, _, payload = read_stream_v3(s.tobytes())
    assert [x["offset"] for x in br] == [0, 0] and len(payload) == 16
    out = v3.deserialize(s)
    assert (out["dim"] == dim).all() and out["pool"][0:8].view(np.float64)[0] == 7.0
