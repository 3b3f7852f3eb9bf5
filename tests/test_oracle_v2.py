"""Pins of the v2 oracle (oracle/bs_oracle_v2.c — wire format v2, structure-shared layers).
None of them retypes the oracle's loops: hand-typed golden bytes, an independent struct reader, numpy.cumsum,
the (separately pinned) v1 oracle on the expanded set, plain memcpy semantics, dense brute force."""
import os

import numpy as np
import pytest

import oracle
import workloads as W
from oracle import v2
from tests.streamreader import read_stream, read_stream_v2
from tests.util import host_addrs, read_hex_fixture, sha256

GOLD = os.path.join(os.path.dirname(__file__), "golden", "g2_golden_stream_v2.hex")
GOLD_SHA = "133e52ad8884ebe1535ea9429e6cb5e257da97c5487132f84bd0bb671437e222"


def golden_set():
    structs = np.zeros(1, dtype=W.STRUCT_REC_DTYPE)
    structs[0] = (2, 0, 2, (1, 1), (-1, 1, 0, 0), 0)
    layers = np.zeros(2, dtype=W.LAYER_REC_DTYPE)
    layers[0] = (0, 7, 0)
    layers[1] = (0, 9, 0)
    qn = np.array([[[0, 0], [1, 1], [0, 0]], [[1, -1], [2, 0], [0, 0]]], dtype=np.int32)
    dim = np.array([[1, 1, 1], [1, 2, 1]], dtype=np.uint32)
    blocks = [np.array([1.0]), np.array([2.0, 3.0]), np.array([4.0]), np.array([5.0, 6.0])]
    return structs, layers, qn, dim, blocks


def small_sets():
    yield W.make_config("1")
    yield W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    yield W.make_set("lognormal", 12, D=200, S=30, M=4, N0=3, n_ops=40, n_site=1, dims="lognormal", sigma=1.0)
    yield W.make_set("few-ops", 13, D=64, S=12, M=2, N0=2, n_ops=5, n_site=1, dims="multinomial")


def v2_stream(bset, keep_unused=False, pool=None, offs=None):
    lv = W.layered_view(bset, keep_unused=keep_unused)
    if pool is None:
        pool, offs = W.fill_pool_host(bset)
    s = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs))
    return s, lv, pool, offs


# ---- G2: golden bytes + independent reader -------------------------------------------------------------------------
def test_fixture_is_the_cited_one():
    raw = read_hex_fixture(GOLD)
    assert len(raw) == 320 and sha256(raw) == GOLD_SHA


def test_oracle_reproduces_golden_bytes():
    structs, layers, qn, dim, blocks = golden_set()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = v2.serialize(structs, layers, qn, dim, addr)
    assert bytes(s) == read_hex_fixture(GOLD)
    assert v2.serialized_size(structs, layers, dim) == (256, 320)
    assert v2.header_bytes(1, 2, 2) == 256


def test_independent_reader_sees_the_stated_fields():
    fixed, structs, layers, blocks, slack, payload = read_stream_v2(read_hex_fixture(GOLD))
    assert fixed == dict(magic=b"BSPARSE1", version=2, endian_tag=0x01020304, dtype=0, n_qn=2, max_rank=3, align=16,
                         n_structs=1, n_struct_blocks=2, n_layers=2, header_bytes=256, payload_bytes=64)
    assert structs == [dict(rank=2, first_block=0, n_blocks=2, dq=(1, 1), sign=(-1, 1, 0, 0), layer_bytes=32)]
    assert layers == [dict(structure=0, tag=7, offset=0), dict(structure=0, tag=9, offset=32)]
    assert blocks == [dict(qn=((0, 0), (1, 1), (0, 0)), dim=(1, 1, 1), structure=0, offset=0),
                      dict(qn=((1, -1), (2, 0), (0, 0)), dim=(1, 2, 1), structure=0, offset=16)]
    assert slack == bytes(32)
    assert np.frombuffer(payload, np.float64).tolist() == [1.0, 0.0, 2.0, 3.0, 4.0, 0.0, 5.0, 6.0]
    assert payload[8:16] == bytes(8) and payload[40:48] == bytes(8)


def test_oracle_deserializes_golden():
    raw = np.frombuffer(read_hex_fixture(GOLD), dtype=np.uint8)
    assert v2.validate_stream(raw) == oracle.OK
    out = v2.deserialize(raw)
    structs, layers, qn, dim, _ = golden_set()
    assert out["structs"]["layer_bytes"].tolist() == [32] and out["layers"]["offset"].tolist() == [0, 32]
    assert out["layers"]["tag"].tolist() == [7, 9]
    assert (out["qn"] == qn).all() and (out["dim"] == dim).all()
    base = out["pool"].ctypes.data
    assert [int(a) - base for a in out["addr"]] == [0, 256, 512, 768]
    assert out["pool"][0:8].view(np.float64)[0] == 1.0
    assert tuple(out["pool"][768:784].view(np.float64)) == (5.0, 6.0)
    assert (out["pool"][8:256] == 0xEE).all()


# ---- the v1 relation: same payload as the expanded set; smaller header --------------------------------------------------
@pytest.mark.parametrize("bset", list(small_sets()), ids=lambda s: s.name)
def test_payload_equals_v1_payload_of_the_expanded_set(bset):
    s2, lv, pool, offs = v2_stream(bset)
    s1 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs))
    i1, i2 = oracle.stream_info(s1), v2.stream_info(s2)
    assert i1["payload_bytes"] == i2["payload_bytes"]
    assert (s1[i1["header_bytes"]:] == s2[i2["header_bytes"]:]).all()
    # block offsets: v1 absolute offset == v2 layer offset + relative offset
    _, _, blocks1, _, _ = read_stream(s1.tobytes())
    _, structs, layers, blocks2, _, _ = read_stream_v2(s2.tobytes())
    a = 0
    for ly in layers:
        st = structs[ly["structure"]]
        for j in range(st["first_block"], st["first_block"] + st["n_blocks"]):
            assert blocks1[a]["offset"] == ly["offset"] + blocks2[j]["offset"]
            assert blocks1[a]["qn"] == blocks2[j]["qn"] and blocks1[a]["dim"] == blocks2[j]["dim"]
            a += 1
    assert a == bset.n_blocks
    if bset.n_tensors > len(structs):
        assert i2["header_bytes"] < i1["header_bytes"]


def test_header_shrinks_by_the_sharing_factor_config2():
    bset = W.make_config("2")
    lv = W.layered_view(bset)
    hb2, _ = v2.serialized_size(lv["structs"], lv["layers"], lv["dim"])
    hb1 = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
    assert hb2 == (64 + 32 * len(lv["structs"]) + 16 * bset.n_tensors + 48 * lv["dim"].shape[0] + 127) // 128 * 128
    assert hb1 > 8 * hb2            # 256 operators share 13 structures


# ---- offsets against numpy ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_offsets_are_prefix_sums_numpy(seed):
    rng = np.random.default_rng(seed)
    C = 7
    nb = rng.integers(0, 9, C)                       # structures with zero blocks included
    Bs = int(nb.sum())
    structs = np.zeros(C, dtype=W.STRUCT_REC_DTYPE)
    structs["rank"] = 3
    structs["n_blocks"] = nb
    structs["first_block"] = np.concatenate([[0], np.cumsum(nb)])[:-1]
    T = 40
    layers = np.zeros(T, dtype=W.LAYER_REC_DTYPE)
    layers["structure"] = rng.integers(0, C, T)
    dim = np.ones((Bs, 3), np.uint32)
    dim[:, 0] = rng.integers(0, 9, Bs)               # zero extents included
    dim[:, 1] = rng.integers(1, 12, Bs)
    dim[:, 2] = rng.integers(1, 4, Bs)
    p = v2.plan(structs, layers, dim)
    d = dim.astype(np.uint64)
    st = (8 * d[:, 0] * d[:, 1] * d[:, 2] + 15) // 16 * 16
    owner = np.repeat(np.arange(C), nb)
    glob = np.concatenate([[0], np.cumsum(st)])
    rel = glob[:-1] - glob[structs["first_block"][owner]] if Bs else np.zeros(0)
    assert (p["rel_offset"] == rel).all()
    lb = np.array([int(st[owner == s].sum()) for s in range(C)], dtype=np.uint64)
    assert (p["layer_bytes"] == lb).all()
    lo = np.concatenate([[0], np.cumsum(lb[layers["structure"]])])
    assert (p["layer_offset"] == lo[:-1]).all() and p["payload_bytes"] == int(lo[-1])
    assert p["n_addr"] == int(nb[layers["structure"]].sum())


# ---- size prediction, round trip, fixpoint ------------------------------------------------------------------------------------
@pytest.mark.parametrize("keep_unused", [False, True])
@pytest.mark.parametrize("bset", list(small_sets()), ids=lambda s: s.name)
def test_size_prediction_round_trip_and_fixpoint(bset, keep_unused):
    s, lv, pool, offs = v2_stream(bset, keep_unused)
    hb, total = v2.serialized_size(lv["structs"], lv["layers"], lv["dim"])
    assert len(s) == total and v2.stream_info(s)["header_bytes"] == hb
    assert v2.validate_stream(s) == oracle.OK
    out = v2.deserialize(s)
    for f in ("rank", "first_block", "n_blocks", "dq", "sign"):
        assert (out["structs"][f] == lv["structs"][f]).all()
    assert (out["layers"]["structure"] == lv["layers"]["structure"]).all()
    assert (out["layers"]["tag"] == lv["layers"]["tag"]).all()
    assert (out["qn"] == lv["qn"]).all() and (out["dim"] == lv["dim"]).all()
    assert len(out["addr"]) == bset.n_blocks
    src = pool.view(np.uint64)
    base = out["pool"].ctypes.data
    ne = bset.nelems
    for i in range(bset.n_blocks):
        n, o, so = int(ne[i]), int(out["addr"][i]) - base, int(offs[i]) // 8
        assert (out["pool"][o:o + 8 * n].view(np.uint64) == src[so:so + n]).all()
    again = v2.serialize(out["structs"], out["layers"], out["qn"], out["dim"], out["addr"])
    assert (again == s).all()
    # every byte of the output buffer is written
    out2 = np.full(total, 0x5A, np.uint8)
    s2 = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), out=out2, capacity=total)
    assert (s2 == s).all()


def test_scatter_mode_and_capacity():
    bset = W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    s, lv, pool, offs = v2_stream(bset)
    dst = np.full(pool.size * 8, 0x11, np.uint8)
    out = v2.deserialize(s, scatter_addr=host_addrs(dst, offs), scatter_dim=lv["dim"])
    assert (out["addr"] == host_addrs(dst, offs)).all()
    src8 = pool.view(np.uint8)
    ne = bset.nelems
    for i in range(bset.n_blocks):
        o, n = int(offs[i]), 8 * int(ne[i])
        assert (dst[o:o + n] == src8[o:o + n]).all()
    bad = lv["dim"].copy()
    bad[0, 0] += 1
    with pytest.raises(oracle.OracleError) as e:
        v2.deserialize(s, scatter_addr=host_addrs(dst, offs), scatter_dim=bad)
    assert e.value.code == oracle.ERR_ARG
    with pytest.raises(oracle.OracleError) as e:
        v2.deserialize(s, pool=np.zeros(16, np.uint8))
    assert e.value.code == oracle.ERR_CAPACITY
    with pytest.raises(oracle.OracleError) as e:
        v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), capacity=len(s) - 16)
    assert e.value.code == oracle.ERR_CAPACITY and e.value.required == len(s)


def test_empty_sets():
    structs = np.zeros(0, dtype=W.STRUCT_REC_DTYPE)
    layers = np.zeros(0, dtype=W.LAYER_REC_DTYPE)
    s = v2.serialize(structs, layers, np.zeros((0, 3, 2), np.int32), np.zeros((0, 3), np.uint32), np.zeros(0, np.uint64))
    assert len(s) == 128 and v2.validate_stream(s) == 0
    # structures without layers, and a layer of a structure without blocks
    structs = np.zeros(2, dtype=W.STRUCT_REC_DTYPE)
    structs["rank"] = 2
    structs["n_blocks"] = (0, 1)
    structs["first_block"] = (0, 0)
    layers = np.zeros(1, dtype=W.LAYER_REC_DTYPE)
    dim = np.array([[2, 3, 1]], np.uint32)
    s = v2.serialize(structs, layers, np.zeros((1, 3, 2), np.int32), dim, np.zeros(0, np.uint64))
    assert v2.validate_stream(s) == 0 and v2.stream_info(s)["payload_bytes"] == 0
    assert v2.counts(s) == (0, 0)


# ---- conservation, read from the stream alone -----------------------------------------------------------------------------------
def test_quantum_number_conservation_from_stream():
    s, lv, _, _ = v2_stream(W.make_config("2"))
    _, structs, layers, blocks, _, _ = read_stream_v2(s.tobytes())
    for b in blocks:
        st = structs[b["structure"]]
        for c in range(2):
            assert sum(st["sign"][k] * b["qn"][k][c] for k in range(3)) == st["dq"][c]
        for leg in range(st["rank"], 3):
            assert b["dim"][leg] == 1 and b["qn"][leg] == (0, 0)


# ---- dense brute force, layer by layer ---------------------------------------------------------------------------------------------
def test_dense_reconstruction_of_every_layer():
    rng = np.random.default_rng(7)
    labels = W.label_grid(9, 2, 3)
    dims = (1 + rng.multinomial(40 - 9, np.full(9, 1 / 9))).astype(int)
    D = int(dims.sum())
    so = np.concatenate([[0], np.cumsum(dims)]).astype(int)
    idx = {(int(n), int(m)): i for i, (n, m) in enumerate(labels)}
    rules = [(1, 1), (0, 0)]
    structs = np.zeros(2, dtype=W.STRUCT_REC_DTYPE)
    qn_l, dim_l, cuts = [], [], []
    for s, rule in enumerate(rules):
        pairs = [(l, idx[(n + rule[0], m + rule[1])]) for l, (n, m) in enumerate(labels) if (n + rule[0], m + rule[1]) in idx]
        structs[s] = (2, len(qn_l), len(pairs), rule, (-1, 1, 0, 0), 0)
        for l, r in pairs:
            qn_l.append([labels[l], labels[r], (0, 0)])
            dim_l.append([dims[l], dims[r], 1])
        cuts.append(pairs)
    layer_struct = [0, 1, 0, 0, 1]
    layers = np.zeros(len(layer_struct), dtype=W.LAYER_REC_DTYPE)
    layers["structure"] = layer_struct
    layers["tag"] = np.arange(len(layer_struct)) + 100
    dense, blocks = [], []
    for t, s in enumerate(layer_struct):                        # the dense matrix comes FIRST; blocks are cut out of it
        mat = np.zeros((D, D))
        for l, r in cuts[s]:
            mat[so[l]:so[l + 1], so[r]:so[r + 1]] = rng.uniform(-1, 1, (dims[l], dims[r]))
        dense.append(mat)
        for l, r in cuts[s]:
            blocks.append(np.ascontiguousarray(mat[so[l]:so[l + 1], so[r]:so[r + 1]]))
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    stream = v2.serialize(structs, layers, np.array(qn_l, np.int32), np.array(dim_l, np.uint32), addr)
    fixed, rs, rl, rb, _, payload = read_stream_v2(stream.tobytes())
    for t, ly in enumerate(rl):                                 # rebuild every layer from the stream alone
        st = rs[ly["structure"]]
        mat = np.zeros((D, D))
        for b in rb[st["first_block"]:st["first_block"] + st["n_blocks"]]:
            l, r = idx[b["qn"][0]], idx[b["qn"][1]]
            n = b["dim"][0] * b["dim"][1]
            vals = np.frombuffer(payload, np.float64, n, ly["offset"] + b["offset"]).reshape(b["dim"][0], b["dim"][1])
            mat[so[l]:so[l + 1], so[r]:so[r + 1]] = vals
        assert (mat.view(np.uint64) == dense[t].view(np.uint64)).all()


# ---- fault injection: every validated field ------------------------------------------------------------------------------------------
def _mutations(s):
    fixed, structs, layers, blocks, _, _ = read_stream_v2(s.tobytes())
    C, T, Bs = fixed["n_structs"], fixed["n_layers"], fixed["n_struct_blocks"]
    srec, lrec = 64, 64 + 32 * C
    brec = lrec + 16 * T
    used = brec + 48 * Bs
    m = [("magic", 0), ("version", 8), ("endian_tag", 12), ("dtype", 16), ("n_qn", 20), ("max_rank", 24), ("align", 28),
         ("n_structs", 32), ("n_struct_blocks", 36), ("n_layers", 40), ("header_bytes", 48), ("payload_bytes", 56),
         ("struct rank", srec), ("struct first_block", srec + 32 + 4), ("struct n_blocks", srec + 8),
         ("struct layer_bytes", srec + 24), ("layer structure", lrec + 16), ("layer offset", lrec + 16 + 8),
         ("block owner", brec + 36), ("block offset", brec + 48 + 40), ("block dim", brec + 24)]
    if used < fixed["header_bytes"]:
        m.append(("header slack", used))
    # an unused leg of a rank-2 block; a pad byte of an odd-sized block
    for j, b in enumerate(blocks):
        if structs[b["structure"]]["rank"] == 2:
            m.append(("unused leg label", brec + 48 * j + 16))
            m.append(("unused leg dim", brec + 48 * j + 32))
            break
    for ly in layers:
        st = structs[ly["structure"]]
        hit = False
        for b in blocks[st["first_block"]:st["first_block"] + st["n_blocks"]]:
            n = b["dim"][0] * b["dim"][1] * b["dim"][2]
            if n % 2:
                m.append(("pad byte", fixed["header_bytes"] + ly["offset"] + b["offset"] + 8 * n + 3))
                hit = True
                break
        if hit:
            break
    return m


def test_fault_injection_every_validated_field():
    bset = W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    s, _, _, _ = v2_stream(bset)
    assert v2.validate_stream(s) == 0
    muts = _mutations(s)
    assert len(muts) >= 24 and any(k == "pad byte" for k, _ in muts)
    for what, pos in muts:
        bad = s.copy()
        bad[pos] ^= 0x04 if what == "struct rank" else 0x01      # rank 2 -> 3 would still be a valid record
        assert v2.validate_stream(bad) == oracle.ERR_CORRUPT, what
        with pytest.raises(oracle.OracleError):
            v2.deserialize(bad)
    assert v2.validate_stream(s[:-16]) == oracle.ERR_CORRUPT
    assert v2.validate_stream(s[:40]) == oracle.ERR_CORRUPT
    # a v1 stream is not a v2 stream and vice versa
    pool, offs = W.fill_pool_host(bset)
    s1 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs))
    assert v2.validate_stream(s1) == oracle.ERR_CORRUPT and oracle.validate_stream(s) == oracle.ERR_CORRUPT


def test_bad_descriptors():
    structs, layers, qn, dim, blocks = golden_set()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    bad = layers.copy()
    bad["structure"][1] = 1
    with pytest.raises(oracle.OracleError) as e:
        v2.serialize(structs, bad, qn, dim, addr)
    assert e.value.code == oracle.ERR_ARG
    bad = structs.copy()
    bad["first_block"][0] = 1
    with pytest.raises(oracle.OracleError) as e:
        v2.serialize(bad, layers, qn, dim, addr)
    assert e.value.code == oracle.ERR_ARG
    bad = structs.copy()
    bad["rank"][0] = 4
    with pytest.raises(oracle.OracleError) as e:
        v2.serialize(bad, layers, qn, dim, addr)
    assert e.value.code == oracle.ERR_UNSUPPORTED


def test_special_bit_patterns_survive():
    structs, layers, qn, dim, _ = golden_set()
    pats = np.array([0x7FF8000000000123, 0x8000000000000000, 0x0000000000000001, 0xFFF0000000000000,
                     0x7FF0000000000000, 0xFFFFFFFFFFFFFFFF], dtype=np.uint64)
    blocks = [pats[0:1].copy(), pats[1:3].copy(), pats[3:4].copy(), pats[4:6].copy()]
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = v2.serialize(structs, layers, qn, dim, addr)
    out = v2.deserialize(s)
    base = out["pool"].ctypes.data
    got = np.concatenate([out["pool"][int(a) - base:int(a) - base + 8 * b.size].view(np.uint64)
                          for a, b in zip(out["addr"], blocks)])
    assert (got == pats).all()


# ---- element types of layered sets (reading E-2) ------------------------------------------
GOLD_F32 = os.path.join(os.path.dirname(__file__), "golden", "g6_golden_stream_v2_f32.hex")
GOLD_F32_SHA = "0b65fe5af21ebb09c2cd433fcad8b1c8621473af4220079b9e0789b1cb581921"
ELEM = {0: 8, 1: 4, 2: 8, 3: 16}


def golden_set_f32():
    structs = np.zeros(1, dtype=W.STRUCT_REC_DTYPE)
    structs[0] = (2, 0, 2, (0, 0), (-1, 1, 0, 0), 0)
    layers = np.zeros(2, dtype=W.LAYER_REC_DTYPE)
    layers[0] = (0, 9, 0)
    layers[1] = (0, 11, 0)
    qn = np.array([[[0, 0], [0, 0], [0, 0]], [[1, 1], [1, 1], [0, 0]]], dtype=np.int32)
    dim = np.array([[1, 3, 1], [1, 1, 1]], dtype=np.uint32)
    blocks = [np.array([1, 2, 3], np.float32), np.array([-1], np.float32), np.array([4, 5, 6], np.float32),
              np.array([-2], np.float32)]
    return structs, layers, qn, dim, blocks


def test_G6_f32_fixture_and_oracle_reproduces_it():
    raw = read_hex_fixture(GOLD_F32)
    assert len(raw) == 320 and sha256(raw) == GOLD_F32_SHA
    structs, layers, qn, dim, blocks = golden_set_f32()
    addr = np.array([b.ctypes.data for b in blocks], dtype=np.uint64)
    s = v2.serialize(structs, layers, qn, dim, addr, dtype=1)
    assert bytes(s) == raw
    assert v2.serialized_size(structs, layers, dim, dtype=1) == (256, 320)
    # the independent struct reader sees the stated fields
    fixed, st, ly, bl, slack, payload = read_stream_v2(raw)
    assert fixed["dtype"] == 1 and fixed["payload_bytes"] == 64
    assert st[0]["layer_bytes"] == 32 and [l["offset"] for l in ly] == [0, 32] and [b["offset"] for b in bl] == [0, 16]
    assert np.frombuffer(payload, np.float32).tolist() == [1, 2, 3, 0, -1, 0, 0, 0, 4, 5, 6, 0, -2, 0, 0, 0]
    # and back: pool slots are align256(nbytes), the bytes behind a block keep their poison
    arr = np.frombuffer(raw, np.uint8)
    assert v2.validate_stream(arr) == oracle.OK and v2.stream_info(arr)["dtype"] == 1
    out = v2.deserialize(arr)
    base = out["pool"].ctypes.data
    assert [int(a) - base for a in out["addr"]] == [0, 256, 512, 768] and v2.counts(arr) == (4, 1024)
    assert out["pool"][0:12].view(np.float32).tolist() == [1, 2, 3] and out["pool"][768:772].view(np.float32)[0] == -2
    assert (out["pool"][12:256] == 0xEE).all() and (out["pool"][772:1024] == 0xEE).all()


def _typed_blocks(bset, pool, offs, e):
    """Block i read as e-byte elements: the first e*n bytes of its fp64 storage (c128: the set's storage is too short, so the
    values are taken from a pool of twice the size built by the caller)."""
    raw = pool.view(np.uint8)
    return [raw[int(o): int(o) + e * int(n)] for o, n in zip(offs, bset.nelems)]


@pytest.mark.parametrize("dtype", [0, 1, 2, 3])
@pytest.mark.parametrize("bset", list(small_sets()), ids=lambda s: s.name)
def test_typed_payload_equals_the_independent_v1_dtype_oracle(bset, dtype):
    """The v2 payload of a typed layered set == the payload of the (independently written, separately pinned) numpy oracle
    of wire format v1 for the same element type on the expanded set; offsets against numpy.cumsum of e-sized blocks."""
    from oracle import dt
    e = ELEM[dtype]
    pool, offs = W.fill_pool_host(bset)
    if e == 16:    # room for 16-byte elements: every block twice as long, same seeded values twice
        big = np.zeros(2 * pool.size + 2, np.float64)
        offs = offs * 2
        for o, n in zip(offs, bset.nelems):
            src = pool[int(o) // 16: int(o) // 16 + int(n)]
            big[int(o) // 8: int(o) // 8 + 2 * int(n)] = np.repeat(src, 2)
        pool = big
    lv = W.layered_view(bset)
    s2 = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), dtype=dtype)
    s1 = dt.serialize(bset.tensors, bset.qn, bset.dim, _typed_blocks(bset, pool, offs, e), dtype)
    i2 = v2.stream_info(s2)
    hb1 = dt.header_bytes(bset.n_tensors, bset.n_blocks)
    assert i2["dtype"] == dtype and i2["payload_bytes"] == len(s1) - hb1
    assert (s2[i2["header_bytes"]:] == s1[hb1:]).all()
    # offsets: numpy.cumsum over align16(e * n), per structure and per layer
    plan = v2.plan(lv["structs"], lv["layers"], lv["dim"], dtype)
    d = lv["dim"].astype(np.uint64)
    st = (np.uint64(e) * d[:, 0] * d[:, 1] * d[:, 2] + np.uint64(15)) // np.uint64(16) * np.uint64(16)
    for k, srec in enumerate(lv["structs"]):
        f, n = int(srec["first_block"]), int(srec["n_blocks"])
        want = np.concatenate([[0], np.cumsum(st[f:f + n])])
        assert plan["rel_offset"][f:f + n].tolist() == want[:-1].tolist() and int(plan["layer_bytes"][k]) == int(want[-1])
    lb = plan["layer_bytes"][lv["layers"]["structure"]]
    assert plan["layer_offset"].tolist() == np.concatenate([[0], np.cumsum(lb)])[:-1].tolist()
    assert v2.serialized_size(lv["structs"], lv["layers"], lv["dim"], dtype)[1] == len(s2)
    # round trip, fixpoint, pool layout (slots of align256(e * n), untouched bytes keep their poison)
    out = v2.deserialize(s2)
    base = out["pool"].ctypes.data
    slots = (np.uint64(e) * bset.nelems + np.uint64(255)) // np.uint64(256) * np.uint64(256)
    assert (out["addr"] - np.uint64(base)).tolist() == np.concatenate([[0], np.cumsum(slots)])[:-1].tolist()
    for a, blk, sl in zip(out["addr"], _typed_blocks(bset, pool, offs, e), slots):
        o = int(a) - base
        assert (out["pool"][o: o + len(blk)] == blk).all() and (out["pool"][o + len(blk): o + int(sl)] == 0xEE).all()
    again = v2.serialize(out["structs"], out["layers"], out["qn"], out["dim"], out["addr"], dtype=dtype)
    assert (again == s2).all()


def test_c64_stream_is_the_f64_stream_but_for_the_dtype_word_and_bad_types_are_refused():
    bset = W.make_set("few-ops", 13, D=64, S=12, M=2, N0=2, n_ops=5, n_site=1, dims="multinomial")
    pool, offs = W.fill_pool_host(bset)
    lv = W.layered_view(bset)
    a = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), dtype=0)
    b = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), dtype=2)
    assert a[16] == 0 and b[16] == 2
    b2 = b.copy()
    b2[16] = 0
    assert (a == b2).all()
    with pytest.raises(oracle.OracleError) as e:
        v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), dtype=4)
    assert e.value.code == oracle.ERR_UNSUPPORTED
    bad = a.copy()
    bad[16] = 4
    assert v2.validate_stream(bad) == oracle.ERR_CORRUPT
    # an f32 stream: every pad length occurs and a non-zero pad byte of each is refused
    f = v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], host_addrs(pool, offs), dtype=1)
    info = v2.stream_info(f)
    plan = v2.plan(lv["structs"], lv["layers"], lv["dim"], 1)
    seen = set()
    for k, srec in enumerate(lv["structs"]):
        layer0 = int(np.nonzero(lv["layers"]["structure"] == k)[0][0])
        for j in range(int(srec["first_block"]), int(srec["first_block"]) + int(srec["n_blocks"])):
            nb = 4 * int(np.prod(lv["dim"][j].astype(np.int64)))
            pad = -nb % 16
            if pad and pad not in seen:
                seen.add(pad)
                bad = f.copy()
                bad[info["header_bytes"] + int(plan["layer_offset"][layer0]) + int(plan["rel_offset"][j]) + nb] = 1
                assert v2.validate_stream(bad) == oracle.ERR_CORRUPT
    assert seen == {4, 8, 12}
