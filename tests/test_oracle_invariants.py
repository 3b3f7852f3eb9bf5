"""Pins P1-P6, P8-P11 of SURVEY §8(c) for the CPU oracle, plus the boundary conditions of D11.
None of these retype the oracle's loop: each checks against numpy, a struct-based reader, plain memcpy
semantics, or a dense brute-force reconstruction."""
import numpy as np
import pytest

import oracle
import workloads as W
from tests.streamreader import block_doubles, read_stream
from tests.util import host_addrs, oracle_stream


def small_sets():
    yield W.make_config("1")
    yield W.make_set("tiny-ops+site", 11, D=48, S=10, M=2, N0=2, n_ops=20, n_site=2, dims="multinomial")
    yield W.make_set("lognormal", 12, D=200, S=30, M=4, N0=3, n_ops=26, n_site=1, dims="lognormal", sigma=1.0)


def random_dims(rng, B):
    dim = np.ones((B, 3), np.uint32)
    dim[:, 0] = rng.integers(0, 9, B)          # zero extents included (D11)
    dim[:, 1] = rng.integers(1, 12, B)
    dim[:, 2] = rng.integers(1, 4, B)
    return dim


# ---- P2 / P3: sizes and offsets against numpy ------------------------------------------------------
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_P3_offsets_are_exclusive_prefix_sum_numpy(seed):
    rng = np.random.default_rng(seed)
    dim = random_dims(rng, 1000)
    nbytes, stored, offset, P = oracle.plan(dim)
    d = dim.astype(np.uint64)
    nb = 8 * d[:, 0] * d[:, 1] * d[:, 2]
    st = (nb + 15) // 16 * 16
    assert (nbytes == nb).all() and (stored == st).all()
    excl = np.concatenate([[0], np.cumsum(st)[:-1]]).astype(np.uint64)
    assert (offset == excl).all()
    assert P == int(st.sum())
    assert (stored % 16 == 0).all() and ((stored - nbytes) < 16).all()


def test_P3_offsets_in_header_records_config2():
    s = W.make_config("2")
    hdr = oracle.emit_header(s.tensors, s.qn, s.dim)
    fixed, tensors, blocks, slack, _ = read_stream(hdr.tobytes() + b"")
    d = s.dim.astype(np.uint64)
    st = (8 * d[:, 0] * d[:, 1] * d[:, 2] + 15) // 16 * 16
    excl = np.concatenate([[0], np.cumsum(st)[:-1]])
    assert [b["offset"] for b in blocks] == [int(x) for x in excl]
    assert fixed["payload_bytes"] == int(st.sum())
    assert fixed["header_bytes"] == len(hdr) == (64 + 32 * s.n_tensors + 48 * s.n_blocks + 127) // 128 * 128
    assert set(slack) <= {0}
    # owning tensor of every block
    owner = np.repeat(np.arange(s.n_tensors), s.tensors["n_blocks"])
    assert [b["tensor"] for b in blocks] == owner.tolist()


@pytest.mark.parametrize("bset", list(small_sets()), ids=lambda s: s.name)
def test_P2_size_prediction_equals_bytes_written(bset):
    stream, _, _ = oracle_stream(bset)
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    assert len(stream) == total
    assert oracle.stream_info(stream)["header_bytes"] == hb
    assert not (stream == 0xCD).all()
    # every byte of the poisoned output buffer was written: re-serialise into a differently poisoned buffer
    pool, offs = W.fill_pool_host(bset)
    out2 = np.full(total, 0x5A, np.uint8)
    s2 = oracle.serialize(bset.tensors, bset.qn, bset.dim, host_addrs(pool, offs), out=out2, capacity=total)
    assert (s2 == stream).all()


# ---- P1: round trip and fixpoint ---------------------------------------------------------------------
@pytest.mark.parametrize("bset", list(small_sets()), ids=lambda s: s.name)
def test_P1_round_trip_identity_and_fixpoint(bset):
    stream, pool, offs = oracle_stream(bset)
    assert oracle.validate_stream(stream) == oracle.OK
    out = oracle.deserialize(stream)
    assert out["tensors"].tobytes() == bset.tensors.tobytes()
    assert (out["qn"] == bset.qn).all() and (out["dim"] == bset.dim).all()
    src = pool.view(np.uint64)
    base = out["pool"].ctypes.data
    ne = bset.nelems
    for i in range(bset.n_blocks):
        n = int(ne[i])
        o = int(out["addr"][i]) - base
        got = out["pool"][o:o + 8 * n].view(np.uint64)
        so = int(offs[i]) // 8
        assert (got == src[so:so + n]).all()
    # fixpoint: serialize(deserialize(S)) == S byte for byte
    again = oracle.serialize(out["tensors"], out["qn"], out["dim"], out["addr"])
    assert (again == stream).all()


# ---- P4: conservation, read from the stream alone ----------------------------------------------------
@pytest.mark.parametrize("cfg", ["1", "2"])
def test_P4_quantum_number_conservation_from_stream(cfg):
    bset = W.make_config(cfg)
    hdr = oracle.emit_header(bset.tensors, bset.qn, bset.dim)
    _, tensors, blocks, _, _ = read_stream(hdr.tobytes())
    for b in blocks:
        t = tensors[b["tensor"]]
        for c in range(2):
            assert sum(t["sign"][k] * b["qn"][k][c] for k in range(3)) == t["dq"][c]
        for leg in range(t["rank"], 3):
            assert b["dim"][leg] == 1 and b["qn"][leg] == (0, 0)
    assert oracle.validate_set(bset.tensors, bset.qn) == 0
    bad = bset.qn.copy()
    bad[0, 0, 0] += 1
    assert oracle.validate_set(bset.tensors, bad) == 1


def test_D12_duplicate_labels_flagged_by_helper_not_by_serializer():
    bset = W.make_config("1")
    qn = bset.qn.copy()
    qn[1] = qn[0]
    assert oracle.validate_set(bset.tensors, qn) == 2
    pool, offs = W.fill_pool_host(bset)
    oracle.serialize(bset.tensors, qn, bset.dim, host_addrs(pool, offs))    # pure movement: no complaint


# ---- P5: dense brute force ----------------------------------------------------------------------------
def _sector_offsets(dims):
    return np.concatenate([[0], np.cumsum(dims)]).astype(int)


@pytest.mark.parametrize("rule", [(0, 0), (1, 1), (-2, 2), (2, 0)])
def test_P5_dense_reconstruction_rank2(rule):
    rng = np.random.default_rng(5)
    labels = W.label_grid(9, 2, 3)
    dims = (1 + rng.multinomial(40 - 9, np.full(9, 1 / 9))).astype(int)
    D = int(dims.sum())
    so = _sector_offsets(dims)
    idx = {(int(n), int(m)): i for i, (n, m) in enumerate(labels)}
    dense = np.zeros((D, D))
    cut = []
    for l, (n, m) in enumerate(labels):
        r = idx.get((n + rule[0], m + rule[1]))
        if r is None:
            continue
        dense[so[l]:so[l + 1], so[r]:so[r + 1]] = rng.uniform(-1, 1, (dims[l], dims[r]))
        cut.append((l, r))
    assert cut, "rule must select at least one block"
    # cut the blocks out of the dense matrix to form the descriptor
    B = len(cut)
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, B, rule, (-1, 1, 0, 0), 0, 0)
    qn = np.zeros((B, 3, 2), np.int32)
    dim = np.ones((B, 3), np.uint32)
    blocks = []
    for i, (l, r) in enumerate(cut):
        qn[i, 0], qn[i, 1] = labels[l], labels[r]
        dim[i, 0], dim[i, 1] = dims[l], dims[r]
        blocks.append(np.ascontiguousarray(dense[so[l]:so[l + 1], so[r]:so[r + 1]]))
    addr = np.array([b.ctypes.data for b in blocks], np.uint64)
    stream = oracle.serialize(tensors, qn, dim, addr)
    # rebuild the dense matrix from the STREAM ALONE with the independent reader
    _, _, recs, _, payload = read_stream(stream.tobytes())
    rebuilt = np.zeros((D, D))
    for rec in recs:
        l, r = idx[rec["qn"][0]], idx[rec["qn"][1]]
        assert rec["dim"] == (dims[l], dims[r], 1)
        rebuilt[so[l]:so[l + 1], so[r]:so[r + 1]] = np.array(block_doubles(payload, rec)).reshape(dims[l], dims[r])
    assert (rebuilt.view(np.uint64) == dense.view(np.uint64)).all()
    # and through the oracle's own deserializer
    out = oracle.deserialize(stream)
    rebuilt2 = np.zeros((D, D))
    base = out["pool"].ctypes.data
    for i in range(B):
        l, r = idx[tuple(out["qn"][i, 0])], idx[tuple(out["qn"][i, 1])]
        o = int(out["addr"][i]) - base
        n = int(out["dim"][i, 0]) * int(out["dim"][i, 1])
        rebuilt2[so[l]:so[l + 1], so[r]:so[r + 1]] = out["pool"][o:o + 8 * n].view(np.float64).reshape(dims[l], dims[r])
    assert (rebuilt2.view(np.uint64) == dense.view(np.uint64)).all()


def test_P5_dense_reconstruction_rank3():
    rng = np.random.default_rng(6)
    labels = W.label_grid(8, 2, 2)
    dl = (1 + rng.multinomial(24 - 8, np.full(8, 1 / 8))).astype(int)
    dr = (1 + rng.multinomial(28 - 8, np.full(8, 1 / 8))).astype(int)
    sl, sr = _sector_offsets(dl), _sector_offsets(dr)
    idx = {(int(n), int(m)): i for i, (n, m) in enumerate(labels)}
    loc = [(0, 0), (1, 1), (1, -1), (2, 0)]
    dense = np.zeros((dl.sum(), 4, dr.sum()))
    cut = []
    for l, (n, m) in enumerate(labels):
        for s, (qn_, qm_) in enumerate(loc):
            r = idx.get((n + qn_, m + qm_))
            if r is None:
                continue
            dense[sl[l]:sl[l + 1], s, sr[r]:sr[r + 1]] = rng.uniform(-1, 1, (dl[l], dr[r]))
            cut.append((l, s, r))
    B = len(cut)
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (3, 0, B, (0, 0), (1, 1, -1, 0), 0, 0)
    qn = np.zeros((B, 3, 2), np.int32)
    dim = np.ones((B, 3), np.uint32)
    blocks = []
    for i, (l, s, r) in enumerate(cut):
        qn[i, 0], qn[i, 1], qn[i, 2] = labels[l], loc[s], labels[r]
        dim[i] = (dl[l], 1, dr[r])
        blocks.append(np.ascontiguousarray(dense[sl[l]:sl[l + 1], s:s + 1, sr[r]:sr[r + 1]]))
    addr = np.array([b.ctypes.data for b in blocks], np.uint64)
    stream = oracle.serialize(tensors, qn, dim, addr)
    assert oracle.validate_set(tensors, qn) == 0
    _, trecs, recs, _, payload = read_stream(stream.tobytes())
    assert trecs[0]["rank"] == 3
    rebuilt = np.zeros_like(dense)
    for rec in recs:
        l, s, r = idx[rec["qn"][0]], loc.index(rec["qn"][1]), idx[rec["qn"][2]]
        rebuilt[sl[l]:sl[l + 1], s, sr[r]:sr[r + 1]] = np.array(block_doubles(payload, rec)).reshape(dl[l], dr[r])
    assert (rebuilt.view(np.uint64) == dense.view(np.uint64)).all()


# ---- P8: special cases that are plain memcpy ------------------------------------------------------------
def test_P8_single_even_block_payload_is_the_block():
    blk = np.random.default_rng(8).uniform(-1, 1, (6, 7))
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 1, (0, 0), (-1, 1, 0, 0), 0, 0)
    stream = oracle.serialize(tensors, np.zeros((1, 3, 2), np.int32), np.array([[6, 7, 1]], np.uint32),
                              np.array([blk.ctypes.data], np.uint64))
    assert len(stream) == 256 + 6 * 7 * 8            # header 64 + 32 + 48 = 144 -> 256
    assert stream[256:].tobytes() == blk.tobytes()


def test_P8_pool_in_stream_order_payload_is_the_pool():
    rng = np.random.default_rng(9)
    B = 40
    dim = np.ones((B, 3), np.uint32)
    dim[:, 0] = rng.integers(1, 6, B)
    dim[:, 1] = 2 * rng.integers(1, 6, B)          # even element counts: stored == nbytes
    ne = dim[:, 0].astype(int) * dim[:, 1]
    pool = rng.uniform(-1, 1, int(ne.sum()))
    offs = np.concatenate([[0], np.cumsum(ne)[:-1]]) * 8
    tensors = np.zeros(2, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 25, (0, 0), (-1, 1, 0, 0), 0, 0)
    tensors[1] = (2, 25, 15, (0, 0), (-1, 1, 0, 0), 1, 0)
    stream = oracle.serialize(tensors, np.zeros((B, 3, 2), np.int32), dim, host_addrs(pool, offs))
    hb = oracle.header_bytes(2, B)
    assert stream[hb:].tobytes() == pool.tobytes()


# ---- P9: placement invariance -----------------------------------------------------------------------------
def test_P9_stream_does_not_depend_on_where_blocks_live():
    a = W.make_set("pl", 21, D=64, S=10, M=2, N0=2, n_ops=13, n_site=1, dims="multinomial", scatter=True)
    b = W.make_set("pl", 21, D=64, S=10, M=2, N0=2, n_ops=13, n_site=1, dims="multinomial", scatter=False,
                   pool_align=64)
    assert (a.dim == b.dim).all() and not (a.pool_off == b.pool_off).all()
    sa, _, _ = oracle_stream(a)
    sb, _, _ = oracle_stream(b)
    assert (sa == sb).all()
    # compact placement of the same values (the slice-wise mode's layout) as well
    pool, offs = W.fill_pool_host(a, 0, a.n_blocks, compact=True)
    sc = oracle.serialize(a.tensors, a.qn, a.dim, host_addrs(pool, offs))
    assert (sc == sa).all()


# ---- O-5 / P6 on the oracle side: header + tensor-range payloads == the stream ------------------------------
def test_O5_slicewise_emission_concatenates_to_the_stream():
    bset = W.make_set("slices", 31, D=96, S=14, M=4, N0=2, n_ops=30, n_site=2, dims="lognormal", sigma=0.8)
    stream, pool, offs = oracle_stream(bset)
    addr = host_addrs(pool, offs)
    hb, total = oracle.serialized_size(bset.n_tensors, bset.dim)
    parts = [oracle.emit_header(bset.tensors, bset.qn, bset.dim)]
    cuts = [0, 1, 7, 8, 20, bset.n_tensors]
    expect_first = 0
    for t0, t1 in zip(cuts[:-1], cuts[1:]):
        first, chunk = oracle.emit_payload_range(bset.tensors, bset.dim, addr, t0, t1, total)
        assert first == expect_first
        expect_first += len(chunk)
        parts.append(chunk)
    assert (np.concatenate(parts) == stream).all()
    # a slice can be produced from regenerated values of its own blocks only
    t0, t1 = 7, 20
    b0, b1 = int(bset.tensors["first_block"][t0]), int(bset.tensors["first_block"][t1])
    cpool, coffs = W.fill_pool_host(bset, b0, b1, compact=True)
    addr2 = np.zeros(bset.n_blocks, np.uint64)
    addr2[b0:b1] = host_addrs(cpool, coffs)
    first, chunk = oracle.emit_payload_range(bset.tensors, bset.dim, addr2, t0, t1, total)
    assert (chunk == stream[hb + first: hb + first + len(chunk)]).all()


# ---- P10: fault injection ---------------------------------------------------------------------------------
def _mutations(stream, bset):
    T, B = bset.n_tensors, bset.n_blocks
    hb = oracle.header_bytes(T, B)
    t0 = 64
    b0 = 64 + 32 * T
    first_rank2_block = b0                                    # tensor 0 is an operator (rank 2)
    odd = int(np.nonzero(bset.nelems % 2 == 1)[0][0])
    _, _, offset, _ = oracle.plan(bset.dim)
    pad_pos = hb + int(offset[odd]) + int(bset.nelems[odd]) * 8
    slack_pos = 64 + 32 * T + 48 * B
    assert slack_pos < hb, "test set must leave header slack"
    yield "magic", 0, 0x01
    yield "version", 8, 0x02
    yield "endian_tag", 12, 0xFF
    yield "dtype", 16, 0x01
    yield "n_qn", 20, 0x01
    yield "max_rank", 24, 0x01
    yield "align", 28, 0x18
    yield "n_tensors", 32, 0x01
    yield "n_blocks", 40, 0x01
    yield "header_bytes", 48, 0x80
    yield "payload_bytes", 56, 0x10
    yield "tensor.rank", t0 + 0, 0x06
    yield "tensor.first_block", t0 + 32 + 4, 0x01
    yield "tensor.n_blocks", t0 + 8, 0x01
    yield "tensor.reserved", t0 + 28, 0x01
    yield "block.tensor", b0 + 36, 0x01
    yield "block.unused_leg_dim", first_rank2_block + 32, 0x02
    yield "block.unused_leg_qn", first_rank2_block + 16, 0x01
    yield "block.dim(changes size)", b0 + 24, 0x01
    yield "block.offset", b0 + 48 + 40, 0x10
    yield "header slack", slack_pos, 0x01
    yield "pad byte", pad_pos, 0x01


def test_P10_every_validated_field_is_validated():
    bset = W.make_set("fault", 41, D=40, S=9, M=2, N0=3, n_ops=13, n_site=1, dims="multinomial")
    stream, _, _ = oracle_stream(bset)
    assert oracle.validate_stream(stream) == oracle.OK
    for name, pos, xor in _mutations(stream, bset):
        bad = stream.copy()
        bad[pos] ^= xor
        assert oracle.validate_stream(bad) == oracle.ERR_CORRUPT, name
        pool = np.full(oracle.pool_bytes(stream) + 64, 0xEE, np.uint8)
        with pytest.raises(oracle.OracleError) as e:
            oracle.deserialize(bad, pool=pool)
        assert e.value.code == oracle.ERR_CORRUPT, name
        assert (pool == 0xEE).all(), f"{name}: output written despite corrupt header"
    assert oracle.validate_stream(stream[:-1]) == oracle.ERR_CORRUPT
    assert oracle.validate_stream(np.concatenate([stream, np.zeros(16, np.uint8)])) == oracle.ERR_CORRUPT
    assert oracle.validate_stream(stream[:63]) == oracle.ERR_CORRUPT


# ---- P11: special bit patterns ------------------------------------------------------------------------------
def test_P11_special_bit_patterns_survive_bitwise():
    pats = np.array([0x7FF8000000000001, 0xFFF0000000000000, 0x8000000000000000, 0x0000000000000001,
                     0x7FF0000000000000, 0x7FF4DEADBEEF0001, 0x000FFFFFFFFFFFFF], dtype=np.uint64)
    tensors = np.zeros(1, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 1, (0, 0), (-1, 1, 0, 0), 0, 0)
    stream = oracle.serialize(tensors, np.zeros((1, 3, 2), np.int32), np.array([[1, 7, 1]], np.uint32),
                              np.array([pats.ctypes.data], np.uint64))
    assert (stream[256:256 + 56].view(np.uint64) == pats).all()
    assert (stream[256 + 56:] == 0).all() and len(stream) == 256 + 64
    out = oracle.deserialize(stream)
    assert (out["pool"][:56].view(np.uint64) == pats).all()


# ---- D11 boundary conditions / descriptor errors -----------------------------------------------------------
def test_D11_empty_set_is_128_bytes():
    tensors = np.zeros(0, dtype=W.TENSOR_REC_DTYPE)
    s = oracle.serialize(tensors, np.zeros((0, 3, 2), np.int32), np.zeros((0, 3), np.uint32), np.zeros(0, np.uint64))
    assert len(s) == 128 and (s[64:] == 0).all()
    info = oracle.stream_info(s)
    assert info == dict(n_tensors=0, n_blocks=0, header_bytes=128, payload_bytes=0, align=16)
    out = oracle.deserialize(s)
    assert len(out["tensors"]) == 0 and out["dim"].shape == (0, 3)


def test_D11_zero_extent_blocks_and_empty_tensors_round_trip():
    tensors = np.zeros(3, dtype=W.TENSOR_REC_DTYPE)
    tensors[0] = (2, 0, 2, (0, 0), (-1, 1, 0, 0), 0, 0)
    tensors[1] = (3, 2, 0, (0, 0), (1, 1, -1, 0), 1, 0)          # empty tensor
    tensors[2] = (2, 2, 2, (0, 0), (-1, 1, 0, 0), 2, 0)
    dim = np.array([[0, 5, 1], [3, 1, 1], [2, 0, 1], [1, 1, 1]], np.uint32)
    data = [np.zeros(0), np.array([1., 2., 3.]), np.zeros(0), np.array([4.])]
    addr = np.array([d.ctypes.data for d in data], np.uint64)
    s = oracle.serialize(tensors, np.zeros((4, 3, 2), np.int32), dim, addr)
    _, _, recs, _, payload = read_stream(s.tobytes())
    assert [r["offset"] for r in recs] == [0, 0, 32, 32]          # zero-size block shares the next one's offset
    assert len(payload) == 48
    out = oracle.deserialize(s)
    assert (out["dim"] == dim).all() and out["tensors"].tobytes() == tensors.tobytes()
    again = oracle.serialize(out["tensors"], out["qn"], out["dim"], out["addr"])
    assert (again == s).all()


def test_descriptor_errors():
    bset = W.make_config("1")
    pool, offs = W.fill_pool_host(bset)
    addr = host_addrs(pool, offs)
    t = bset.tensors.copy()
    t["n_blocks"][0] -= 1
    with pytest.raises(oracle.OracleError) as e:
        oracle.serialize(t, bset.qn, bset.dim, addr)
    assert e.value.code == oracle.ERR_ARG
    t = bset.tensors.copy()
    t["rank"][0] = 4
    with pytest.raises(oracle.OracleError) as e:
        oracle.serialize(t, bset.qn, bset.dim, addr)
    assert e.value.code == oracle.ERR_UNSUPPORTED
    hb, total = oracle.serialized_size(1, bset.dim)
    with pytest.raises(oracle.OracleError) as e:
        oracle.serialize(bset.tensors, bset.qn, bset.dim, addr, capacity=total - 1)
    assert e.value.code == oracle.ERR_CAPACITY and e.value.required == total


def test_scatter_mode_places_blocks_at_caller_addresses():
    bset = W.make_set("scat", 51, D=30, S=8, M=2, N0=3, n_ops=5, n_site=0, dims="multinomial")
    stream, pool, offs = oracle_stream(bset)
    dst = np.full(pool.nbytes, 0xEE, np.uint8)
    addr = (np.uint64(dst.ctypes.data) + offs).astype(np.uint64)
    out = oracle.deserialize(stream, scatter_addr=addr, scatter_dim=bset.dim)
    assert (out["addr"] == addr).all()
    ne = bset.nelems
    for i in range(bset.n_blocks):
        o, n = int(offs[i]), int(ne[i]) * 8
        assert dst[o:o + n].tobytes() == pool.view(np.uint8)[o:o + n].tobytes()
    wrong = bset.dim.copy()
    wrong[0, 0] += 1
    with pytest.raises(oracle.OracleError) as e:
        oracle.deserialize(stream, scatter_addr=addr, scatter_dim=wrong)
    assert e.value.code == oracle.ERR_ARG
