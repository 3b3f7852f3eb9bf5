"""bs_oracle_dtype.py — TEST INFRASTRUCTURE ONLY.  Plain, slow numpy/struct definition of wire format v1 for the element
types other than fp64 ("complex128 / fp32 dtypes").

What it follows.  The same passages as bs_oracle.c (PAPER.md L63 meta data, L85 one contiguous stream, L90-92 the
pointer structure first, L106 exact size prediction, L108 identical object back); DMRG scratch data is real fp64 in the
paper's runs, complex for relativistic / complex-hopping Hamiltonians and fp32 in mixed-precision variants, and the
serializer does no arithmetic on the values, so the element type only decides HOW MANY BYTES a block has.
Reading: the header's dtype field selects the element size e —
    0 = f64 (e = 8)   1 = f32 (e = 4)   2 = c64 (e = 8, two f32)   3 = c128 (e = 16, two f64)
and everything else is wire format v1 unchanged:  nbytes_i = e * prod(dim_i);  stored_i = align16(nbytes_i) (so an f32
block carries 0, 4, 8 or 12 zero pad bytes);  offset_i = sum_{j<i} stored_j;  pool slot = align256(nbytes_i).

Written step by step with struct.pack and one Python loop per block — independent of bs_oracle.c (no shared code), so
for dtype 0 the two are a cross-check of each other.  Pins (tests/test_oracle_dtype.py): byte-equality with the
(separately pinned) C oracle for f64; a hand-typed golden f32 stream; c128 payload == the C oracle's f64 payload of the
set with its last extent doubled; c64 stream == the f64 stream but for the dtype word; round trip; fault injection.
Unpinned: nothing.

Round 2, reading D19 (see bs_oracle.c): ``align`` is 16 or 8 — stored_i = align_up(nbytes_i, align) and nothing else
changes.  With align = 8 an f32 block carries 0 or 4 zero pad bytes and every other type none; the payload is then the
plain concatenation of the stored blocks and the stream's total a multiple of 8.  Pins (tests/test_oracle_align8.py):
G7 hand-typed golden stream, byte equality with the C oracle for f64, offsets against numpy.cumsum, round trip.
"""
from __future__ import annotations

import struct

import numpy as np

from .bs_oracle import ERR_ARG, ERR_CORRUPT, ERR_UNSUPPORTED, OracleError

F64, F32, C64, C128 = 0, 1, 2, 3
ELEM_BYTES = {F64: 8, F32: 4, C64: 8, C128: 16}


def _align(x: int, a: int) -> int:
    return (x + a - 1) // a * a


def header_bytes(T: int, B: int) -> int:
    return _align(64 + 32 * T + 48 * B, 128)


def plan(dim, dtype: int, align: int = 16):
    """nbytes, stored, offset per block and the payload size (the "pointer structure", L90-92)."""
    if dtype not in ELEM_BYTES:
        raise OracleError(ERR_UNSUPPORTED, "dtype")
    if align not in (8, 16):
        raise OracleError(ERR_UNSUPPORTED, "align")
    e = ELEM_BYTES[dtype]
    nbytes, stored, offset = [], [], []
    run = 0
    for d in np.asarray(dim, dtype=np.uint64).reshape(-1, 3):
        nb = e * int(d[0]) * int(d[1]) * int(d[2])
        st = _align(nb, align)
        nbytes.append(nb)
        stored.append(st)
        offset.append(run)
        run += st
    return nbytes, stored, offset, run


def serialize(tensors, qn, dim, blocks, dtype: int, align: int = 16) -> np.ndarray:
    """blocks[i] = the raw bytes of block i (any object with the buffer protocol, exactly nbytes_i long)."""
    T, B = len(tensors), len(blocks)
    dim = np.asarray(dim, dtype=np.uint32).reshape(-1, 3)
    qn = np.asarray(qn, dtype=np.int32).reshape(-1, 3, 2)
    nbytes, stored, offset, P = plan(dim, dtype, align)
    first = 0
    for t in tensors:                                    # tensors partition the block table in order
        if int(t["rank"]) not in (2, 3):
            raise OracleError(ERR_UNSUPPORTED, "rank")
        if int(t["first_block"]) != first:
            raise OracleError(ERR_ARG, "partition")
        first += int(t["n_blocks"])
    if first != B or len(dim) != B:
        raise OracleError(ERR_ARG, "partition")
    hb = header_bytes(T, B)
    out = bytearray(hb + P)
    struct.pack_into("<8sIIIIII QQQQ", out, 0, b"BSPARSE1", 1, 0x01020304, dtype, 2, 3, align, T, B, hb, P)
    pos = 64
    for t in tensors:
        out[pos:pos + 32] = np.asarray(t).tobytes()      # tensor records travel byte for byte
        pos += 32
    for k, t in enumerate(tensors):
        for i in range(int(t["first_block"]), int(t["first_block"]) + int(t["n_blocks"])):
            struct.pack_into("<6i3IIQ", out, pos, *[int(x) for x in qn[i].reshape(-1)], *[int(x) for x in dim[i]], k, offset[i])
            pos += 48
    for i in range(B):
        raw = bytes(blocks[i])
        if len(raw) != nbytes[i]:
            raise OracleError(ERR_ARG, "block size")
        out[hb + offset[i]: hb + offset[i] + nbytes[i]] = raw     # the pad up to stored_i stays zero
    return np.frombuffer(bytes(out), np.uint8).copy()


def deserialize(stream) -> dict:
    """Validate in the order of SURVEY §8(c) deserialize(S, n) and rebuild.  Returns tensors (raw 32-byte records), qn,
    dim, dtype, blocks (list of bytes) and the BS_LAYOUT_POOL image (pool, pool_off)."""
    s = bytes(np.ascontiguousarray(stream, dtype=np.uint8))
    n = len(s)
    if n < 64:
        raise OracleError(ERR_CORRUPT, "short")
    magic, ver, endian, dtype, n_qn, max_rank, align, T, B, hb, P = struct.unpack_from("<8sIIIIII QQQQ", s, 0)
    if magic != b"BSPARSE1" or ver != 1 or endian != 0x01020304 or dtype not in ELEM_BYTES or n_qn != 2 or max_rank != 3 \
            or align not in (8, 16) or T >= 1 << 32 or B >= 1 << 32 or hb != header_bytes(T, B) or hb > n or hb + P != n:
        raise OracleError(ERR_CORRUPT, "fixed header")
    e = ELEM_BYTES[dtype]
    recs = []
    first = 0
    for t in range(T):
        rank, fb, nb, dq0, dq1, s0, s1, s2, s3, tag, res = struct.unpack_from("<IIIii4bII", s, 64 + 32 * t)
        if rank not in (2, 3) or fb != first or res != 0:
            raise OracleError(ERR_CORRUPT, "tensor record")
        first += nb
        recs.append((rank, fb, nb))
    if first != B:
        raise OracleError(ERR_CORRUPT, "partition")
    qn = np.zeros((B, 3, 2), np.int32)
    dim = np.zeros((B, 3), np.uint32)
    blocks, pool_off = [], []
    run = cursor = 0
    base = 64 + 32 * T
    for k, (rank, fb, nb) in enumerate(recs):
        for i in range(fb, fb + nb):
            f = struct.unpack_from("<6i3IIQ", s, base + 48 * i)
            q, d, owner, off = f[:6], f[6:9], f[9], f[10]
            nbytes = e * d[0] * d[1] * d[2]
            if owner != k or off != run or (rank == 2 and (d[2] != 1 or q[4] != 0 or q[5] != 0)):
                raise OracleError(ERR_CORRUPT, "block record")
            st = _align(nbytes, align)
            if run + st > P or any(s[hb + run + nbytes: hb + run + st]):
                raise OracleError(ERR_CORRUPT, "pad / range")
            qn[i] = np.array(q, np.int32).reshape(3, 2)
            dim[i] = d
            blocks.append(s[hb + run: hb + run + nbytes])
            pool_off.append(cursor)
            cursor += _align(nbytes, 256)
            run += st
    if run != P or any(s[base + 48 * B: hb]):
        raise OracleError(ERR_CORRUPT, "payload size / slack")
    pool = np.full(max(cursor, 1), 0xEE, np.uint8)
    for b, o in zip(blocks, pool_off):
        pool[o:o + len(b)] = np.frombuffer(b, np.uint8)
    return dict(tensors=s[64:64 + 32 * T], qn=qn, dim=dim, dtype=dtype, align=align, blocks=blocks, pool=pool,
                pool_off=np.array(pool_off, np.uint64), pool_bytes=cursor)
