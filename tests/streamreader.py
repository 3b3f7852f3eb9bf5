"""Independent reader of wire format v1 written with Python ``struct`` only ("a cheap second
opinion on the oracle").  It re-types the field list of DESIGN.md "Wire format v1" and shares nothing with
oracle/ or the CUDA path.  Used by the -m "not gpu" pins and by the GPU parity tests as a cross-check."""
import struct


def read_stream(buf: bytes):
    buf = bytes(buf)
    magic, version, endian, dtype, n_qn, max_rank, align, T, B, hb, P = struct.unpack_from("<8sIIIIIIQQQQ", buf, 0)
    fixed = dict(magic=magic, version=version, endian_tag=endian, dtype=dtype, n_qn=n_qn, max_rank=max_rank,
                 align=align, n_tensors=T, n_blocks=B, header_bytes=hb, payload_bytes=P)
    tensors = []
    pos = 64
    for _ in range(T):
        rank, first, nb, dq0, dq1, s0, s1, s2, s3, tag, reserved = struct.unpack_from("<IIIiibbbbII", buf, pos)
        tensors.append(dict(rank=rank, first_block=first, n_blocks=nb, dq=(dq0, dq1), sign=(s0, s1, s2, s3), tag=tag,
                            reserved=reserved))
        pos += 32
    blocks = []
    for _ in range(B):
        q = struct.unpack_from("<6i", buf, pos)
        d0, d1, d2, tensor, offset = struct.unpack_from("<IIIIQ", buf, pos + 24)
        blocks.append(dict(qn=((q[0], q[1]), (q[2], q[3]), (q[4], q[5])), dim=(d0, d1, d2), tensor=tensor, offset=offset))
        pos += 48
    slack = buf[pos:hb]
    payload = buf[hb:hb + P]
    return fixed, tensors, blocks, slack, payload


def block_doubles(payload: bytes, blk):
    n = blk["dim"][0] * blk["dim"][1] * blk["dim"][2]
    return struct.unpack_from(f"<{n}d", payload, blk["offset"])


def read_stream_v2(buf: bytes):
    """Wire format v2 (structure-shared layers), field list re-typed with ``struct``."""
    buf = bytes(buf)
    magic, version, endian, dtype, n_qn, max_rank, align, C, Bs, T, hb, P = struct.unpack_from("<8sIIIIIIIIQQQ", buf, 0)
    fixed = dict(magic=magic, version=version, endian_tag=endian, dtype=dtype, n_qn=n_qn, max_rank=max_rank, align=align,
                 n_structs=C, n_struct_blocks=Bs, n_layers=T, header_bytes=hb, payload_bytes=P)
    pos = 64
    structs = []
    for _ in range(C):
        rank, first, nb, dq0, dq1, s0, s1, s2, s3, layer_bytes = struct.unpack_from("<IIIiibbbbQ", buf, pos)
        structs.append(dict(rank=rank, first_block=first, n_blocks=nb, dq=(dq0, dq1), sign=(s0, s1, s2, s3),
                            layer_bytes=layer_bytes))
        pos += 32
    layers = []
    for _ in range(T):
        s, tag, off = struct.unpack_from("<IIQ", buf, pos)
        layers.append(dict(structure=s, tag=tag, offset=off))
        pos += 16
    blocks = []
    for _ in range(Bs):
        q = struct.unpack_from("<6i", buf, pos)
        d0, d1, d2, s, offset = struct.unpack_from("<IIIIQ", buf, pos + 24)
        blocks.append(dict(qn=((q[0], q[1]), (q[2], q[3]), (q[4], q[5])), dim=(d0, d1, d2), structure=s, offset=offset))
        pos += 48
    slack = buf[pos:hb]
    payload = buf[hb:hb + P]
    return fixed, structs, layers, blocks, slack, payload


def read_stream_v3(buf: bytes):
    """Wire format v3 (tensors of rank up to 4), field list re-typed with ``struct``: the v1
    fixed header and tensor records, 64-byte block records with four legs."""
    buf = bytes(buf)
    magic, version, endian, dtype, n_qn, max_rank, align, T, B, hb, P = struct.unpack_from("<8sIIIIIIQQQQ", buf, 0)
    fixed = dict(magic=magic, version=version, endian_tag=endian, dtype=dtype, n_qn=n_qn, max_rank=max_rank,
                 align=align, n_tensors=T, n_blocks=B, header_bytes=hb, payload_bytes=P)
    tensors = []
    pos = 64
    for _ in range(T):
        rank, first, nb, dq0, dq1, s0, s1, s2, s3, tag, reserved = struct.unpack_from("<IIIiibbbbII", buf, pos)
        tensors.append(dict(rank=rank, first_block=first, n_blocks=nb, dq=(dq0, dq1), sign=(s0, s1, s2, s3), tag=tag,
                            reserved=reserved))
        pos += 32
    blocks = []
    for _ in range(B):
        q = struct.unpack_from("<8i", buf, pos)
        d0, d1, d2, d3, tensor, reserved, offset = struct.unpack_from("<IIIIIIQ", buf, pos + 32)
        blocks.append(dict(qn=((q[0], q[1]), (q[2], q[3]), (q[4], q[5]), (q[6], q[7])), dim=(d0, d1, d2, d3), tensor=tensor,
                           reserved=reserved, offset=offset))
        pos += 64
    slack = buf[pos:hb]
    payload = buf[hb:hb + P]
    return fixed, tensors, blocks, slack, payload
