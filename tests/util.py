"""Shared test plumbing: run the oracle on a workloads.BlockSparseSet (host memory)."""
import hashlib

import numpy as np

import oracle
import workloads as W


def read_hex_fixture(path):
    b = bytearray()
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        b += bytes.fromhex(line.split(":", 1)[1].replace(" ", ""))
    return bytes(b)


def sha256(b) -> str:
    return hashlib.sha256(bytes(b)).hexdigest()


def host_addrs(pool: np.ndarray, offs: np.ndarray) -> np.ndarray:
    return (np.uint64(pool.ctypes.data) + offs.astype(np.uint64)).astype(np.uint64)


def oracle_stream(bset, pool=None, offs=None):
    """Whole stream from the oracle for a set whose values come from the seeded generator."""
    if pool is None:
        pool, offs = W.fill_pool_host(bset)
    addr = host_addrs(pool, offs)
    return oracle.serialize(bset.tensors, bset.qn, bset.dim, addr), pool, offs


def blocks_from(addr, dim, base_ptr, pool_u8):
    """List of uint64 views (bit patterns) of each block, given host addresses inside pool_u8."""
    out = []
    d = dim.astype(np.uint64)
    for i in range(len(addr)):
        n = int(d[i, 0] * d[i, 1] * d[i, 2])
        o = int(addr[i]) - base_ptr
        out.append(pool_u8[o:o + 8 * n].view(np.uint64))
    return out
