"""Counter-based value generator: uniform[-1, 1) fp64, identical bits on host and device.

value(seed, i, e) for element ``e`` of block ``i`` is the ``(i << 32 | e)``-th output
(0-based) of the SplitMix64 sequence started at ``seed`` mapped to [-1, 1):

    z  = seed + (ctr + 1) * 0x9E3779B97F4A7C15           (mod 2^64)
    z  = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9
    z  = (z ^ (z >> 27)) * 0x94D049BB133111EB
    z ^= z >> 31
    u  = z >> 11                                          (53 bits)
    value = u * 2^-52 - 1.0                               (exact in IEEE fp64)

Every step is exact, so numpy here, the C helper in ``csrc/bsfill_host.c`` and the
device kernel in ``csrc/bsworkload.cu`` produce the same bits.  This is input
generation only (SURVEY §8(d) "Values"); the serializer never looks at values.
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64_at(seed: int, ctr: np.ndarray) -> np.ndarray:
    """The ``ctr``-th (0-based) SplitMix64 output for ``seed``, vectorised over ``ctr`` (uint64)."""
    ctr = np.asarray(ctr, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (ctr + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def _to_unit(z: np.ndarray) -> np.ndarray:
    u = (z >> np.uint64(11)).astype(np.float64)  # < 2^53: exact
    return u * (2.0 ** -52) - 1.0


def block_values(seed: int, block_ids: np.ndarray, nelems: np.ndarray) -> np.ndarray:
    """Values of the given blocks, concatenated in the given order (flat float64)."""
    block_ids = np.asarray(block_ids, dtype=np.uint64)
    nelems = np.asarray(nelems, dtype=np.int64)
    total = int(nelems.sum())
    if total == 0:
        return np.empty(0, dtype=np.float64)
    starts = np.zeros(len(nelems), dtype=np.int64)
    np.cumsum(nelems[:-1], out=starts[1:])
    e = np.arange(total, dtype=np.int64) - np.repeat(starts, nelems)
    ctr = (np.repeat(block_ids, nelems) << np.uint64(32)) | e.astype(np.uint64)
    return _to_unit(splitmix64_at(seed, ctr))


def fill_pool_host(bset, block_lo: int = 0, block_hi: int | None = None,
                   compact: bool = False, chunk_elems: int = 1 << 24):
    """Materialise block values on the host.

    compact=False: returns (pool, byte_offsets) laid out exactly as ``bset.pool_off`` (whole set only).
    compact=True : returns (pool, byte_offsets) for blocks [block_lo, block_hi) packed back to back at
                   64-byte-aligned offsets — what the slice-wise oracle runs use for the large configs.
    """
    B = bset.n_blocks
    if block_hi is None:
        block_hi = B
    ids = np.arange(block_lo, block_hi, dtype=np.int64)
    nel = bset.nelems[block_lo:block_hi].astype(np.int64)
    if compact:
        sz = (nel * 8 + 63) // 64 * 64
        offs = np.zeros(len(ids), dtype=np.uint64)
        if len(ids) > 1:
            offs[1:] = np.cumsum(sz[:-1]).astype(np.uint64)
        pool_bytes = int(sz.sum())
    else:
        if block_lo != 0 or block_hi != B:
            raise ValueError("scattered placement is defined for the whole set only")
        offs = bset.pool_off.copy()
        pool_bytes = int(bset.pool_bytes)
    pool = np.zeros(max(pool_bytes // 8, 1), dtype=np.float64)
    # chunked so that the temporaries stay bounded
    i = 0
    n = len(ids)
    csum = np.concatenate([[0], np.cumsum(nel)])
    while i < n:
        j = int(np.searchsorted(csum, csum[i] + chunk_elems, side="right")) - 1
        j = max(j, i + 1)
        j = min(j, n)
        vals = block_values(bset.seed, ids[i:j], nel[i:j])
        dst = (np.repeat(offs[i:j] // np.uint64(8), nel[i:j]).astype(np.int64)
               + (np.arange(len(vals), dtype=np.int64) - np.repeat(csum[i:j] - csum[i], nel[i:j])))
        pool[dst] = vals
        i = j
    return pool, offs
