"""Whole-stream parity at BASELINE.json's full sizes: the C oracle run slice-wise over EVERY tensor range of a set whose
source pool lives on the device.

The oracle's inputs never come from the CUDA path: the source pool is filled by the seeded generator's device twin
(workloads/csrc/bsworkload.cu, harness code shared by both sides), copied to host memory once, and spot-checked there
against the host generator (workloads.values).  A slice is a range of tensors [t0, t1) of about ``slice_bytes`` of payload;
for it the oracle serializes the sub-set {tensors t0..t1-1} (a complete, valid stream of its own):

  - its payload is, byte for byte, payload[off(b0) : off(b1)) of the full stream (the payload of a tensor
    range does not depend on the other tensors), and
  - oracle.deserialize of it is, byte for byte, pool[slot(b0) : slot(b1)) of the full set's BS_LAYOUT_POOL image (D14: slots
    are a prefix sum in block order), untouched poison included.
"""
import numpy as np
import torch

import oracle
import workloads as W

SLICE_BYTES = 256 << 20


def equal_bytes(a: np.ndarray, b: np.ndarray) -> bool:
    """a == b for two uint8 arrays without a temporary the size of the inputs (torch.equal is threaded and early-outs)."""
    return a.shape == b.shape and torch.equal(torch.from_numpy(a), torch.from_numpy(b))


def first_difference(a: np.ndarray, b: np.ndarray) -> int:
    n = min(len(a), len(b))
    step = 1 << 24
    for lo in range(0, n, step):
        bad = np.nonzero(a[lo:lo + step] != b[lo:lo + step])[0]
        if bad.size:
            return lo + int(bad[0])
    return n


class HostPool:
    """The device source pool of an Uploaded(fill='device') set, copied to pageable host memory through one pinned buffer."""

    def __init__(self, bset, d_pool: torch.Tensor, check_tensors=6, seed=7):
        n = d_pool.numel()
        self.pool = np.empty(n, np.uint8)
        stage = torch.empty(min(n, 512 << 20), dtype=torch.uint8, pin_memory=True)
        for lo in range(0, n, stage.numel()):
            m = min(stage.numel(), n - lo)
            stage[:m].copy_(d_pool[lo:lo + m])
            self.pool[lo:lo + m] = stage[:m].numpy()
        self.addr = (np.uint64(self.pool.ctypes.data) + bset.pool_off).astype(np.uint64)
        # the device fill is the seeded generator: sampled tensors against the host generator, bit for bit
        rng = np.random.default_rng(seed)
        for t in sorted({0, bset.n_tensors - 1} | set(int(x) for x in rng.choice(bset.n_tensors, size=check_tensors, replace=False))):
            b0 = int(bset.tensors["first_block"][t])
            b1 = b0 + int(bset.tensors["n_blocks"][t])
            ref, offs = W.fill_pool_host(bset, b0, b1, compact=True)
            ref = ref.view(np.uint8)
            for i in range(b0, b1):
                nb = int(bset.nelems[i]) * 8
                o = int(bset.pool_off[i])
                assert (self.pool[o:o + nb] == ref[int(offs[i - b0]): int(offs[i - b0]) + nb]).all(), \
                    f"device fill of block {i} differs from the seeded host generator"


class OracleSlices:
    """Iterates over tensor ranges of ~slice_bytes; for each yields what the oracle says the stream payload and the
    deserialized pool image of that range are."""

    def __init__(self, bset, host_addr: np.ndarray, slice_bytes: int = SLICE_BYTES, want_pool: bool = True):
        self.bset, self.addr, self.want_pool = bset, host_addr, want_pool
        nb = bset.nelems * np.uint64(8)
        self.stored = (nb + np.uint64(15)) // np.uint64(16) * np.uint64(16)      # test-side restatement, only to cut slices
        self.slots = (nb + np.uint64(255)) // np.uint64(256) * np.uint64(256)
        fb = np.minimum(bset.tensors["first_block"].astype(np.int64), max(bset.n_blocks - 1, 0))
        per_t = np.add.reduceat(self.stored, fb) if bset.n_tensors and bset.n_blocks else np.zeros(bset.n_tensors, np.uint64)
        per_t[bset.tensors["n_blocks"] == 0] = 0
        cuts, acc = [0], 0
        for t in range(bset.n_tensors):
            acc += int(per_t[t])
            if acc >= slice_bytes:
                cuts.append(t + 1)
                acc = 0
        if cuts[-1] != bset.n_tensors:
            cuts.append(bset.n_tensors)
        self.cuts = cuts
        self._out = None
        self._pool = None

    def __iter__(self):
        b = self.bset
        for t0, t1 in zip(self.cuts[:-1], self.cuts[1:]):
            b0 = int(b.tensors["first_block"][t0])
            b1 = int(b.tensors["first_block"][t1 - 1] + b.tensors["n_blocks"][t1 - 1])
            sub_t = b.tensors[t0:t1].copy()
            sub_t["first_block"] -= b0
            hb_s, tot_s = oracle.serialized_size(t1 - t0, b.dim[b0:b1])
            if self._out is None or self._out.size < tot_s:
                self._out = np.empty(int(tot_s * 1.25) + 4096, np.uint8)
            s = oracle.serialize(sub_t, b.qn[b0:b1], b.dim[b0:b1], self.addr[b0:b1], capacity=tot_s, out=self._out)
            pool = None
            if self.want_pool:
                need = oracle.pool_bytes(s)
                if self._pool is None or self._pool.size < need:
                    self._pool = np.empty(int(need * 1.25) + 4096, np.uint8)
                self._pool[:need] = 0xEE
                pool = oracle.deserialize(s, pool=self._pool[:max(need, 1)])["pool"][:need]
            yield dict(t0=t0, t1=t1, b0=b0, b1=b1, payload=s[hb_s:], pool=pool)


class DeviceReader:
    """Reads ranges of a device byte tensor into one reusable pinned buffer (returns a numpy view, valid until the next read)."""

    def __init__(self, nbytes: int = SLICE_BYTES + (SLICE_BYTES >> 1)):
        self.stage = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)

    def read(self, t: torch.Tensor, lo: int, n: int) -> np.ndarray:
        if n > self.stage.numel():
            self.stage = torch.empty(int(n * 1.25), dtype=torch.uint8, pin_memory=True)
        self.stage[:n].copy_(t[lo:lo + n])
        return self.stage[:n].numpy()


def check_against_oracle(bset, host_addr, header=None, payload_reader=None, pool_reader=None, hb=None, total=None, need=None):
    """100 % of what the CUDA path produced against the oracle, slice by slice.
    header         : numpy bytes [0, hb) of the CUDA stream            -> oracle.emit_header
    payload_reader : (lo, n) -> numpy payload bytes [lo, lo + n)       -> the payload of the oracle's stream of every slice
    pool_reader    : (lo, n) -> numpy bytes of the BS_LAYOUT_POOL image -> oracle.deserialize of every slice, every block and
                     every untouched (poisoned 0xEE) byte between blocks
    Returns (payload bytes compared, pool bytes compared)."""
    if header is not None:
        want_h = oracle.emit_header(bset.tensors, bset.qn, bset.dim)
        assert len(header) == len(want_h) and (hb is None or hb == len(want_h))
        assert equal_bytes(header, want_h), f"header differs first at byte {first_difference(header, want_h)}"
    off = poff = 0
    for sl in OracleSlices(bset, host_addr, want_pool=pool_reader is not None):
        n = len(sl["payload"])
        if payload_reader is not None:
            got = payload_reader(off, n)
            assert equal_bytes(got, sl["payload"]), (f"tensors [{sl['t0']}, {sl['t1']}): payload differs first at payload byte "
                                                     f"{off + first_difference(got, sl['payload'])}")
        off += n
        if pool_reader is not None:
            m = len(sl["pool"])
            got = pool_reader(poff, m)
            assert equal_bytes(got, sl["pool"]), (f"tensors [{sl['t0']}, {sl['t1']}): pool image differs first at pool byte "
                                                  f"{poff + first_difference(got, sl['pool'])}")
            poff += m
    if total is not None:
        assert hb + off == total, "the slices do not tile the payload"
    if need is not None and pool_reader is not None:
        assert poff == need, "the slices do not tile the pool"
    return off, poff
