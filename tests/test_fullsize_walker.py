"""The slice-wise walk the full-size GPU tests use (tests/fullsize.py) against the oracle run in one piece: the payloads of
the slices concatenate to the whole stream's payload and their pool images to the whole pool image.
Test infrastructure checked on the CPU, so that a mistake in the slicing cannot hide a mismatch on the GPU box."""
import numpy as np

import oracle
import workloads as W
from tests.fullsize import OracleSlices, check_against_oracle
from tests.util import host_addrs


def test_slices_tile_the_stream_and_the_pool():
    for bset in (W.make_config("2", n_ops=60), W.make_set("lognormal", 12, D=300, S=30, M=4, N0=3, n_ops=40, n_site=2,
                                                           dims="lognormal", sigma=1.0)):
        pool, offs = W.fill_pool_host(bset)
        addr = host_addrs(pool, offs)
        whole = oracle.serialize(bset.tensors, bset.qn, bset.dim, addr)
        hb = oracle.header_bytes(bset.n_tensors, bset.n_blocks)
        ref = oracle.deserialize(whole)
        need = oracle.pool_bytes(whole)
        for slice_bytes in (1 << 16, 1 << 20, 1 << 40):
            sl = list(OracleSlices(bset, addr, slice_bytes=slice_bytes))
            assert sl[0]["t0"] == 0 and sl[-1]["t1"] == bset.n_tensors
            assert all(a["t1"] == b["t0"] for a, b in zip(sl[:-1], sl[1:]))
        n_slices = 0
        payload, image = [], []
        for s in OracleSlices(bset, addr, slice_bytes=1 << 18):
            payload.append(s["payload"].copy())
            image.append(s["pool"].copy())
            n_slices += 1
        assert n_slices >= 3
        assert (np.concatenate(payload) == whole[hb:]).all()
        assert (np.concatenate(image) == ref["pool"][:need]).all()
        # and the checker itself: passes on the oracle's own bytes, fails on one flipped payload byte / pool byte
        check_against_oracle(bset, addr, header=whole[:hb], payload_reader=lambda lo, n: whole[hb + lo: hb + lo + n],
                             pool_reader=lambda lo, n: ref["pool"][lo: lo + n], hb=hb, total=len(whole), need=need)
        bad = whole.copy()
        bad[hb + (len(whole) - hb) // 2] ^= 1
        try:
            check_against_oracle(bset, addr, payload_reader=lambda lo, n: bad[hb + lo: hb + lo + n])
            raise RuntimeError("a flipped payload byte went unnoticed")
        except AssertionError:
            pass
        badp = ref["pool"].copy()
        badp[need - 1] ^= 1          # the last byte of the last slot: untouched poison
        try:
            check_against_oracle(bset, addr, pool_reader=lambda lo, n: badp[lo: lo + n])
            raise RuntimeError("a flipped pool byte went unnoticed")
        except AssertionError:
            pass
