"""GPU-side test plumbing: upload a workloads set, call the C ABI through the Python binding."""
import numpy as np
import torch

import paper_2412_04676_b200 as bs
import workloads as W

DEV = "cuda"


class Uploaded:
    """A BlockSparseSet resident on the device: pool + descriptor arrays."""

    def __init__(self, bset, host_pool=None, host_offs=None, fill="host", misalign: int = 0):
        self.bset = bset
        if fill == "device":
            from workloads.device import fill_pool_device
            self.pool, self.addr = fill_pool_device(bset, DEV)
            self.host_pool, self.host_offs = None, bset.pool_off
        else:
            if host_pool is None:
                host_pool, host_offs = W.fill_pool_host(bset)
            self.host_pool, self.host_offs = host_pool, host_offs
            raw = torch.from_numpy(host_pool.view(np.uint8).copy())
            if misalign:
                buf = torch.zeros(raw.numel() + 64, dtype=torch.uint8, device=DEV)
                buf[misalign:misalign + raw.numel()] = raw.to(DEV)
                self.pool = buf
                base = buf.data_ptr() + misalign
            else:
                self.pool = raw.to(DEV)
                base = self.pool.data_ptr()
            self.addr = (np.uint64(base) + host_offs.astype(np.uint64)).astype(np.uint64)
        self.dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, self.addr, DEV)


def gpu_serialize(dset, capacity, opts=None, poison=0xCD, ws=None):
    """bs_serialize into a poisoned buffer.  Returns (stream uint8 tensor [capacity], result dict)."""
    out = torch.full((max(capacity, 16),), poison, dtype=torch.uint8, device=DEV)
    if ws is None:
        ws = bs.Workspace(dset.n_tensors, dset.n_blocks, max(capacity, 1 << 16), DEV)
    bs.serialize(dset.desc, out.data_ptr(), capacity, ws.ptr, ws.nbytes, ws.result_ptr, opts, bs.current_stream())
    res = ws.read_result()
    return out, res


def gpu_deserialize(stream_t, nbytes, cap_t, cap_b, pool_bytes, flags=bs.LAYOUT_POOL, opts=None, out=None, poison=0xEE):
    if out is None:
        out = bs.DeviceSet.empty(cap_t, cap_b, DEV, fill=0xAB)
    pool = torch.full((max(pool_bytes, 256),), poison, dtype=torch.uint8, device=DEV)
    ws = bs.Workspace(cap_t, cap_b, max(nbytes, 1 << 16), DEV)
    bs.deserialize(stream_t.data_ptr(), nbytes, out.desc, pool.data_ptr(), pool_bytes, flags, ws.ptr, ws.nbytes,
                   ws.result_ptr, opts, bs.current_stream())
    res = ws.read_result()
    return out, pool, res
