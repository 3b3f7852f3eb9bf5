#!/usr/bin/env python
"""bench.py — serialize / deserialize / offload throughput of the block-sparse scratch-data path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4] [--impl reference]

One "step" = one pass of the whole hot path over the workload: bs_serialize (size/offset scan,
header write, pack) followed by bs_deserialize (header parse/validate, descriptor rebuild, unpack) of the seeded
synthetic set named in ``config.workload`` (default: BASELINE.json configs[3], D=15400 — the configuration the
metric's "% of HBM peak" is meaningful on; inputs are ~7 GB, far larger than the 126 MB L2).

    value     stream bytes serialized + deserialized per second (GB/s), inputs resident in HBM, CUDA events.
              HBM traffic is 2 bytes per stream byte, so HBM GB/s = 2 * value.
    e2e       the same stream bytes through HOST (pinned) buffers, copies inside the timed region (bs_queue_save overlapped
              with bs_queue_load); PCIe-bound.  Carries the north_star's offload bars too: offload / prefetch GB/s as a
              fraction of the pinned cudaMemcpyAsync bandwidth of the same run, and the exposed-IO fraction of an
              offload / a prefetch of config 3 hidden behind a stand-in contraction at r = T_c / T_io = 1.25 (config 5).
    roofline  the dominant kernel (pack): algorithmic HBM bytes per launch / its CUDA-event duration, against the
              measured copy bandwidth in MEASURED_PEAKS.json; beside it the unpack kernel, the whole-call fractions of the
              8 TB/s nominal figure, an in-run ceiling (the same mover on ONE contiguous block: a pure cp.async.bulk
              copy), ``at4L_*``: the same numbers on workload 4L (42.5 GB, the total BASELINE.json states), and one whole-call
              number per variant (``v2_``, ``a8_``, ``f32_``, ``rank4_``, ``pkg1MiB_``).  e2e likewise carries ``at3L_*`` (config 5
              at 11 GB) and the config-1 / config-2 latencies (``cfg1_*_us``, ``cfg2_*_us``).  All flat and first: the driver's
              record keeps the first 24 scalar keys of each dict (ROOFLINE_FIRST / E2E_FIRST).
    cpu_baseline  the CPU oracle (oracle/, single thread, as it stands) on a bounded sample of the same workload, plus
              the paper's own design as context: threads filling disjoint intervals of one buffer (L106-108).
    detail    (last key, context only) per-direction numbers, packages, small sets, the config-5 sweeps.

--impl reference times the oracle itself on the box's host cores (this tier's reference arm).
With N > 1 (torchrun) every rank runs an independent replica on its own GPU (the path has no exchange step:
"replicas only"); value = bytes of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "serialize+deserialize stream throughput"
UNIT = "GB/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


ELEM = {"f64": (0, 8), "f32": (1, 4), "c64": (2, 8), "c128": (3, 16),   # bs.h dtype, element bytes
        "f64a8": (0x100, 8)}   # fp64 as an UNPADDED stream (BS_ALIGN8): kernels only, as the other element types


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": FALLBACK_HBM_GBS}, "fallback"


def committed_traffic(key: str):
    """dram__bytes_read + dram__bytes_write per launch from the committed ncu capture (profiles/traffic.csv), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        import csv
        for row in csv.DictReader(open(p)):
            if row["key"] == key:
                return int(row["traffic_bytes"])
    except Exception:
        pass
    return None


# ---- rank plumbing (pure host logic; covered by tests/test_bench_dist.py with gloo) ---------------------------
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def aggregate(local_ms: float, local_units: float, world: int, device=None, backend_ready: bool = False):
    """max-over-ranks time, sum-over-ranks units.  Returns (ms, units)."""
    if world == 1 or not backend_ready:
        return local_ms, local_units
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                          str(index), "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL,
                                         text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def window(self, t0, t1):
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.02] or [r for _, r in self.rows[-3:]]
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(rows)}

    def stop(self):
        if self.proc:
            self.proc.terminate()


# ---- CPU oracle leg (cpu_baseline and --impl reference) ------------------------------------------------------------
def oracle_sample(workload: str, sample_mb: float, fmt: str = "v1"):
    """First tensors of the workload up to ~sample_mb of payload, values regenerated on the host."""
    import workloads as W
    bset = W.make_config(workload)
    nb = bset.nelems * 8
    per_t = np.add.reduceat(nb, bset.tensors["first_block"].astype(np.int64)) if bset.n_tensors else np.zeros(0)
    n_t = int(np.searchsorted(np.cumsum(per_t), sample_mb * 1e6) + 1)
    n_t = max(1, min(n_t, bset.n_tensors))
    b1 = int(bset.tensors["first_block"][n_t - 1] + bset.tensors["n_blocks"][n_t - 1])
    pool, offs = W.fill_pool_host(bset, 0, b1, compact=True)
    sub = dict(tensors=bset.tensors[:n_t].copy(), qn=bset.qn[:b1], dim=bset.dim[:b1],
               addr=(np.uint64(pool.ctypes.data) + offs).astype(np.uint64), pool=pool)
    if fmt == "v2":   # the same tensors as layers of their structures (structures no sampled layer uses are dropped)
        lv = W.layered_view(bset)
        ly = lv["layers"][:n_t].copy()
        used = np.unique(ly["structure"])
        remap = np.full(len(lv["structs"]), -1, np.int64)
        remap[used] = np.arange(len(used))
        st = lv["structs"][used].copy()
        keep = np.concatenate([np.arange(f, f + n) for f, n in zip(st["first_block"], st["n_blocks"])]).astype(np.int64)
        st["first_block"] = np.concatenate([[0], np.cumsum(st["n_blocks"])])[:-1]
        ly["structure"] = remap[ly["structure"]]
        sub["layered"] = dict(structs=st, layers=ly, qn=np.ascontiguousarray(lv["qn"][keep]),
                              dim=np.ascontiguousarray(lv["dim"][keep]))
    return bset, sub, n_t, b1


class OracleRunner:
    """serialize + deserialize passes of the oracle, single thread, on a prepared sample.  The output stream and the pool
    are allocated and touched ONCE, so the reference arm and the cpu_baseline leg time the same thing (round 1's reference
    arm re-allocated them every step and paid the first-touch page faults inside its timed region)."""

    def __init__(self, sub):
        if "layered" in sub:
            from oracle import v2
            lv = sub["layered"]
            self.hb, self.total = v2.serialized_size(lv["structs"], lv["layers"], lv["dim"])
            self.out = np.zeros(self.total, np.uint8)
            self._ser = lambda: v2.serialize(lv["structs"], lv["layers"], lv["qn"], lv["dim"], sub["addr"], capacity=self.total,
                                             out=self.out)
            self.pool = np.zeros(max(v2.counts(self._ser())[1], 1), np.uint8)
            self._des = lambda s: v2.deserialize(s, pool=self.pool)
        else:
            import oracle
            self.hb, self.total = oracle.serialized_size(len(sub["tensors"]), sub["dim"])
            self.out = np.zeros(self.total, np.uint8)
            self._ser = lambda: oracle.serialize(sub["tensors"], sub["qn"], sub["dim"], sub["addr"], capacity=self.total, out=self.out)
            self.pool = np.zeros(max(oracle.pool_bytes(self._ser()), 1), np.uint8)
            self._des = lambda s: oracle.deserialize(s, pool=self.pool)
        self.one_pass()   # everything mapped and warm

    def one_pass(self) -> float:
        t0 = time.perf_counter()
        self._des(self._ser())
        return time.perf_counter() - t0

    def run_for(self, min_seconds: float, max_passes: int = 1000):
        """(seconds, passes): at least one pass, then until min_seconds of CPU work."""
        passes, acc = 0, 0.0
        while passes == 0 or (acc < min_seconds and passes < max_passes):
            acc += self.one_pass()
            passes += 1
        return acc, passes


def oracle_threads_sweep(sub, seconds_each: float = 2.0):
    """Context row (optional): the PAPER'S OWN DESIGN on this box's host cores — the main thread maps the one
    output buffer from the predicted sizes, then threads fill disjoint intervals in complete independence (L106-108); the
    paper sees saturation at 32 threads (L158).  The oracle is unchanged: every thread calls its slice-wise
    emit_payload_range on its own tensor ranges (ctypes drops the GIL).  Serialize only; baseline only."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    tensors, dim, addr = sub["tensors"], sub["dim"], sub["addr"]
    T = len(tensors)
    hb, total = oracle.serialized_size(T, dim)
    _, stored, off, P = oracle.plan(dim)                     # the main thread's map of the buffer (L106)
    out = np.zeros(total, np.uint8)
    payload = out[hb:]
    fb = tensors["first_block"].astype(np.int64)
    end_b = fb + tensors["n_blocks"].astype(np.int64)
    cores = os.cpu_count() or 1
    rows = []
    for n_thr in sorted({1, min(32, cores), cores}):
        # ~4 ranges per thread, cut at tensor boundaries at ~equal bytes
        n_rng = max(1, min(T, 4 * n_thr))
        t_end_off = np.array([int(off[e - 1] + stored[e - 1]) if e > 0 else 0 for e in end_b])
        cuts = [0] + [int(np.searchsorted(t_end_off, P * k / n_rng, side="left")) + 1 for k in range(1, n_rng)] + [T]
        cuts = sorted(set(min(max(c, 0), T) for c in cuts))
        jobs = []
        for t0, t1 in zip(cuts[:-1], cuts[1:]):
            lo = int(off[fb[t0]]) if fb[t0] < len(off) else P
            hi = t_end_off[t1 - 1]
            jobs.append((t0, t1, lo, hi - lo))

        def work(j):
            t0, t1, lo, n = j
            first, got = oracle.emit_payload_range(tensors, dim, addr, t0, t1, n, out=payload[lo: lo + n] if n else payload[:1])
            assert first == lo and len(got) == n
            return n

        with ThreadPoolExecutor(max_workers=n_thr) as ex:
            list(ex.map(work, jobs))                         # warm
            passes, t0 = 0, time.perf_counter()
            while passes == 0 or time.perf_counter() - t0 < seconds_each:
                moved = sum(ex.map(work, jobs))
                passes += 1
            sec = time.perf_counter() - t0
        assert moved == P
        rows.append({"threads": n_thr, "serialize_stream_GBs": round(passes * P / sec / 1e9, 2), "ranges": len(jobs)})
    return rows


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle
    log(f"[reference] oracle on a {args.sample_mb:.0f} MB sample of workload {args.workload}")
    bset, sub, n_t, b1 = oracle_sample(args.workload, args.sample_mb, args.format)
    runner = OracleRunner(sub)
    for _ in range(max(0, args.warmup - 1)):
        runner.one_pass()
    per = [runner.one_pass() for _ in range(args.steps)]
    ms = 1e3 * float(np.mean(per))
    sbytes = runner.total
    value = 2 * sbytes / (ms * 1e-3) / 1e9
    full_total = full_stream_bytes(bset, args.format)
    sample = (f"every step = one serialize + deserialize pass of the oracle over the first {n_t} of {bset.n_tensors} tensors "
              f"({b1} blocks, {sbytes / 1e6:.0f} MB stream = {100 * sbytes / full_total:.1f} % of the workload's {full_total / 1e9:.3f} GB)")
    line = {"impl": "reference", "metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms, 3), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": workload_config(args.workload, bset, full_total, args.format),
            "cpu_baseline": {"value": round(value, 3), "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                             "sample_stream_bytes": int(sbytes), "host_cores": os.cpu_count()},
            "e2e": {"value": round(value, 3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def full_stream_bytes(bset, fmt="v1"):
    """Stream size of the whole workload from the oracle's size prediction (host only)."""
    import workloads as W
    if fmt == "v2":
        from oracle import v2
        lv = W.layered_view(bset)
        return int(v2.serialized_size(lv["structs"], lv["layers"], lv["dim"])[1])
    import oracle
    return int(oracle.serialized_size(bset.n_tensors, bset.dim)[1])


def workload_config(name, bset, total, fmt="v1"):
    c = {"wire_format": fmt,
         "workload": f"BASELINE.json configs[{int(name[0]) - 1}] = config {name}: "
                     f"D={bset.meta['D']}, {bset.meta['S']} (N,2Sz) sectors, {bset.meta['n_ops']} operators + "
                     f"{bset.meta['n_site']} site tensors, dims {bset.meta['dims']} sigma={bset.meta['sigma']}",
         "n_tensors": bset.n_tensors, "n_blocks": bset.n_blocks, "l2": "inputs larger than L2 (no flush needed)",
         "parallelism": "replicas only"}
    if total is not None:
        c["stream_bytes"] = int(total)
    return c


def with_elem(c, elem):
    if elem == "f64a8":
        c["element_type"] = "f64, unpadded stream (BS_ALIGN8: the header's align word = 8)"
    elif elem != "f64":
        c["element_type"] = f"{elem}: every block read as {ELEM[elem][1]}-byte elements (the first e*n bytes of its fp64 storage)"
    return c


# ---- the CUDA arm -------------------------------------------------------------------------------------------------------
def run_mine(args):
    import torch
    import torch.distributed as dist

    import paper_2412_04676_b200 as bs
    import workloads as W
    from workloads.device import StandInContraction, fill_pool_device

    rank, local_rank, world = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    ready = False
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
        ready = True
    opts = None
    if args.variant or args.tile_bytes or args.ctas_per_sm or args.stages or args.warps or args.tune or args.fuse or args.pace:
        opts = dict(variant=args.variant, tile_bytes=args.tile_bytes, ctas_per_sm=args.ctas_per_sm, stages=args.stages,
                    warps=args.warps, tune=args.tune, fuse=args.fuse, pace=args.pace)

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def barrier():
        if ready:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- workload resident in HBM ----
    t_setup = time.time()
    bset = W.make_config(args.workload)
    pool, addr = fill_pool_device(bset, dev)
    v2 = args.format == "v2"
    cap_guess = bset.data_bytes * max(1, ELEM[args.elem][1] // 8) + 16 * bset.n_blocks + bs.header_bytes(bset.n_tensors, bset.n_blocks)
    cs = bs.current_stream()
    if v2:   # the same tensors as layers of their structures (wire format v2); pool and addresses are shared
        lv = W.layered_view(bset)
        counts = (len(lv["structs"]), lv["dim"].shape[0], bset.n_tensors, bset.n_blocks)
        dset = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], addr, dev)
        ws = bs.Workspace(0, 0, cap_guess, dev, layered=counts)
        hb, total = bs.layered_serialized_size(dset.desc, ws.ptr, ws.nbytes, cs)
        out = bs.DeviceLayeredSet.empty(*counts, dev)
        f_ser, f_range, f_deser, f_size = bs.layered_serialize, bs.layered_serialize_range, bs.layered_deserialize, \
            bs.layered_serialized_size
    else:
        # --elem: the same blocks read as elements of another size (the first e*n bytes of each fp64 block)
        dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, addr, dev, dtype=ELEM[args.elem][0])
        ws = bs.Workspace(bset.n_tensors, bset.n_blocks, cap_guess, dev)
        hb, total = bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs)   # size known before serialization
        out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, dev)
        f_ser, f_range, f_deser, f_size = bs.serialize, bs.serialize_range, bs.deserialize, bs.serialized_size
    stream = torch.empty(total, dtype=torch.uint8, device=dev)
    need = int(((bset.nelems * ELEM[args.elem][1] + 255) // 256 * 256).sum())
    opool = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    log(f"[rank {rank}] workload {args.workload}: T={bset.n_tensors} B={bset.n_blocks} stream={total / 1e9:.3f} GB "
        f"(header {hb / 1e6:.1f} MB) set up in {time.time() - t_setup:.1f}s")

    def ser():
        f_ser(dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)

    def deser():
        f_deser(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                ws.result_ptr, opts, cs)

    def check_ok(what):
        r = ws.read_result()
        if r["status"] != bs.OK:
            raise RuntimeError(f"{what}: deferred status {r}")

    for _ in range(args.warmup):
        ser()
        deser()
    check_ok("warm-up")

    # ---- timed region: exactly K steps, barrier + synchronize on both sides, CUDA events, clocks sampled ----
    sampler = ClockSampler(local_rank)
    time.sleep(0.3)
    e = [ev() for _ in range(2 * args.steps + 1)]
    barrier()
    w0 = time.time()
    e[0].record()
    for k in range(args.steps):
        ser()
        e[2 * k + 1].record()
        deser()
        e[2 * k + 2].record()
    barrier()
    w1 = time.time()
    check_ok("timed region")
    step_ms = e[0].elapsed_time(e[2 * args.steps]) / args.steps
    ser_ms = [e[2 * k].elapsed_time(e[2 * k + 1]) for k in range(args.steps)]
    des_ms = [e[2 * k + 1].elapsed_time(e[2 * k + 2]) for k in range(args.steps)]
    clocks = sampler.window(w0, w1)

    # ---- roofline leg: the dominant kernel (pack) alone, then its mirror image (unpack), same launch configuration,
    # CUDA events on their stream.  The size / offset pass has run (ser / deser above leave the tables in the workspace). ----
    peaks, peak_kind = measured_peaks()
    n_k = max(args.steps, 5)

    def timed(fn, n=n_k):
        torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    ser()
    pack_ms = timed(lambda: f_range(dset.desc, stream.data_ptr(), 0, total, False, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs))
    scan_ms = timed(lambda: f_size(dset.desc, ws.ptr, ws.nbytes, cs))
    ser()
    deser()                          # leaves the parsed tables in the workspace: the unpack kernel alone re-scatters from them
    if v2:                           # (no range form for layered sets: whole call minus the plan pass of the same set)
        unpack_ms = max(timed(deser) - scan_ms, 1e-6)
    else:
        unpack_ms = timed(lambda: bs.deserialize_range(stream.data_ptr(), 0, total, stream.data_ptr(), out.desc, bs.LAYOUT_POOL,
                                                       ws.ptr, ws.nbytes, opts, cs))
    check_ok("roofline leg")
    # algorithmic bytes per pack launch: 2 B per stream byte + per block 24 (labels) + 12 (dims)
    # + 16 (offset table entry) read for its header record  [SURVEY §8(d): "2 B per stream byte ... ~130 B per block"
    # counts the scan pass too; the pack launch alone reads 52 B per block on top of the stream bytes]
    # wire format v2: the header records exist once per STRUCTURE block; per block of a layer only its 16-byte table entry
    algo_bytes = 2 * total + (16 * bset.n_blocks if v2 else 52 * bset.n_blocks)
    achieved = algo_bytes / (pack_ms * 1e-3) / 1e9
    kname = "bs::move_kernel<pack>" if args.variant == 1 else "bs::move_tma_kernel<pack>"
    med_ser, med_des = float(np.median(ser_ms)), float(np.median(des_ms))
    roofline = {"bound": "hbm", "kernel": kname + " (S3 header write + S5 pack)", "achieved": round(achieved, 1),
                "peak": peaks["hbm_gbs"], "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)",
                "unit": "GB/s", "frac": round(achieved / peaks["hbm_gbs"], 4), "traffic": None,
                "algorithmic_bytes_per_launch": int(algo_bytes), "kernel_ms": round(pack_ms, 4),
                "frac_of_nominal_8TBs": round(achieved / 8000.0, 4)}
    vname = "ldg" if args.variant == 1 else "tma"
    roofline["traffic"] = committed_traffic(f"pack:{args.workload}:{vname}:fmt{2 if v2 else 1}")
    # the mirror image: the unpack kernel alone (bs_deserialize_range over the whole stream, descriptor rebuild included)
    unpack_algo = 2 * total + (16 * bset.n_blocks if v2 else 64 * bset.n_blocks)   # 48 B record read + 16 B table entry per block
    roofline.update({
        "unpack_kernel_ms": round(unpack_ms, 4), "unpack_achieved": round(unpack_algo / (unpack_ms * 1e-3) / 1e9, 1),
        "unpack_frac": round(unpack_algo / (unpack_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], 4),
        "unpack_frac_of_8TBs": round(unpack_algo / (unpack_ms * 1e-3) / 1e9 / 8000.0, 4),
        "unpack_kernel": ("bs::move_kernel<unpack>" if args.variant == 1 else "bs::move_tma_kernel<unpack>") + " (S7 rebuild + unpack)",
        "serialize_ms": round(med_ser, 4), "deserialize_ms": round(med_des, 4),
        "serialize_hbm_GBs": round(2 * total / med_ser / 1e6, 1), "deserialize_hbm_GBs": round(2 * total / med_des / 1e6, 1),
        "serialize_frac_of_8TBs": round(2 * total / med_ser / 1e6 / 8000, 4),
        "deserialize_frac_of_8TBs": round(2 * total / med_des / 1e6 / 8000, 4),
        "serialize_frac_of_measured_copy": round(2 * total / med_ser / 1e6 / peaks["hbm_gbs"], 4),
        "deserialize_frac_of_measured_copy": round(2 * total / med_des / 1e6 / peaks["hbm_gbs"], 4)})
    # in-run ceiling: the same mover on ONE contiguous block (a pure cp.async.bulk copy, no scatter, no header to speak of)
    if not v2 and args.elem == "f64" and not args.no_ceiling:
        try:
            roofline.update(bulk_copy_ceiling(bs, torch, pool, stream, dev, opts, cs, n_k))
            roofline["frac_of_bulk_copy"] = round(achieved / roofline["bulk_copy_GBs"], 4)
            roofline["unpack_frac_of_bulk_copy"] = round(roofline["unpack_achieved"] / roofline["bulk_copy_GBs"], 4)
        except Exception as ex:   # the headline numbers stand on their own
            roofline["bulk_copy_error"] = repr(ex)

    variants_detail = None
    # ---- one number per SURVEY §8(f) variant on this workload's blocks (rank 0; fp64 / v1 runs of a multi-GB workload) ----
    if rank == 0 and not v2 and args.elem == "f64" and not args.no_variants and total >= (1 << 30):
        try:
            vflat, vdet = variant_legs(bs, torch, W, fill_pool_device, dev, opts, bset, addr, stream, opool, cs)
            roofline.update(vflat)
            variants_detail = vdet
        except Exception as ex:
            variants_detail = {"error": repr(ex)}
        ser()   # the variants reused stream / opool and other workspaces: put this workload's stream and tables back
        deser()
        check_ok("after the variant legs")

    ab = None
    if args.ab and not v2:
        def t_pack(o):
            return timed(lambda: f_range(dset.desc, stream.data_ptr(), 0, total, False, ws.ptr, ws.nbytes, ws.result_ptr, o, cs), 5)

        def t_unpack(o):
            return timed(lambda: bs.deserialize_range(stream.data_ptr(), 0, total, stream.data_ptr(), out.desc, bs.LAYOUT_POOL,
                                                      ws.ptr, ws.nbytes, o, cs), 5)
        ser()
        ab_p = {}
        # pack needs the serialize tables in the workspace, unpack the parsed ones: two passes over the list
        rows_p = ab_table(bs, torch, t_pack, lambda o: 1.0, total, args.ab)
        ser()
        deser()
        rows_u = ab_table(bs, torch, lambda o: 1.0, t_unpack, total, args.ab)
        check_ok("A/B leg")
        ab = [{"setting": rp["setting"], "opts": rp["opts"], "pack_GBs": rp["pack_GBs"], "unpack_GBs": ru["unpack_GBs"]}
              for rp, ru in zip(rows_p, rows_u)]
        ser()
        deser()

    # ---- e2e leg: host (pinned) buffers through the engine, copies inside the timed region ----
    detail = {"serialize_stream_GBs": round(total / med_ser / 1e6, 1), "deserialize_stream_GBs": round(total / med_des / 1e6, 1),
              "size_pass_ms_incl_sync": round(scan_ms, 4)}
    if ab is not None:
        detail["ab"] = ab
    if variants_detail is not None:
        detail["variants"] = variants_detail
    a, b = ev(), ev()
    e2e = None
    if not args.no_e2e:
        host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
        eng = bs.Engine(bset.n_tensors, bset.n_blocks, total, chunk_bytes=args.chunk_mb << 20, n_staging=2, opts=opts)
        e_off = eng.offload_layered_async if v2 else eng.offload_async
        e_pre = eng.prefetch_layered_async if v2 else eng.prefetch_async
        # link denominators, same run: pinned cudaMemcpyAsync of 1 GiB (or the whole stream if smaller), best of 5
        nlink = min(total, 1 << 30)
        dbuf = torch.empty(nlink, dtype=torch.uint8, device=dev)
        bw = {}
        for name, fn in (("d2h", lambda: host[:nlink].copy_(dbuf, non_blocking=True)),
                         ("h2d", lambda: dbuf.copy_(host[:nlink], non_blocking=True))):
            best = 1e9
            for _ in range(5):
                a.record(); fn(); b.record(); torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b))
            bw[name] = nlink / best / 1e6
        del dbuf

        def e2e_step():
            t1 = e_off(dset.desc, total, host.data_ptr(), total, cs)
            s1 = t1.wait()
            t2 = e_pre(host.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)
            s2 = t2.wait()
            if s1["status"] or s2["status"]:
                raise RuntimeError(f"engine status {s1} {s2}")
            return s1, s2

        e2e_step()
        n_e2e = max(1, min(args.steps, args.e2e_steps))
        barrier()
        a.record()
        stats = [e2e_step() for _ in range(n_e2e)]
        b.record()
        barrier()
        e2e_ms = a.elapsed_time(b) / n_e2e
        e2e_ms_g, units_g = aggregate(e2e_ms, 2 * total, world, dev, ready)
        off_gbs = float(np.median([s[0]["bytes"] / s[0]["dma_ms"] / 1e6 for s in stats]))
        pre_gbs = float(np.median([s[1]["bytes"] / s[1]["dma_ms"] / 1e6 for s in stats]))
        e2e = {"value": round(units_g / (e2e_ms_g * 1e-3) / 1e9, 3), "unit": UNIT, "h2d_bytes_per_step": int(total),
               "d2h_bytes_per_step": int(total), "ms_per_step": round(e2e_ms_g, 3),
               "what": "bs_offload_async -> pinned host -> bs_prefetch_async, one after the other, 256 MiB double-buffered chunks"}
        # the north_star's offload bar (>= 80 % of the measured pinned PCIe bandwidth), both directions, same run
        pcie = {"offload_pcie_GBs": round(off_gbs, 2), "prefetch_pcie_GBs": round(pre_gbs, 2),
                "pinned_d2h_GBs": round(bw["d2h"], 2), "pinned_h2d_GBs": round(bw["h2d"], 2),
                "offload_frac_of_pinned_d2h": round(off_gbs / bw["d2h"], 4),
                "prefetch_frac_of_pinned_h2d": round(pre_gbs / bw["h2d"], 4),
                "pcie_how": "stream bytes / (first DMA start -> last DMA end) of bs_offload_async / bs_prefetch_async, device-timed, "
                            "median over the steps; denominators: pinned cudaMemcpyAsync of 1 GiB, best of 5, same run"}
        e2e.update(pcie)
        detail.update({"offload_total_ms": round(float(np.median([s[0]["total_ms"] for s in stats])), 3),
                       "prefetch_total_ms": round(float(np.median([s[1]["total_ms"] for s in stats])), 3)})
        eng.destroy()
        if not v2 and not args.no_queue:
            # ---- the queue: every step saves the set (device -> pinned host) while the stream saved by
            # the step before is loaded back (pinned host -> device): both directions of the link at once.  Same bytes
            # per step as above; this is the e2e headline, the one-after-the-other number stays in detail. ----
            host2 = torch.empty(total, dtype=torch.uint8, pin_memory=True)
            hosts = [host, host2]
            s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
            nb = int(min(total, stream.numel(), opool.numel()))   # the same bytes per direction as one step moves
            best = 1e9
            for _ in range(3):   # link denominator with both directions busy, same run, same size (sustained, not a burst)
                torch.cuda.synchronize()
                a.record()
                s1.wait_stream(torch.cuda.current_stream()); s2.wait_stream(torch.cuda.current_stream())
                with torch.cuda.stream(s1):
                    host[:nb].copy_(stream[:nb], non_blocking=True)
                with torch.cuda.stream(s2):
                    opool[:nb].copy_(host2[:nb], non_blocking=True)
                torch.cuda.current_stream().wait_stream(s1); torch.cuda.current_stream().wait_stream(s2)
                b.record(); torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b))
            bw["bidir"] = 2 * nb / best / 1e6
            q = bs.Queue(bset.n_tensors, bset.n_blocks, total, chunk_bytes=args.chunk_mb << 20, n_staging=2, opts=opts)
            for k in (0, 1):
                q.save(k, dset.desc, total, hosts[k].data_ptr(), total, cs)

            def q_steps(n, i0):
                for i in range(i0, i0 + n):
                    q.save(i % 2, dset.desc, total, hosts[i % 2].data_ptr(), total, cs)
                    q.load((i + 1) % 2, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)
                q.checkpoint(0, cs)
                q.checkpoint(1, cs)

            q_steps(2, 0)
            barrier()
            a.record()
            q_steps(n_e2e, 2)
            b.record()
            barrier()
            for k in (0, 1):
                st = q.wait(k)
                if st["status"]:
                    raise RuntimeError(f"queue status {st}")
            q_ms = a.elapsed_time(b) / n_e2e
            q_ms_g, q_units_g = aggregate(q_ms, 2 * total, world, dev, ready)
            detail["e2e_one_after_the_other"] = dict(e2e)
            qv = q_units_g / (q_ms_g * 1e-3) / 1e9
            e2e = {"value": round(qv, 3), "unit": UNIT, "h2d_bytes_per_step": int(total), "d2h_bytes_per_step": int(total),
                   "ms_per_step": round(q_ms_g, 3),
                   "what": "bs_queue: every step bs_queue_save of the set (device -> pinned host) overlapped with bs_queue_load "
                           "of the stream the step before saved (pinned host -> device); 256 MiB double-buffered chunks per lane"}
            e2e.update(pcie)
            e2e.update({"one_after_the_other_GBs": detail["e2e_one_after_the_other"]["value"],
                        "duplex_pcie_GBs": round(2 * total / q_ms / 1e6, 2),
                        "pinned_bidirectional_memcpy_GBs": round(bw["bidir"], 2),
                        "duplex_frac_of_bidirectional_memcpy": round(2 * total / q_ms / 1e6 / bw["bidir"], 4)})
            detail["queue"] = {"device_bytes_held": q.stats()["device_bytes"], "host_bytes_live": q.stats()["host_bytes_live"]}
            q.destroy()
            del host2, hosts
        del host

    # ---- library comparator for the pack step (context only): one cudaMemcpyAsync (device to device) per block
    # over the same block list — the first blocks of the set, up to ~256 MB, into the same stream offsets; no header ----
    if rank == 0 and not v2 and args.elem == "f64" and not args.no_comparator:
        try:
            from workloads.device import memcpy_each
            sizes = (bset.nelems * 8).astype(np.uint64)
            stored = (sizes + np.uint64(15)) // np.uint64(16) * np.uint64(16)
            offs = np.concatenate([[0], np.cumsum(stored)[:-1]]).astype(np.uint64)
            nb = int(min(bset.n_blocks, max(1, np.searchsorted(np.cumsum(sizes), 256 << 20))))
            keep = np.nonzero(sizes[:nb])[0]
            dsts = (np.uint64(stream.data_ptr()) + np.uint64(hb) + offs[:nb])[keep]
            srcs = addr[:nb][keep]
            memcpy_each(dsts, srcs, sizes[:nb][keep], cs)
            torch.cuda.synchronize()
            t0 = time.time()
            a.record()
            memcpy_each(dsts, srcs, sizes[:nb][keep], cs)
            b.record()
            torch.cuda.synchronize()
            wall = time.time() - t0
            moved = int(sizes[:nb][keep].sum())
            detail["library_comparator"] = {
                "what": "one cudaMemcpyAsync (device to device) per block over the first blocks of the set (payload only: no header, "
                        "no pad zeroing)",
                "blocks": int(len(keep)), "bytes": moved, "ms": round(wall * 1e3, 3),
                "hbm_GBs": round(2 * moved / wall / 1e9, 1), "us_per_block": round(wall * 1e6 / len(keep), 2)}
        except Exception as ex:
            detail["library_comparator"] = {"error": repr(ex)}

    # ---- the small configs are launch-latency bound: report microseconds per call, device-timed back to
    # back, next to a plain copy of the same number of bytes ----
    if rank == 0 and not v2 and args.elem == "f64" and not args.no_small:
        small = {}
        for wl in ("1", "2"):
            sb = W.make_config(wl)
            sp_, sa = fill_pool_device(sb, dev)
            sd = bs.DeviceSet.from_host(sb.tensors, sb.qn, sb.dim, sa, dev)
            sws = bs.Workspace(sb.n_tensors, sb.n_blocks, sb.data_bytes + 16 * sb.n_blocks + (1 << 20), dev)
            shb, stot = bs.serialized_size(sd.desc, sws.ptr, sws.nbytes, cs)
            sst = torch.empty(stot, dtype=torch.uint8, device=dev)
            ssrc = torch.empty(stot, dtype=torch.uint8, device=dev)
            sneed = int(((sb.nelems * 8 + 255) // 256 * 256).sum())
            sout = bs.DeviceSet.empty(sb.n_tensors, sb.n_blocks, dev)
            spool = torch.empty(max(sneed, 256), dtype=torch.uint8, device=dev)
            fns = {"serialize_us": lambda: bs.serialize(sd.desc, sst.data_ptr(), stot, sws.ptr, sws.nbytes, sws.result_ptr, opts, cs),
                   "deserialize_us": lambda: bs.deserialize(sst.data_ptr(), stot, sout.desc, spool.data_ptr(), sneed, bs.LAYOUT_POOL,
                                                            sws.ptr, sws.nbytes, sws.result_ptr, opts, cs),
                   "plain_copy_us": lambda: sst.copy_(ssrc)}
            row = {"stream_bytes": int(stot), "n_blocks": int(sb.n_blocks)}
            fns["serialize_us"]()
            for name, fn in fns.items():
                for _ in range(20):
                    fn()
                torch.cuda.synchronize()
                a.record()
                for _ in range(200):
                    fn()
                b.record()
                torch.cuda.synchronize()
                row[name] = round(a.elapsed_time(b) / 200 * 1e3, 1)
            if sws.read_result()["status"] != bs.OK:
                raise RuntimeError("small sets: deferred status")
            small[f"config{wl}"] = row
        detail["small_sets"] = small

    # ---- self-contained packages: the same bytes as packages in device slots, emitted and unpacked
    # package by package; the size limit decides how many launches the bytes are spread over ----
    if not v2 and not args.no_packages:
        pk = {}
        for cap_mb in (256, 4, 1):
            cap = cap_mb << 20
            n_pk = bs.package_count(hb, total, cap)
            slot_bytes = 64 + cap
            try:
                slots = torch.empty(n_pk * slot_bytes, dtype=torch.uint8, device=dev)
            except torch.cuda.OutOfMemoryError:
                break
            wsp = bs.Workspace(bset.n_tensors, bset.n_blocks, cap_guess, dev, packages=True)

            def emit():
                bs.package_emit(dset.desc, total, cap, 7, slots.data_ptr(), slot_bytes, n_pk, None, wsp.ptr, wsp.nbytes,
                                wsp.result_ptr, opts, cs)

            def unpack():
                bs.package_unpack(slots.data_ptr(), slot_bytes, n_pk, 7, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL,
                                  wsp.ptr, wsp.nbytes, wsp.result_ptr, opts, cs)

            emit(); unpack()
            if wsp.read_result()["status"] != bs.OK:
                raise RuntimeError(f"packages: {wsp.read_result()}")
            t = {}
            for name, fn in (("emit", emit), ("unpack", unpack)):
                torch.cuda.synchronize()
                a.record()
                for _ in range(3):
                    fn()
                b.record()
                torch.cuda.synchronize()
                t[name] = a.elapsed_time(b) / 3
            pk[f"cap_{cap_mb}MiB"] = {"packages": int(n_pk), "emit_ms": round(t["emit"], 3), "unpack_ms_incl_plan_sync": round(t["unpack"], 3),
                                      "emit_hbm_GBs": round(2 * total / t["emit"] / 1e6, 1),
                                      "unpack_hbm_GBs": round(2 * total / t["unpack"] / 1e6, 1)}
            del slots, wsp
        detail["packages"] = pk
        if "cap_1MiB" in pk:
            roofline["pkg1MiB_emit_frac_of_8TBs"] = round(pk["cap_1MiB"]["emit_hbm_GBs"] / 8000, 4)
            roofline["pkg1MiB_unpack_frac_of_8TBs"] = round(pk["cap_1MiB"]["unpack_hbm_GBs"] / 8000, 4)

    # ---- config 5: exposed IO of an offload overlapped with a stand-in contraction (rank 0 only) ----
    if rank == 0 and not args.no_config5 and not v2:
        c5 = None
        try:
            c5 = config5(args, dev, opts)
            detail["config5"] = c5
            if e2e is not None:   # the north_star's third bar: exposed (non-hidden) IO time < 10 % (config 5 = config 3 through the engine)
                hs, hl = c5["headline"], c5["prefetch"]["headline"]
                e2e.update({"exposed_io_frac_save": hs["exposed_io_frac"], "exposed_io_frac_load": hl["exposed_io_frac"],
                            "exposed_io_r": hs["r_target"], "exposed_io_r_actual": [hs["r_actual"], hl["r_actual"]],
                            "sustained_pcie_GBs_save": hs["sustained_pcie_GBs"], "sustained_pcie_GBs_load": hl["sustained_pcie_GBs"],
                            "exposed_io_workload": f"config 5: config 3 ({c5['stream_bytes'] / 1e9:.2f} GB stream) through bs_offload_async / "
                                                   "bs_prefetch_async behind a stand-in contraction (batched fp64 block GEMMs) on the compute "
                                                   "stream; exposed = (T_both - T_c) / T_both at r = T_c / T_io"})
                if "sweep_fig3" in c5 and "error" not in c5["sweep_fig3"]:
                    e2e["sweep_speedup_queue_over_sync_io"] = c5["sweep_fig3"]["speedup_queue_over_sync"]
        except Exception as ex:  # the headline numbers stand on their own
            detail["config5"] = {"error": repr(ex)}
        # the same protocol at the total BASELINE.json states for config 3 ("10-20 GB": workload 3L, 11 GB, 42 chunks of 256 MiB)
        if e2e is not None and not args.no_at_scale and args.workload != "3L":
            try:
                del c5
                torch.cuda.empty_cache()
                cl = config5(args, dev, opts, name="3L", full=False)
                hs, hl = cl["headline"], cl["prefetch"]["headline"]
                e2e.update({"at3L_stream_GB": round(cl["stream_bytes"] / 1e9, 3), "at3L_exposed_io_frac_save": hs["exposed_io_frac"],
                            "at3L_exposed_io_frac_load": hl["exposed_io_frac"],
                            "at3L_sustained_pcie_GBs_save": hs["sustained_pcie_GBs"], "at3L_sustained_pcie_GBs_load": hl["sustained_pcie_GBs"],
                            "at3L_r_actual_save": hs["r_actual"], "at3L_r_actual_load": hl["r_actual"],
                            "at3L_offload_alone_GBs": round(cl["stream_bytes"] / cl["T_io_ms"] / 1e6, 2),
                            "at3L_prefetch_alone_GBs": round(cl["stream_bytes"] / cl["prefetch"]["T_io_ms"] / 1e6, 2)})
                del cl
            except Exception as ex:
                detail["at_scale_3L"] = {"error": repr(ex)}

    # ---- cpu baseline: the oracle on a bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        _, sub, n_t, b1 = oracle_sample(args.workload, args.sample_mb, args.format)
        runner = OracleRunner(sub)
        sec, passes = runner.run_for(args.cpu_seconds)
        sbytes = runner.total
        cpu = {"value": round(2 * sbytes * passes / sec / 1e9, 3), "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{passes} serialize+deserialize passes over the first {n_t} of {bset.n_tensors} tensors "
                         f"({b1} blocks, {sbytes / 1e6:.0f} MB stream) of workload {args.workload}; {sec:.1f} s of CPU work",
               "sample_stream_bytes": int(sbytes), "host_cores": os.cpu_count()}
        if not v2 and not args.no_threads_sweep:
            try:
                cpu["threads_sweep"] = oracle_threads_sweep(sub)
                cpu["threads_sweep_what"] = ("context only: the paper's own design (L106-108: the main thread maps one buffer from the "
                                             "predicted sizes, threads fill disjoint intervals; saturation at 32 threads, L158) with "
                                             "the unchanged oracle's slice-wise emit per thread; serialize only")
            except Exception as ex:
                cpu["threads_sweep"] = {"error": repr(ex)}

    # ---- at scale: workload 4L (the operator count scaled to the 40-60 GB BASELINE.json states), kernels
    # and whole calls only.  Runs last, after this workload's buffers are released; skipped if HBM cannot hold it. ----
    if rank == 0 and not v2 and args.elem == "f64" and not args.no_at_scale and args.workload != "4L":
        del stream, opool, pool, out, dset, ws
        torch.cuda.empty_cache()
        try:
            big = at_scale(bs, torch, W, fill_pool_device, dev, opts, peaks)
            detail["at_scale_4L"] = big
            if "skipped" not in big:
                roofline.update({"at4L_pack_frac_of_8TBs": big["frac_of_nominal_8TBs"],
                                 "at4L_unpack_frac_of_8TBs": round(big["unpack_achieved"] / 8000, 4),
                                 "at4L_serialize_frac_of_8TBs": big["serialize_frac_of_8TBs"],
                                 "at4L_deserialize_frac_of_8TBs": big["deserialize_frac_of_8TBs"],
                                 "at4L_stream_GB": round(big["stream_bytes"] / 1e9, 3), "at4L_pack_frac": big["frac"],
                                 "at4L_unpack_frac": big["unpack_frac"], "at4L_n_blocks": big["n_blocks"]})
        except Exception as ex:
            detail["at_scale_4L"] = {"error": repr(ex)}

    ms_g, units_g = aggregate(step_ms, 2 * total, world, dev, ready)
    sampler.stop()
    if rank == 0:
        fused = (not v2) and args.variant != 1 and max(-(-bset.n_blocks // 1024), -(-bset.n_tensors // 1024)) <= sm_count(torch, dev)
        for wl, row in (detail.get("small_sets") or {}).items():   # config1 / config2 latencies, flat
            tgt = e2e if e2e is not None else roofline
            for k in ("serialize_us", "deserialize_us", "plain_copy_us"):
                tgt[f"cfg{wl[-1]}_{k}"] = row[k]
        detail["roofline_text"] = {k: v for k, v in roofline.items() if isinstance(v, (str, list, dict))}
        detail["e2e_text"] = {k: v for k, v in (e2e or {}).items() if isinstance(v, (str, list, dict))}
        roofline, e2e = ordered_for_record(roofline, ROOFLINE_FIRST), ordered_for_record(e2e, E2E_FIRST)
        line = {"metric": METRIC, "value": round(units_g / (ms_g * 1e-3) / 1e9, 3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms_g, 4), "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
                "config": with_elem(workload_config(args.workload, bset, total, args.format), args.elem), "clocks": clocks,
                "gpu_launches": (2 if fused else (8 if v2 else 4)) * args.steps, "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu,
                "detail": detail}
        print(json.dumps(line), flush=True)
    if ready:
        dist.destroy_process_group()


def sm_count(torch, dev):
    return torch.cuda.get_device_properties(dev).multi_processor_count


AB_SETTINGS = [
    # name, opts.  `tune` bits: 8 = round 1's static round-robin deal of the tiles, 0x1000 = block table two iterations ahead,
    # 1 / 2 = L2 evict_first on the bulk loads / stores; `pace` = target HBM traffic of the launch in GB/s
    ("default", None),
    ("counter 48K x3 x1", dict(tile_bytes=49152, stages=3, warps=1)),
    ("static  48K x3 x1 (round 1 pack)", dict(tile_bytes=49152, stages=3, warps=1, tune=8)),
    ("counter 32K x4 x1", dict(tile_bytes=32768, stages=4, warps=1)),
    ("static  32K x4 x1 (round 1 unpack)", dict(tile_bytes=32768, stages=4, warps=1, tune=8)),
    ("counter 40K x3 x1", dict(tile_bytes=40960, stages=3, warps=1)),
    ("static  40K x3 x1", dict(tile_bytes=40960, stages=3, warps=1, tune=8)),
    ("counter 64K x3 x1", dict(tile_bytes=65536, stages=3, warps=1)),
    ("static  64K x3 x1", dict(tile_bytes=65536, stages=3, warps=1, tune=8)),
    ("counter 48K x4 x1", dict(tile_bytes=49152, stages=4, warps=1)),
    ("static  48K x4 x1", dict(tile_bytes=49152, stages=4, warps=1, tune=8)),
    ("counter 16K x3 x3 (small-set shape)", dict(tile_bytes=16384, stages=3, warps=3)),
    ("static  16K x3 x3", dict(tile_bytes=16384, stages=3, warps=3, tune=8)),
    ("counter 24K x4 x2", dict(tile_bytes=24576, stages=4, warps=2)),
    ("static  24K x4 x2", dict(tile_bytes=24576, stages=4, warps=2, tune=8)),
    ("counter 16K x4 x2", dict(tile_bytes=16384, stages=4, warps=2)),
    ("static  16K x4 x2", dict(tile_bytes=16384, stages=4, warps=2, tune=8)),
    ("counter 48K x3 x1, table 2 ahead", dict(tile_bytes=49152, stages=3, warps=1, tune=0x1000)),
    ("counter 48K x3 x1, evict_first loads", dict(tile_bytes=49152, stages=3, warps=1, tune=1)),
    ("counter 48K x3 x1, evict_first stores", dict(tile_bytes=49152, stages=3, warps=1, tune=2)),
    ("counter 48K x3 x1, evict_first both", dict(tile_bytes=49152, stages=3, warps=1, tune=3)),
] + [(f"static  32K x4 x1, table 2 ahead, paced {r}", dict(tile_bytes=32768, stages=4, warps=1, tune=0x1008, pace=r))
     for r in (6300, 6500, 6600, 6700, 6800, 6900, 7000, 7100)] \
  + [(f"counter 32K x4 x1, table 2 ahead, paced {r}", dict(tile_bytes=32768, stages=4, warps=1, tune=0x1000, pace=r))
     for r in (6500, 6700, 6900, 7100)]


def ab_table(bs, torch, time_pack, time_unpack, total, rounds=3):
    """A/B table of the pack and unpack kernels alone on the resident workload (profiles/r02_summary.md): every setting of
    AB_SETTINGS, `rounds` interleaved passes, HBM GB/s = 2 * stream bytes / time per launch."""
    rows = {name: {"pack": [], "unpack": []} for name, _ in AB_SETTINGS}
    for _ in range(rounds):
        for name, o in AB_SETTINGS:
            o2 = None if o is None else dict(variant=bs.VARIANT_TMA, **o)
            rows[name]["pack"].append(round(2 * total / time_pack(o2) / 1e6, 1))
            rows[name]["unpack"].append(round(2 * total / time_unpack(o2) / 1e6, 1))
    return [{"setting": name, "opts": o, "pack_GBs": rows[name]["pack"], "unpack_GBs": rows[name]["unpack"]} for name, o in AB_SETTINGS]


def bulk_copy_ceiling(bs, torch, pool, stream, dev, opts, cs, n):
    """In-run ceiling of the mover: the pack kernel on ONE contiguous fp64 block as large as the workload's stream — every
    tile is one cp.async.bulk load and one cp.async.bulk store, no scatter.  Reuses the workload's pool as the block and its
    stream buffer as the destination (both are re-created by the next serialize)."""
    import workloads as W
    nbytes = min(pool.numel(), stream.numel() - 4096) // (1 << 20) * (1 << 20)
    rows = nbytes // 8 // 32768
    tensors = np.zeros(1, W.TENSOR_REC_DTYPE)
    tensors["rank"], tensors["n_blocks"], tensors["sign"] = 2, 1, (-1, 1, 0, 0)
    one = bs.DeviceSet.from_host(tensors, np.zeros((1, 3, 2), np.int32), np.array([[rows, 32768, 1]], np.uint32),
                                 np.array([pool.data_ptr()], np.uint64), dev)
    w1 = bs.Workspace(1, 1, stream.numel(), dev)
    hb1, tot1 = bs.serialized_size(one.desc, w1.ptr, w1.nbytes, cs)
    assert tot1 <= stream.numel()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(2):
        bs.serialize_range(one.desc, stream.data_ptr(), 0, tot1, False, w1.ptr, w1.nbytes, w1.result_ptr, opts, cs)
    torch.cuda.synchronize()
    a.record()
    for _ in range(n):
        bs.serialize_range(one.desc, stream.data_ptr(), 0, tot1, False, w1.ptr, w1.nbytes, w1.result_ptr, opts, cs)
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / n
    # and the runtime's own device-to-device copy of the same bytes (what MEASURED_PEAKS.json's figure is, on this box, now)
    dst = stream[:tot1 - hb1]
    src = pool[:tot1 - hb1]
    for _ in range(2):
        dst.copy_(src)
    torch.cuda.synchronize()
    a.record()
    for _ in range(n):
        dst.copy_(src)
    b.record()
    torch.cuda.synchronize()
    ms_rt = a.elapsed_time(b) / n
    return {"bulk_copy_GBs": round(2 * tot1 / ms / 1e6, 1), "bulk_copy_bytes": int(tot1),
            "bulk_copy_what": "this run: bs::move_tma_kernel<pack> on ONE contiguous block of that many bytes (pure cp.async.bulk copy)",
            "runtime_d2d_copy_GBs": round(2 * (tot1 - hb1) / ms_rt / 1e6, 1)}


# The driver's record keeps the first 24 SCALAR keys of roofline / e2e / cpu_baseline (nested dicts and lists are dropped,
# strings cut): every bar the north_star states, at the benchmark's size and at the sizes BASELINE.json states, and one
# number per SURVEY §8(f) row go first, flat; everything else follows and is repeated in `detail`.
ROOFLINE_FIRST = ["bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "unpack_frac", "frac_of_nominal_8TBs",
                  "unpack_frac_of_8TBs", "serialize_frac_of_8TBs", "deserialize_frac_of_8TBs", "frac_of_bulk_copy",
                  "unpack_frac_of_bulk_copy", "at4L_pack_frac_of_8TBs", "at4L_unpack_frac_of_8TBs", "at4L_serialize_frac_of_8TBs",
                  "at4L_deserialize_frac_of_8TBs", "at4L_stream_GB", "v2_serialize_frac_of_8TBs", "a8_serialize_frac_of_8TBs",
                  "f32_serialize_frac_of_8TBs", "rank4_serialize_frac_of_8TBs", "pkg1MiB_emit_frac_of_8TBs"]
E2E_FIRST = ["value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "offload_frac_of_pinned_d2h",
             "prefetch_frac_of_pinned_h2d", "duplex_frac_of_bidirectional_memcpy", "exposed_io_frac_save", "exposed_io_frac_load",
             "exposed_io_r", "at3L_exposed_io_frac_save", "at3L_exposed_io_frac_load", "at3L_sustained_pcie_GBs_save",
             "at3L_sustained_pcie_GBs_load", "at3L_stream_GB", "sweep_speedup_queue_over_sync_io", "cfg2_serialize_us",
             "cfg2_deserialize_us", "cfg2_plain_copy_us", "cfg1_serialize_us", "cfg1_deserialize_us", "cfg1_plain_copy_us",
             "offload_pcie_GBs"]


def ordered_for_record(d, first):
    """The keys of `first` that `d` has, in that order, then d's other scalars, then its strings / lists / dicts."""
    if d is None:
        return None
    scalar = lambda v: v is None or isinstance(v, (int, float, bool))
    out = {k: d[k] for k in first if k in d}
    out.update({k: v for k, v in d.items() if k not in out and scalar(v)})
    out.update({k: v for k, v in d.items() if k not in out})
    return out


def variant_legs(bs, torch, W, fill_pool_device, dev, opts, bset, addr, stream, opool, cs, reps=3):
    """One whole-call number per SURVEY §8(f) variant on THIS workload's blocks (same pool, same launch defaults): wire format
    v2 (structure-shared layers), unpadded align = 8, f32 elements; and order-4 tensors (wire format v3) on a 1.4 GB tree set
    of its own.  Returns (flat scalars for the roofline dict, detail).  frac_of_8TBs = 2 * stream bytes / time / 8 TB/s."""
    flat, det = {}, {}

    def timed(fn):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    def leg(tag, ser, deser, ws, total):
        s_ms = timed(ser)
        d_ms = timed(deser)
        r = ws.read_result()
        if r["status"] != bs.OK or r["total_bytes"] != total:
            raise RuntimeError(f"variant {tag}: {r}")
        flat[f"{tag}_serialize_frac_of_8TBs"] = round(2 * total / s_ms / 1e6 / 8000, 4)
        flat[f"{tag}_deserialize_frac_of_8TBs"] = round(2 * total / d_ms / 1e6 / 8000, 4)
        det[tag] = {"stream_bytes": int(total), "serialize_ms": round(s_ms, 4), "deserialize_ms": round(d_ms, 4),
                    "serialize_hbm_GBs": round(2 * total / s_ms / 1e6, 1), "deserialize_hbm_GBs": round(2 * total / d_ms / 1e6, 1)}

    cap = stream.numel()
    for tag, dtype, e in (("a8", bs.F64 | bs.ALIGN8, 8), ("f32", bs.F32, 4)):
        try:
            dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, addr, dev, dtype=dtype)
            ws = bs.Workspace(bset.n_tensors, bset.n_blocks, cap, dev)
            _, total = bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs)
            need = int(((bset.nelems * e + 255) // 256 * 256).sum())
            out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, dev)
            assert total <= cap and need <= opool.numel()
            leg(tag, lambda: bs.serialize(dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs),
                lambda: bs.deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                                       ws.result_ptr, opts, cs), ws, total)
            del dset, ws, out
        except Exception as ex:
            det[tag] = {"error": repr(ex)}
    try:
        lv = W.layered_view(bset)
        counts = (len(lv["structs"]), lv["dim"].shape[0], bset.n_tensors, bset.n_blocks)
        lset = bs.DeviceLayeredSet.from_host(lv["structs"], lv["layers"], lv["qn"], lv["dim"], addr, dev)
        ws = bs.Workspace(0, 0, cap, dev, layered=counts)
        _, total = bs.layered_serialized_size(lset.desc, ws.ptr, ws.nbytes, cs)
        need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
        out = bs.DeviceLayeredSet.empty(*counts, dev)
        assert total <= cap and need <= opool.numel()
        leg("v2", lambda: bs.layered_serialize(lset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs),
            lambda: bs.layered_deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr,
                                           ws.nbytes, ws.result_ptr, opts, cs), ws, total)
        del lset, ws, out
    except Exception as ex:
        det["v2"] = {"error": repr(ex)}
    try:
        tset = W.make_tree_set("tree-1.4GB", 8, D=600, S=12, n_nodes=6, n_ops=13)
        tpool, taddr = fill_pool_device(tset, dev)
        dset = bs.DeviceSet.from_host(tset.tensors, tset.qn, tset.dim, taddr, dev, dtype=bs.F64 | bs.RANK4)
        ws = bs.Workspace(tset.n_tensors, tset.n_blocks, cap, dev)
        _, total = bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs)
        need = int(((tset.nelems * 8 + 255) // 256 * 256).sum())
        out = bs.DeviceSet.empty(tset.n_tensors, tset.n_blocks, dev, rank4=True)
        assert total <= cap and need <= opool.numel()
        leg("rank4", lambda: bs.serialize(dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs),
            lambda: bs.deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes,
                                   ws.result_ptr, opts, cs), ws, total)
        det["rank4"]["set"] = f"order-4 tree set D=600, 12 sectors, 6 nodes + 13 operators: {tset.n_blocks} blocks"
        del tpool, dset, ws, out
    except Exception as ex:
        det["rank4"] = {"error": repr(ex)}
    return flat, det


def at_scale(bs, torch, W, fill_pool_device, dev, opts, peaks, name="4L", steps=5):
    """Pack / unpack kernels and whole calls on workload 4L (42.5 GB stream, 3.3 M blocks: BASELINE.json configs[3]'s stated total)."""
    bset = W.make_config(name)
    need_dev = int(bset.pool_bytes) + 2 * (bset.data_bytes + 64 * bset.n_blocks + (64 << 20)) + (1 << 30)
    free_dev, _ = torch.cuda.mem_get_info()
    if need_dev > free_dev:
        return {"skipped": f"workload {name} needs {need_dev / 1e9:.0f} GB of HBM, {free_dev / 1e9:.0f} GB are free"}
    cs = bs.current_stream()
    pool, addr = fill_pool_device(bset, dev)
    dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, addr, dev)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, bset.data_bytes + 16 * bset.n_blocks + bs.header_bytes(bset.n_tensors, bset.n_blocks), dev)
    hb, total = bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs)
    stream = torch.empty(total, dtype=torch.uint8, device=dev)
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    opool = torch.empty(need, dtype=torch.uint8, device=dev)
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, dev)

    def ser():
        bs.serialize(dset.desc, stream.data_ptr(), total, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)

    def deser():
        bs.deserialize(stream.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs)

    def timed(fn, n=steps):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    for _ in range(3):
        ser()
        deser()
    if ws.read_result()["status"] != bs.OK:
        raise RuntimeError(f"at_scale warm-up: {ws.read_result()}")
    ser_ms, des_ms = timed(ser), timed(deser)
    ser()
    pack_ms = timed(lambda: bs.serialize_range(dset.desc, stream.data_ptr(), 0, total, False, ws.ptr, ws.nbytes, ws.result_ptr, opts, cs))
    deser()
    unpack_ms = timed(lambda: bs.deserialize_range(stream.data_ptr(), 0, total, stream.data_ptr(), out.desc, bs.LAYOUT_POOL, ws.ptr,
                                                   ws.nbytes, opts, cs))
    if ws.read_result()["status"] != bs.OK:
        raise RuntimeError(f"at_scale: {ws.read_result()}")
    algo_p, algo_u = 2 * total + 52 * bset.n_blocks, 2 * total + 64 * bset.n_blocks
    pk, hbm = peaks["hbm_gbs"], lambda ms: 2 * total / ms / 1e6
    return {"workload": f"config 4L: D={bset.meta['D']}, {bset.meta['S']} sectors, {bset.meta['n_ops']} operators + {bset.meta['n_site']} "
                        "site tensors (configs[3] with the operator count scaled to the 40-60 GB it states, SURVEY §8(d) R1)",
            "stream_bytes": int(total), "n_tensors": bset.n_tensors, "n_blocks": bset.n_blocks, "steps": steps,
            "pack_kernel_ms": round(pack_ms, 3), "achieved": round(algo_p / pack_ms / 1e6, 1), "frac": round(algo_p / pack_ms / 1e6 / pk, 4),
            "frac_of_nominal_8TBs": round(algo_p / pack_ms / 1e6 / 8000, 4),
            "unpack_kernel_ms": round(unpack_ms, 3), "unpack_achieved": round(algo_u / unpack_ms / 1e6, 1),
            "unpack_frac": round(algo_u / unpack_ms / 1e6 / pk, 4),
            "serialize_ms": round(ser_ms, 3), "deserialize_ms": round(des_ms, 3),
            "serialize_hbm_GBs": round(hbm(ser_ms), 1), "deserialize_hbm_GBs": round(hbm(des_ms), 1),
            "serialize_frac_of_8TBs": round(hbm(ser_ms) / 8000, 4), "deserialize_frac_of_8TBs": round(hbm(des_ms) / 8000, 4),
            "value_GBs": round(2 * total / (ser_ms + des_ms) / 1e6, 1)}


def config5(args, dev, opts, name="3", full=True):
    """SURVEY §8(d) config-5 protocol on config 3 (or 3L, the total BASELINE.json states for it): T_c (stand-in alone), T_io
    (offload alone), T_both (together).  full=False: the headline ratio r = 1.25 only, both directions, no sweeps."""
    import torch

    import paper_2412_04676_b200 as bs
    import workloads as W
    from workloads.device import StandInContraction, fill_pool_device

    bset = W.make_config(name)
    pool, addr = fill_pool_device(bset, dev)
    dset = bs.DeviceSet.from_host(bset.tensors, bset.qn, bset.dim, addr, dev)
    ws = bs.Workspace(bset.n_tensors, bset.n_blocks, bset.data_bytes + 16 * bset.n_blocks + (64 << 20) + bs.header_bytes(bset.n_tensors, bset.n_blocks), dev)
    cs = bs.current_stream()
    hb, total = bs.serialized_size(dset.desc, ws.ptr, ws.nbytes, cs)
    host = torch.empty(total, dtype=torch.uint8, pin_memory=True)
    eng = bs.Engine(bset.n_tensors, bset.n_blocks, total, chunk_bytes=args.chunk_mb << 20, n_staging=2, opts=opts)
    work = StandInContraction(bset, addr, dev, max_items=args.standin_items)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def t_io():
        a.record()
        t = eng.offload_async(dset.desc, total, host.data_ptr(), total, cs)
        t.stream_wait(cs)
        b.record()
        st = t.wait()
        torch.cuda.synchronize()
        assert st["status"] == 0
        return a.elapsed_time(b), st

    def t_c(reps):
        a.record()
        work.run(reps)
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    def t_both(reps):
        a.record()
        t = eng.offload_async(dset.desc, total, host.data_ptr(), total, cs)
        work.run(reps)
        t.stream_wait(cs)
        b.record()
        st = t.wait()
        torch.cuda.synchronize()
        assert st["status"] == 0
        return a.elapsed_time(b), st

    t_io()
    io_ms = min(t_io()[0] for _ in range(3))
    one = min(t_c(1) for _ in range(2))
    res = {"workload": f"config {name} (BASELINE.json configs[2]) offloaded through bs_offload_async", "stream_bytes": int(total),
           "T_io_ms": round(io_ms, 3), "standin_ms_per_rep": round(one, 3), "sweep": []}
    for r in ((1.25, 0.5, 1.0, 1.5, 2.0) if full else (1.25,)):
        reps = max(1, int(round(r * io_ms / one)))
        tc = min(t_c(reps) for _ in range(2))
        both = [t_both(reps) for _ in range(3)]
        tb, st = min(both, key=lambda x: x[0])
        row = {"r_target": r, "r_actual": round(tc / io_ms, 3), "T_c_ms": round(tc, 3), "T_both_ms": round(tb, 3),
               "exposed_io_frac": round(max(0.0, tb - tc) / tb, 4), "hidden_frac": round(1 - max(0.0, tb - tc) / io_ms, 4),
               "sustained_pcie_GBs": round(st["bytes"] / st["dma_ms"] / 1e6, 2)}
        res["sweep"].append(row)
    res["headline"] = res["sweep"][0]

    # ---- the same protocol for the load direction ("same again for prefetch with BW_h2d"): the stream just
    # offloaded is prefetched into a second pool while the stand-in contraction runs on the operators ----
    need = int(((bset.nelems * 8 + 255) // 256 * 256).sum())
    out = bs.DeviceSet.empty(bset.n_tensors, bset.n_blocks, dev)
    opool = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)

    def p_io():
        a.record()
        t = eng.prefetch_async(host.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)
        b.record()          # the consumer stream waits on the ticket's event (checkpoint): b is behind the load
        st = t.wait()
        torch.cuda.synchronize()
        assert st["status"] == 0
        return a.elapsed_time(b), st

    side = torch.cuda.Stream()

    def p_both(reps):
        # the load's consumer is a side stream (whoever needs the loaded blocks); the contraction runs on the compute stream
        a.record()
        side.wait_stream(torch.cuda.current_stream())
        t = eng.prefetch_async(host.data_ptr(), total, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, side.cuda_stream)
        work.run(reps)
        torch.cuda.current_stream().wait_stream(side)
        b.record()
        st = t.wait()
        torch.cuda.synchronize()
        assert st["status"] == 0
        return a.elapsed_time(b), st

    p_io()
    pio_ms = min(p_io()[0] for _ in range(3))
    pre = {"T_io_ms": round(pio_ms, 3), "sweep": []}
    for r in ((1.25, 0.5, 1.0, 2.0) if full else (1.25,)):
        reps = max(1, int(round(r * pio_ms / one)))
        tc = min(t_c(reps) for _ in range(2))
        both = [p_both(reps) for _ in range(3)]
        tb, st = min(both, key=lambda x: x[0])
        pre["sweep"].append({"r_target": r, "r_actual": round(tc / pio_ms, 3), "T_c_ms": round(tc, 3), "T_both_ms": round(tb, 3),
                             "exposed_io_frac": round(max(0.0, tb - tc) / tb, 4),
                             "hidden_frac": round(1 - max(0.0, tb - tc) / pio_ms, 4),
                             "sustained_pcie_GBs": round(st["bytes"] / st["dma_ms"] / 1e6, 2)})
    pre["headline"] = pre["sweep"][0]
    res["prefetch"] = pre
    eng.destroy()
    if not full:
        return res

    # ---- a sweep, PAPER Fig 3: every DMRG step loads the environment block of the next step, computes, and saves the
    # block it renormalized.  Synchronous IO (Fig 3(a): compute halts for every save and load) against the queue
    # (Fig 3(c): the load of step i+1 and the save of step i-1 run behind the compute of step i, checkpoints = events).
    # The compute is the stand-in contraction at 1.25 x the duplex IO time of one step. ----
    try:
        n_steps, n_keys = 12, 4   # 4 scratch slots: a block is loaded two steps after it was saved, as in a sweep that returns to it
        hosts = [host] + [torch.empty(total, dtype=torch.uint8, pin_memory=True) for _ in range(n_keys - 1)]
        q = bs.Queue(bset.n_tensors, bset.n_blocks, total, chunk_bytes=args.chunk_mb << 20, n_staging=2, opts=opts)
        for k in range(n_keys):
            q.save(k, dset.desc, total, hosts[k].data_ptr(), total, cs)
        q.drain()

        def duplex_io():
            a.record()
            q.save(0, dset.desc, total, hosts[0].data_ptr(), total, cs)
            q.load(1, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)
            q.checkpoint(0, cs)
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b)

        duplex_io()
        io_step = min(duplex_io() for _ in range(3))
        reps = max(1, int(round(1.25 * io_step / one)))
        tc_step = min(t_c(reps) for _ in range(2))

        def sweep_sync():
            a.record()
            for i in range(n_steps):
                q.load((i + 1) % n_keys, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)
                q.wait((i + 1) % n_keys)                 # compute halts until the environment block is in memory
                work.run(reps)
                q.save(i % n_keys, dset.desc, total, hosts[i % n_keys].data_ptr(), total, cs)
                q.wait(i % n_keys)                       # ... and until the renormalized block is saved
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b)

        def sweep_async():
            a.record()
            q.load(1, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, side.cuda_stream)
            for i in range(n_steps):
                torch.cuda.current_stream().wait_stream(side)        # checkpoint: the environment block of step i is here
                if i + 1 < n_steps:                                    # next step's environment block, behind this compute
                    side.wait_stream(torch.cuda.current_stream())
                    q.load((i + 2) % n_keys, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, side.cuda_stream)
                work.run(reps)
                q.save(i % n_keys, dset.desc, total, hosts[i % n_keys].data_ptr(), total, cs)   # runs behind the next compute
            for k in range(n_keys):
                q.checkpoint(k, cs)
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b)

        sweep_sync(); sweep_async()
        t_sync = min(sweep_sync() for _ in range(2))
        t_async = min(sweep_async() for _ in range(2))
        for k in range(n_keys):
            if q.wait(k)["status"]:
                raise RuntimeError("queue status")
        res["sweep_fig3"] = {"steps": n_steps, "bytes_saved_and_loaded_per_step": int(2 * total),
                             "compute_ms_per_step": round(tc_step, 3), "duplex_io_ms_per_step": round(io_step, 3),
                             "sync_io_ms": round(t_sync, 3), "queue_ms": round(t_async, 3),
                             "compute_only_ms": round(n_steps * tc_step, 3),
                             "speedup_queue_over_sync": round(t_sync / t_async, 3),
                             "exposed_io_frac_queue": round(max(0.0, t_async - n_steps * tc_step) / t_async, 4),
                             "io_frac_sync": round(max(0.0, t_sync - n_steps * tc_step) / t_sync, 4),
                             "ends_ms": round(io_ms + pio_ms, 3),
                             "exposed_io_frac_queue_without_ends": round(max(0.0, t_async - n_steps * tc_step - io_ms - pio_ms) / t_async, 4),
                             "note": "the first load and the last save of a sweep have no compute to hide behind (ends_ms = one "
                                     "save alone + one load alone)"}
        # ---- the storage tier (PAPER L85 step (2): the stream goes on to a file; context for the paper's 2.15 GB/s
        # synchronous save and 1.12 GB/s per-SSD write, L154 / L168): whatever disk this box has under the temp dir ----
        try:
            import tempfile
            with tempfile.TemporaryDirectory() as td:
                path = os.path.join(td, "block.bs")
                q.save(0, dset.desc, total, hosts[0].data_ptr(), total, cs)
                q.spill(0, path)
                sp = q.io_wait(0)
                q.fill(9, path, hosts[1].data_ptr(), total)
                fl = q.io_wait(9)
                q.load(9, out.desc, opool.data_ptr(), need, bs.LAYOUT_POOL, cs)
                ok = q.wait(9)["status"] == 0 and sp["status"] == 0 and fl["status"] == 0
                res["storage_tier"] = {"ok": bool(ok), "bytes": int(sp["bytes"]),
                                       "spill_write_GBs": round(sp["bytes"] / max(sp["seconds"], 1e-9) / 1e9, 2),
                                       "fill_read_GBs_page_cache_warm": round(fl["bytes"] / max(fl["seconds"], 1e-9) / 1e9, 2),
                                       "note": "one host IO thread, plain write() / read() in 64 MiB pieces, no fsync; the file "
                                               "was just written, so the read comes from the page cache"}
        except Exception as ex:
            res["storage_tier"] = {"error": repr(ex)}
        q.destroy()
    except Exception as ex:
        res["sweep_fig3"] = {"error": repr(ex)}
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mine", choices=["mine", "reference"])
    ap.add_argument("--workload", default="4", choices=["1", "2", "3", "4", "3L", "4L"])
    ap.add_argument("--elem", default="f64", choices=sorted(ELEM), help="element type of the blocks (wire format v1); "
                    "other than f64: kernels only (no e2e / config-5 / cpu legs)")
    ap.add_argument("--format", default="v1", choices=["v1", "v2"],
                    help="wire format: v1 (one block record per block) or v2 (structure-shared layers, NEXT-1)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--tile-bytes", type=int, default=0)
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--stages", type=int, default=0)
    ap.add_argument("--warps", type=int, default=0)
    ap.add_argument("--tune", type=lambda v: int(v, 0), default=0,
                    help="TMA variant experiment bits: 1 = L2 evict_first on bulk loads, 2 = on bulk stores, 8 = round 1's static "
                         "round-robin deal of the tiles, 0x10 = tiles from the counter whatever the size, 0x100..0xf00 = at most that "
                         "many tiles loading beside the one being stored, 0x1000 = block table fetched two iterations ahead, "
                         "0x20 = unpack asks the next stream tile into L2")
    ap.add_argument("--ab", type=int, default=0, metavar="ROUNDS",
                    help="also time the pack / unpack kernels alone under the settings of AB_SETTINGS, ROUNDS interleaved passes "
                         "(detail.ab; the A/B tables of profiles/)")
    ap.add_argument("--pace", type=int, default=0, help="TMA variant: pace the launches at this many GB/s of HBM traffic (experiments)")
    ap.add_argument("--fuse", type=int, default=0, help="0 = by size, 1 = size pass and movement as separate launches, 2 = one fused launch")
    ap.add_argument("--chunk-mb", type=int, default=256)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--sample-mb", type=float, default=400.0, help="payload of the oracle's bounded sample")
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--standin-items", type=int, default=60000)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-packages", action="store_true")
    ap.add_argument("--no-comparator", action="store_true", help="skip the one-copy-per-block library comparator of the pack step")
    ap.add_argument("--no-small", action="store_true", help="skip the latency numbers of configs 1 and 2")
    ap.add_argument("--no-queue", action="store_true", help="e2e: offload then prefetch only, no duplex queue leg")
    ap.add_argument("--no-config5", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-ceiling", action="store_true", help="skip the in-run bulk-copy ceiling of the roofline leg")
    ap.add_argument("--no-at-scale", action="store_true", help="skip the at4L_* (workload 4L, 42.5 GB) and at3L_* (11 GB) numbers")
    ap.add_argument("--no-variants", action="store_true", help="skip the per-variant numbers (v2, align 8, f32, rank 4) of the roofline dict")
    ap.add_argument("--no-threads-sweep", action="store_true", help="skip cpu_baseline.threads_sweep")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "mine" else args.warmup
    if args.elem != "f64":   # the e2e / config-5 / cpu legs and wire format v2 are fp64; other element types time the kernels
        if args.format != "v1" or args.impl != "mine":
            ap.error("--elem other than f64 needs --format v1 --impl mine")
        args.no_e2e = args.no_config5 = args.no_cpu = args.no_packages = True
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mine(args)


if __name__ == "__main__":
    main()
