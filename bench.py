#!/usr/bin/env python
"""bench.py -- throughput of the phase-space source hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4|5] [--impl ours|reference]

One "step" is one pass of the whole hot path over one synthetic
phase-space: psl_reset -> psl_load_chunk x n -> psl_build_batches (-> per-beam builds in INDEX mode).
The default workload is BASELINE.json configs[1] (config 2: 1e7 records, 1e6-record chunks, 3 x 64 keys).
Prints ONE JSON line:
  value        particles/s, whole job, inputs already resident in HBM when the timed region starts
  e2e          the same metric through the C-ABI with PINNED HOST buffers: the H2D copy of every chunk and
               the D2H read of counts[] / offsets[] / statistics are inside the timed region
  roofline     dominant kernel: algorithmic bytes per launch / its average duration (CUDA events recorded
               by the library on its own stream during the timed steps) against the measured HBM copy rate
  cpu_baseline the oracle, as it stands, timed on this box's host cores (rank 0, N=1 only)
With N > 1 (torchrun) every rank runs the same workload shape on its own shard of the record stream
(records [rank*n, (rank+1)*n)); the path has no exchange step, so there is no collective in the data path
("scaling": "weak").  --impl reference times the oracle on the host cores (the reference arm of this tier).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "phase-space particles/s decoded+binned+sorted"
UNIT = "particles/s"
RECORD_BYTES = 28
SOA_BYTES = 32  # E x y u v w wt src_index per survivor


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--records", type=int, default=0, help="override the number of records (0 = the config's own)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def measured_peaks():
    """(hbm GB/s, source).  MEASURED_PEAKS.json is driver-written; the fallback is B200_PROFILING.md's."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML while the timed regions run"""

    def __init__(self, index: int, period_s: float = 0.004):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.max_mhz = period_s, [], set(), None
        self._stop_evt = threading.Event()
        self._active = threading.Event()
        self.h = None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    NAMES = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
             0x80: "hw_power_brake_slowdown"}

    def run(self):
        if self.h is None:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            if self._active.is_set():
                try:
                    self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                    for bit, name in self.NAMES.items():
                        if r & bit:
                            self.reasons.add(name)
                except Exception:
                    pass
            time.sleep(self.period)

    def region(self, on: bool):
        (self._active.set if on else self._active.clear)()

    def finish(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=1.0)
        return {"sm_mhz": int(statistics.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------------
# workload
# ------------------------------------------------------------------------------------------------------
def workload_for(args):
    import workloads as W

    w = W.config(args.config, args.records or None)
    if args.records and args.config in (2, 5):
        # keep the chunk size of the full-size config when it still divides the stream into >= 2 chunks
        full = W.config(args.config).chunk_records
        if full and full < args.records:
            w.chunk_records = full
    return w


def describe(w, n_gpus, extra=None):
    g = w.grid
    c = {
        "workload": w.name, "baseline_config_index": int(w.name[3]), "records_per_gpu": w.n_records,
        "record_bytes": RECORD_BYTES, "chunk_records": w.chunk_records or w.n_records,
        "keys": w.n_keys, "mode": "index" if w.mode == 1 else "onthefly", "beams": len(w.beams),
        "n_ebins": g["n_ebins"], "position_bins": [g["n_xbins"], g["n_ybins"]],
        "sharding": "record-index ranges per rank, no data-path collective" if n_gpus > 1 else "single GPU",
        "l2_policy": "%s (%.0f MB of records read and up to %.0f MB of output written per step vs 126 MB L2)"
                     % ("inputs larger than L2" if w.n_records * RECORD_BYTES > 126e6 else "SMALLER THAN L2: not a valid timing",
                        w.n_records * RECORD_BYTES / 1e6, w.n_records * SOA_BYTES / 1e6),
    }
    if extra:
        c.update(extra)
    return c


def oracle_step(orc, rec, beams):
    """what one step computes, by the definition: filter + stable sort, once per beam"""
    ns = 0
    for b in beams:
        ns += orc.build(rec, b)["n_survivors"]
    return ns


def time_oracle(w, rank_first, budget_s=10.0, max_sample=20_000_000):
    """the oracle as it stands on a bounded sample of the workload; returns (particles/s, description)"""
    import workloads as W
    from oracle import psl_oracle as O

    n = min(w.n_records, max_sample)
    rec = W.generate(w.gen, rank_first, n)
    orc = O.Oracle(w.grid, w.geometry, flags=w.flags)
    reps, t_total = 0, 0.0
    while reps < 1 or (t_total < budget_s and reps < 64):
        t0 = time.perf_counter()
        oracle_step(orc, rec, w.beams)
        t_total += time.perf_counter() - t0
        reps += 1
    sample = "%s %d records of %s x %d beam build(s), %d repetition(s), %.1f s of single-thread CPU work" % (
        "all" if n == w.n_records else "the first", n, w.name, len(w.beams), reps, t_total)
    return n * reps / t_total, sample


def time_oracle_all_cores(w, rank_first, n_sample=8_000_000):
    """SURVEY 8(d)'s second CPU line: C independent oracle instances on C contiguous shards of the sample, one per
    host core, run at the same time (the oracle itself stays single-threaded; ctypes drops the GIL in the call)"""
    import threading

    import workloads as W
    from oracle import psl_oracle as O

    cores = os.cpu_count() or 1
    n = min(w.n_records, max(n_sample, min(cores * 200_000, 32_000_000)))
    rec = W.generate(w.gen, rank_first, n)
    per = (n + cores - 1) // cores
    shards = [rec[i * per:min(n, (i + 1) * per)] for i in range(cores) if i * per < n]
    orcs = [O.Oracle(w.grid, w.geometry, flags=w.flags) for _ in shards]
    def work(o, s_):
        for _ in range(reps):
            oracle_step(o, s_, w.beams)

    reps, dt = 1, 0.0
    while True:  # repeat with more repetitions per instance until the run lasts about two seconds
        threads = [threading.Thread(target=work, args=(o, s_)) for o, s_ in zip(orcs, shards)]
        t0 = time.perf_counter()
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        dt = time.perf_counter() - t0
        if dt >= 2.0 or reps >= 256:
            break
        reps = min(256, max(reps * 2, int(reps * 2.5 / max(dt, 1e-3))))
    n *= reps
    return {"value": n / dt, "unit": UNIT, "cores": len(shards), "kind": "oracle",
            "sample": "%d independent single-threaded oracle instances, one per shard of the first %d records of %s, "
                      "%d repetition(s) each, %.1f s wall" % (len(shards), n // reps, w.name, reps, dt)}


def run_reference(args):
    """--impl reference: the oracle on the host cores, on the same config / metric / unit"""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import workloads as W
    from oracle import psl_oracle as O

    w = workload_for(args)
    n = min(w.n_records, 5_000_000)
    rec = W.generate(w.gen, 0, n)
    orc = O.Oracle(w.grid, w.geometry, flags=w.flags)
    for _ in range(min(args.warmup, 3)):
        oracle_step(orc, rec, w.beams)
    steps = max(1, min(args.steps, 30))
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(orc, rec, w.beams)
    dt = time.perf_counter() - t0
    value = n * steps / dt
    sample = "each step = the first %d records of %s, oracle/psl_oracle.c single-threaded" % (n, w.name)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": min(args.warmup, 3), "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": describe(w, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------------
def algorithmic_bytes(cls, n, n_idx, m_sel, n_surv_beams, proj, index_mode=False, compacted=False):
    """algorithmic bytes one step's launches of kernel class `cls` must move"""
    out_b = SOA_BYTES + (8 if proj else 0)
    if cls == "count":
        # one read of every packed record; INDEX mode adds pass B's histogram, which reads the 4-byte key of every
        # keyed record; for a rejecting beam with few keys it also writes the survivors as 32-byte keyed records
        return RECORD_BYTES * n + (4 * n_idx if index_mode else 0) + (32 * n_surv_beams if compacted else 0)
    if cls == "scatter":
        if compacted:
            return 32 * n_surv_beams + out_b * n_surv_beams  # read the compacted survivors, write their SoA
        return RECORD_BYTES * n + out_b * n_surv_beams  # read every record, write the survivors' SoA
    if cls == "index_a":
        return RECORD_BYTES * n + 32 * n_idx          # packed records in, 32-byte keyed records out
    if cls == "index_b":
        return 32 * n_idx + 32 * n_idx                # keyed records in, 7 SoA arrays + the key per slot out
    if cls == "beam":
        return RECORD_BYTES * m_sel + out_b * n_surv_beams  # only the ROI-selected bins are read
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1302_1861_b200 as P
    import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libpsl_b200 has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = workload_for(args)
    n = w.n_records
    first_record = rank * n  # this rank's shard of the stream
    chunks = list(w.chunks())

    # inputs: generated once into pinned host memory (the e2e source), copied once to the device (the resident source)
    host = torch.empty(n * RECORD_BYTES, dtype=torch.uint8).pin_memory()
    W.generate_into(w.gen, first_record, n, host.data_ptr(), threads=os.cpu_count() or 1)
    resident = host.to(dev)
    host_chunks = [host[f * RECORD_BYTES:(f + c) * RECORD_BYTES] for f, c in chunks]
    dev_chunks = [resident[f * RECORD_BYTES:(f + c) * RECORD_BYTES] for f, c in chunks]

    ctx = P.PslContext(w.grid, w.geometry, w.mode, max_records=n, max_host_records=0 if args.no_e2e else n,
                       max_chunks=len(chunks) + 1, flags=w.flags, device=local)
    beams = [None if b is None else ctx.beam(b) for b in w.beams]
    K = w.n_keys
    h_counts = torch.empty(K, dtype=torch.int32).pin_memory()
    h_offsets = torch.empty(K + 1, dtype=torch.int32).pin_memory()
    info = {}

    def step(src_chunks, read_back):
        ctx.reset()
        for c in src_chunks:
            ctx.load_chunk(c)
        n_surv = 0
        for b in beams:
            ctx.build_batches(b)
            if read_back:
                counts, offsets = ctx.get_tables()
                h_counts.copy_(counts, non_blocking=True)
                h_offsets.copy_(offsets, non_blocking=True)
                n_surv += ctx.get_stats()["n_survivors"]  # synchronises: the result is on the host
        return n_surv

    def timed(src_chunks, read_back, steps):
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler.region(True)
        e0.record()
        for _ in range(steps):
            step(src_chunks, read_back)
        e1.record()
        torch.cuda.synchronize()
        sampler.region(False)
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)  # timing only: the slowest rank defines the job
            dist.barrier()
            ms = float(t.item())
        return ms

    sampler = ClockSampler(local)
    sampler.start()

    # ---- device-resident: warm-up, then EXACTLY --steps timed steps --------------------------------------
    for _ in range(max(args.warmup, 3)):
        step(dev_chunks, False)
    torch.cuda.synchronize()
    l0 = ctx.kernel_launches()
    ms = timed(dev_chunks, False, args.steps)
    launches = ctx.kernel_launches() - l0
    # the same steps once more with the library's per-kernel event brackets on (they cost a few microseconds per
    # launch, so they stay out of the timed region above): kernel shares and the roofline of the dominant kernel
    ctx.profile_enable(True)
    ctx.profile_read()
    ms_prof = timed(dev_chunks, False, args.steps)
    prof = ctx.profile_read()
    ctx.profile_enable(False)

    # what the last step produced (sizes the algorithmic bytes)
    st = ctx.get_stats()
    n_idx = n - st["n_invalid"] - st["n_outside_grid"]
    surv_all, m_sel_all = 0, 0
    if len(beams) == 1:
        surv_all = st["n_survivors"]
        m_sel_all = n_idx - st["n_roi_skipped"]
    else:
        for b in beams:
            s = ctx.build_batches(b, want_stats=True)
            surv_all += s["n_survivors"]
            m_sel_all += n_idx - s["n_roi_skipped"]
    info.update(n_valid_in_grid=n_idx, survivors_per_step=surv_all, roi_selected_per_step=m_sel_all)

    # ---- end to end: pinned host chunks in, tables + statistics out, every step ---------------------------
    e2e = None
    n_batches = w.grid["n_types"] * w.grid["n_ebins"]
    # per beam build: counts[K] + offsets[K+1] (read here) + batch offsets + statistics (read by the library);
    # INDEX mode adds the one-off offsets[K+1] copy that drives the ROI segment list
    d2h_bytes = len(beams) * ((2 * K + 1) * 4 + (n_batches + 1) * 4 + 64) + ((K + 1) * 4 if w.mode == 1 else 0)
    if not args.no_e2e:
        # the host-link ceiling, measured here: plain pinned cudaMemcpyAsync of the same chunks into one device buffer
        land = torch.empty(max(c for _, c in chunks) * RECORD_BYTES, dtype=torch.uint8, device=dev)
        for rep_ in range(2):
            torch.cuda.synchronize()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record()
            for hc in host_chunks:
                land[:hc.numel()].copy_(hc, non_blocking=True)
            c1.record()
            torch.cuda.synchronize()
            h2d_peak = n * RECORD_BYTES / (c0.elapsed_time(c1) * 1e-3) / 1e9
        del land
        for _ in range(3):
            step(host_chunks, True)
        e2e_steps = max(3, min(args.steps, 10 if n > 50_000_000 else args.steps))
        ms_e = timed(host_chunks, True, e2e_steps)
        e2e = {"value": world * n * e2e_steps / (ms_e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": n * RECORD_BYTES,
               "d2h_bytes_per_step": d2h_bytes,
               "steps": e2e_steps, "ms_per_step": ms_e / e2e_steps,
               "h2d_gbs": n * RECORD_BYTES * e2e_steps / (ms_e * 1e-3) / 1e9,
               "h2d_peak_gbs": h2d_peak,  # plain pinned copies of the same chunks, same run
               "h2d_frac": n * RECORD_BYTES * e2e_steps / (ms_e * 1e-3) / 1e9 / h2d_peak,
               "source": "pinned host memory, %d chunk(s) per step through psl_load_chunk(PSL_MEM_PINNED)" % len(chunks)}
    clocks = sampler.finish()

    # ---- roofline of the dominant kernel -------------------------------------------------------------------
    peak, peak_src = measured_peaks()
    proj = bool(w.flags & P.OUT_PROJ)
    # ONTHEFLY, K <= 256, a beam that rejects: the histogram kernel compacts the survivors and the scatter reads those
    compacted = (w.mode == 0 and (w.n_keys + 7) // 8 * 8 <= 256 and os.environ.get("PSL_NO_COMPACT") is None
                 and any(b is not None and (b.get("jaws") is not None or (w.flags & P.DROP_ZERO_WEIGHT)) for b in w.beams))
    kernels = {}
    for cls, (tot_ms, brackets) in prof.items():
        if brackets == 0 or cls in ("scan", "other"):
            if brackets:
                kernels[cls] = {"ms_per_step": tot_ms / args.steps, "launches_per_step": brackets / args.steps}
            continue
        per_step_bytes = algorithmic_bytes(cls, n, n_idx, m_sel_all, surv_all, proj, w.mode == 1, compacted)
        kernels[cls] = {"ms_per_step": tot_ms / args.steps, "launches_per_step": brackets / args.steps,
                        "avg_launch_ms": tot_ms / brackets,
                        "algorithmic_bytes_per_step": per_step_bytes,
                        "gbs": per_step_bytes * args.steps / (tot_ms * 1e-3) / 1e9 if tot_ms > 0 else None}
    dom = max((c for c in kernels if "gbs" in kernels[c]), key=lambda c: kernels[c]["ms_per_step"])
    d = kernels[dom]
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            traffic = json.load(f).get(w.name, {}).get(dom)
    except Exception:
        pass
    roofline = {"bound": "hbm", "kernel": dom, "achieved": d["gbs"], "peak": peak, "unit": "GB/s",
                "frac": d["gbs"] / peak, "peak_source": peak_src,
                "frac_of_nominal_8000": d["gbs"] / 8000.0,  # also against the nominal ~8 TB/s
                "bytes_per_launch": d["algorithmic_bytes_per_step"] / d["launches_per_step"],
                "avg_launch_ms": d["avg_launch_ms"], "traffic": traffic,
                "step_frac": sum(k["algorithmic_bytes_per_step"] for k in kernels.values() if "gbs" in k)
                             / (ms / args.steps * 1e-3) / 1e9 / peak,
                "ms_per_step_with_brackets": ms_prof / args.steps}

    if rank == 0:
        line = {
            "metric": METRIC, "value": world * n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": describe(w, world, info), "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "kernels": kernels,
        }
        if world == 1 and not args.no_cpu_baseline:
            v, sample = time_oracle(w, first_record)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                                    "host_cores_available": os.cpu_count(),
                                    "all_cores": time_oracle_all_cores(w, first_record)}
        print(json.dumps(line))
    ctx.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
