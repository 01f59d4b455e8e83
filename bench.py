#!/usr/bin/env python
"""bench.py -- throughput of the phase-space source hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference] [--verify] [--variant 5b]

One "step" is one pass of the whole hot path over one synthetic
phase-space: psl_reset -> psl_load_chunk x n -> psl_build_batches per beam (INDEX mode: the first build also
finalises the PSL index).  The default workload is the largest single-GPU configuration of BASELINE.json,
configs[4] = config 5 (1e9 records = 28 GB in 105 pinned chunks of 268 435 440 bytes, PSL index over 1 228 800
keys, nine IMRT beams); if this box cannot hold it (host or device memory) the run falls back to config 4 and says
so in `config.fallback`.  `--config 2|3|4` time the other configurations.  Prints ONE JSON line:
  value        particles/s, whole job, inputs already resident in HBM when the timed region starts; the timed
               region is a window of EXACTLY --steps steps, repeated (>= 3 windows, >= 0.5 s in all) and the
               MEDIAN window reported (`windows_ms` lists all of them)
  e2e          the same metric through the C-ABI with PINNED HOST buffers: the H2D copy of every chunk and
               the D2H read of counts[] / offsets[] / statistics are inside the timed region
  per_phase    one step cut at its phase boundaries with CUDA events: load (per-chunk histograms), index build,
               every beam
  roofline     dominant kernel: algorithmic bytes per launch / its average duration (CUDA events recorded
               by the library on its own stream during a bracketed repeat of the timed steps) against the measured
               HBM copy rate
  cpu_baseline the oracle, as it stands, timed on this box's host cores (rank 0, N=1 only)
With N > 1 (torchrun) every rank runs the same workload shape on its own shard of the record stream
(records [rank*n, (rank+1)*n)); the path has no exchange step in the data path ("scaling": "weak"); the one
optional exchange of section 8(e) (all-gather of counts[K] -> global slots) runs once over NCCL outside the timed
region and is reported as `exchange_ms`.  --impl reference times the oracle on the host cores (the reference arm
of this tier).
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
KEYED_BYTES = 32  # one record of the PSL index: {key, E, x, y, u, v, wt, src_index}
SOA_BYTES = 32    # E x y u v w wt src_index per survivor


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=0, choices=[0, 1, 2, 3, 4, 5],
                    help="BASELINE.json config (1-based); 0 = the largest one this box holds (5, else 4)")
    ap.add_argument("--records", type=int, default=0, help="override the number of records (0 = the config's own)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-next", action="store_true", help="skip the section-8(f) phase lines (sampling layer / shipments)")
    ap.add_argument("--variant", choices=["5a", "5b"], default="5a",
                    help="config 5 only: 5a = stream once, index on the device, nine beam builds (the default); 5b = "
                         "SURVEY 8(d)'s literal per-beam re-stream of the whole phase-space from pinned host memory")
    ap.add_argument("--verify", action="store_true",
                    help="after the timed regions, check the full-size result against the oracle (streaming counts)")
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
def pick_config(args, world):
    """(config index, fallback note or None).  --config 0: config 5 if this box can hold it, else config 4."""
    if args.config:
        return args.config, None
    if args.records:
        return 5, None
    import workloads as W

    need_host = world * (W.config(5).n_records * RECORD_BYTES + (2 << 30)) + (6 << 30)
    try:
        import psutil

        avail = psutil.virtual_memory().available
        if avail < need_host:
            return 4, "config 5 needs %.0f GB of pinned host memory for %d rank(s); %.0f GB available" % (
                need_host / 1e9, world, avail / 1e9)
    except Exception:
        pass
    try:
        import torch

        if torch.cuda.is_available():
            import paper_1302_1861_b200 as P

            w5 = W.config(5)
            ws = P.workspace_bytes(w5.grid, w5.geometry, w5.mode, w5.n_records, max_chunks=len(list(w5.chunks())) + 1)
            free, _total = torch.cuda.mem_get_info(int(os.environ.get("LOCAL_RANK", "0")))
            need_dev = ws + w5.n_records * RECORD_BYTES + (3 << 30)
            if free < need_dev:
                return 4, "config 5 needs %.0f GB of device memory (workspace + resident copy); %.0f GB free" % (
                    need_dev / 1e9, free / 1e9)
    except Exception:
        pass
    return 5, None


def workload_for(args, world=1):
    import workloads as W

    idx, note = pick_config(args, world)
    w = W.config(idx, args.records or None)
    if args.records and idx in (2, 5):
        # keep the chunk size of the full-size config when it still divides the stream into >= 2 chunks
        full = W.config(idx).chunk_records
        if full and full < args.records:
            w.chunk_records = full
    return w, note


def describe(w, n_gpus, note=None):
    """the `config` object: identical for the CUDA arm and the reference arm"""
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
    if note:
        c["fallback"] = note
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

    n = min(w.n_records, max_sample if len(w.beams) == 1 else max_sample // 4)
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
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return 0
    import workloads as W
    from oracle import psl_oracle as O

    w, note = workload_for(args, world)
    # a bounded sample per step: about a second of single-thread work whatever the number of beams
    n = min(w.n_records, 5_000_000 if len(w.beams) == 1 else 1_000_000)
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
    sample = "each step = the first %d records of %s x %d beam build(s), oracle/psl_oracle.c single-threaded" % (
        n, w.name, len(w.beams))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": min(args.warmup, 3), "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": describe(w, args.gpus, note),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------------
def algorithmic_bytes(cls, n, n_idx, m_sel, n_surv_beams, proj, compacted=False):
    """algorithmic bytes one step's launches of kernel class `cls` must move"""
    out_b = SOA_BYTES + (8 if proj else 0)
    if cls == "count":
        # one read of every packed record; for a rejecting beam with few keys it also writes the survivors as
        # 32-byte keyed records
        return RECORD_BYTES * n + (KEYED_BYTES * n_surv_beams if compacted else 0)
    if cls == "count_keys":
        return 4 * n_idx                              # pass B's histogram needs the 4-byte key of every keyed record
    if cls == "scatter":
        if compacted:
            return KEYED_BYTES * n_surv_beams + out_b * n_surv_beams  # read the compacted survivors, write their SoA
        return RECORD_BYTES * n + out_b * n_surv_beams  # read every record, write the survivors' SoA
    if cls == "index_a":
        return RECORD_BYTES * n + KEYED_BYTES * n_idx   # packed records in, 32-byte keyed records out
    if cls == "index_b":
        return KEYED_BYTES * n_idx + KEYED_BYTES * n_idx  # keyed records in, the index (keyed records by full key) out
    if cls == "beam":
        return KEYED_BYTES * m_sel + (out_b + 4) * n_surv_beams  # only the ROI-selected index records are read; SoA + key out
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1302_1861_b200 as P
    import workloads as W
    from paper_1302_1861_b200 import sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libpsl_b200 has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w, note = workload_for(args, world)
    if world > 1:  # every rank must time the same configuration
        pick = torch.tensor([int(w.name[3])], device=dev)
        dist.all_reduce(pick, op=dist.ReduceOp.MIN)
        if int(pick.item()) != int(w.name[3]):
            args.config = int(pick.item())
            w, _ = workload_for(args, world)
            note = "another rank could not hold config 5"
    n = w.n_records
    first_record = rank * n  # this rank's shard of the stream
    chunks = list(w.chunks())

    # inputs: generated once into pinned host memory (the e2e source), copied once to the device (the resident source)
    host = torch.empty(n * RECORD_BYTES, dtype=torch.uint8, pin_memory=True)  # pinned from the start: no pageable twin
    # every rank generates its own shard: share the host cores between the ranks of the node
    W.generate_into(w.gen, first_record, n, host.data_ptr(), threads=max(1, (os.cpu_count() or 1) // world))
    resident = host.to(dev)
    host_chunks = [host[f * RECORD_BYTES:(f + c) * RECORD_BYTES] for f, c in chunks]
    dev_chunks = [resident[f * RECORD_BYTES:(f + c) * RECORD_BYTES] for f, c in chunks]

    launch_cap = 0 if args.no_next else (6_000_000 if w.mode == 1 else 1 << 20)
    ctx = P.PslContext(w.grid, w.geometry, w.mode, max_records=n, max_host_records=0 if (args.no_e2e and not args.verify) else n,
                       max_chunks=len(chunks) + 1, flags=w.flags, device=local, max_launch_records=launch_cap)
    beams = [None if b is None else ctx.beam(b) for b in w.beams]
    K = w.n_keys
    h_counts = torch.empty(K, dtype=torch.int32).pin_memory()
    h_offsets = torch.empty(K + 1, dtype=torch.int32).pin_memory()

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
            ms = sharding.max_over_ranks(ms, device=dev)  # timing only: the slowest rank defines the job
            dist.barrier()
        return ms

    sampler = ClockSampler(local)
    sampler.start()

    # ---- device-resident: warm-up, then windows of EXACTLY --steps timed steps; the median window is reported ---
    for _ in range(max(args.warmup, 3)):
        step(dev_chunks, False)
    torch.cuda.synchronize()
    l0 = ctx.kernel_launches()
    windows = [timed(dev_chunks, False, args.steps)]
    launches = ctx.kernel_launches() - l0
    n_win = max(3, min(200, int(500.0 / max(windows[0], 1e-3)) + 1))  # >= 3 windows and >= 0.5 s of timed GPU work
    if world > 1:
        t = torch.tensor([n_win], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        n_win = int(t.item())
    while len(windows) < n_win:
        windows.append(timed(dev_chunks, False, args.steps))
    ms = statistics.median(windows)

    # the same steps once more with the library's per-kernel event brackets on (they cost a few microseconds per
    # launch, so they stay out of the timed region above): kernel shares and the roofline of the dominant kernel
    ctx.profile_enable(True)
    ctx.profile_read()
    ms_prof = timed(dev_chunks, False, args.steps)
    prof = ctx.profile_read()

    # ---- one step cut at its phase boundaries (brackets still on: the beam class gives the first build's beam share)
    def ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    torch.cuda.synchronize()
    ctx.reset()
    marks = [ev()]
    for c in dev_chunks:
        ctx.load_chunk(c)
    marks.append(ev())
    first_beam_ms = None
    for i, b in enumerate(beams):
        ctx.build_batches(b)
        marks.append(ev())
        if i == 0:
            first_beam_ms = ctx.profile_read()["beam"][0]  # synchronises
    torch.cuda.synchronize()
    build_ms = [marks[i + 1].elapsed_time(marks[i + 2]) for i in range(len(beams))]
    per_phase = {"load_ms": marks[0].elapsed_time(marks[1]), "build_ms": build_ms,
                 "note": "one device-resident step, CUDA events between the calls, per-kernel brackets on"}
    if w.mode == 1:
        per_phase["index_build_ms"] = build_ms[0] - first_beam_ms  # the first build finalises the index, then runs beam 0
        per_phase["beam_ms"] = [first_beam_ms] + build_ms[1:]
    ctx.profile_enable(False)

    # what one step produces (sizes the algorithmic bytes)
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
    workload_stats = dict(n_valid_in_grid=n_idx, survivors_per_step=surv_all, roi_selected_per_step=m_sel_all)

    # ---- section 8(f) phase lines (outside the timed value): sampling layer over the index / capacity-N shipments ---
    nxt = None
    if launch_cap and w.mode == 1 and all(b is not None for b in beams):
        total_psl, lens = ctx.plan_set(beams, max(n_idx, 1), seed=1, rr_group=4)
        # a plan whose largest division fills about two thirds of the launch buffer
        n_sim = max(1, int(n_idx * min(1.0, 4_000_000 / max(max(lens), 1))))
        torch.cuda.synchronize()
        p0 = ev()
        total_psl, lens = ctx.plan_set(beams, n_sim, seed=1, rr_group=4)
        p1 = ev()
        torch.cuda.synchronize()
        b_big = max(range(len(lens)), key=lambda i: lens[i])
        t_big, e_big = divmod(b_big, w.grid["n_ebins"])
        ctx.sample_batch(t_big, e_big)
        reps = 5
        s0 = ev()
        for _ in range(reps):
            la = ctx.sample_batch(t_big, e_big)
        s1 = ev()
        torch.cuda.synchronize()
        ms_s = s0.elapsed_time(s1) / reps
        nxt = {"plan_set_ms": p0.elapsed_time(p1), "n_total_psl": total_psl, "n_simulate": n_sim, "fields": len(beams),
               "division": [t_big, e_big], "list_entries": la["n_list"], "launched": la["n_launch"],
               "sample_batch_ms": ms_s, "list_entries_per_s": la["n_list"] / (ms_s * 1e-3),
               # list out (5 B) + one 32-byte index record in per entry + 38 B per launched particle out
               "gbs": (37.0 * la["n_list"] + 38.0 * la["n_launch"]) / (ms_s * 1e-3) / 1e9,
               "what": "psl_plan_set (budgets) + psl_sample_batch of the fullest (type, energy) division: round-robin launch "
                       "list, per-field jaws / weights / rotations / surface projection, compaction; device time incl. the "
                       "call's final synchronisation"}
    elif launch_cap and w.mode == 0:
        ctx.build_batches(beams[0])
        ctx.flush_schedule(65536)
        torch.cuda.synchronize()
        s0 = ev()
        fl = ctx.flush_schedule(65536)
        s1 = ev()
        torch.cuda.synchronize()
        nxt = {"flush_schedule_ms": s0.elapsed_time(s1), "capacity": 65536, "shipments": fl["n_events"],
               "what": "psl_flush_schedule: bins of 65536 particles shipped when full (PAPER.md:47)"}

    # ---- section 8(e)'s one optional exchange, once over NCCL, outside the timed value ----------------------
    exchange_ms = None
    if world > 1:
        counts, _ = ctx.get_tables()
        for rep in range(2):
            torch.cuda.synchronize()
            x0 = ev()
            slot0, total = sharding.global_offsets(counts)
            x1 = ev()
            torch.cuda.synchronize()
            exchange_ms = sharding.max_over_ranks(x0.elapsed_time(x1), device=dev)
        assert int(total.sum().item()) >= int(counts.to(torch.int64).sum().item())
        del slot0, total

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
    compacted = (w.mode == 0 and (w.n_keys + 7) // 8 * 8 <= 256 and not (w.flags & P.NO_COMPACT)
                 and any(b is not None and (b.get("jaws") is not None or (w.flags & P.DROP_ZERO_WEIGHT)) for b in w.beams))
    kernels = {}
    for cls, (tot_ms, brackets) in prof.items():
        if brackets == 0:
            continue
        per_step_bytes = algorithmic_bytes(cls, n, n_idx, m_sel_all, surv_all, proj, compacted)
        kernels[cls] = {"ms_per_step": tot_ms / args.steps, "launches_per_step": brackets / args.steps}
        if per_step_bytes:
            kernels[cls].update(avg_launch_ms=tot_ms / brackets, algorithmic_bytes_per_step=per_step_bytes,
                                gbs=per_step_bytes * args.steps / (tot_ms * 1e-3) / 1e9 if tot_ms > 0 else None)
    dom = max((c for c in kernels if "gbs" in kernels[c]), key=lambda c: kernels[c]["ms_per_step"])
    d = kernels[dom]
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            traffic = json.load(f).get(w.name, {}).get(dom)
    except Exception:
        pass
    step_bytes = sum(k["algorithmic_bytes_per_step"] for k in kernels.values() if "gbs" in k)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": d["gbs"], "peak": peak, "unit": "GB/s",
                "frac": d["gbs"] / peak, "peak_source": peak_src,
                "frac_of_nominal_8000": d["gbs"] / 8000.0,  # also against the nominal ~8 TB/s
                "bytes_per_launch": d["algorithmic_bytes_per_step"] / d["launches_per_step"],
                "avg_launch_ms": d["avg_launch_ms"], "traffic": traffic,
                "step_algorithmic_bytes": step_bytes,
                "step_frac": step_bytes / (ms / args.steps * 1e-3) / 1e9 / peak,
                "ms_per_step_with_brackets": ms_prof / args.steps}
    if w.mode == 1:
        # the index build against SURVEY 8(d)'s two budgets: 56 B/record floor (read once, write once) and
        # 28 + 2 x 56 = 140 B/record for two stable digit passes
        ib = per_phase["index_build_ms"] + per_phase["load_ms"]
        roofline["index_build_ms"] = ib
        roofline["index_build_frac_of_140B_budget"] = 140.0 * n / (ib * 1e-3) / 1e9 / peak
        roofline["index_build_frac_of_56B_floor"] = 56.0 * n / (ib * 1e-3) / 1e9 / peak

    verify = run_verify(ctx, w, host, beams, step, host_chunks) if args.verify and rank == 0 else None

    if rank == 0:
        line = {
            "metric": METRIC, "value": world * n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": describe(w, world, note), "workload_stats": workload_stats,
            "windows_ms": windows, "timed_gpu_s": sum(windows) * 1e-3,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "per_phase": per_phase, "roofline": roofline, "kernels": kernels,
        }
        if nxt is not None:
            line["next_8f"] = nxt
        if exchange_ms is not None:
            line["exchange_ms"] = exchange_ms
        if verify is not None:
            line["verify"] = verify
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


def run_restream(args):
    """--variant 5b: no index is kept; for EVERY beam the whole phase-space is streamed
    again from pinned host memory in the configuration's chunks ("copied in chunks") and that beam's
    batches are built on the fly from the chunks -- jaws, fluence map, MU weight, stable (type, energy) order; keys have
    no position part, the jaw test is the cull.  The synthetic stream is not position-sorted, so no chunk can be
    skipped as a whole: all 105 chunks cross the host link for each of the nine beams (252 GB per step), which is the
    bound.  One GPU; the value IS the end-to-end value (there is no resident input in this variant)."""
    import torch

    import paper_1302_1861_b200 as P
    import workloads as W

    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("bench.py --variant 5b: one GPU")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libpsl_b200 has no CPU path")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    w = W.config(5, args.records or None)
    if args.records and W.config(5).chunk_records < args.records:
        w.chunk_records = W.config(5).chunk_records
    n = w.n_records
    chunks = list(w.chunks())
    grid = dict(w.grid, n_xbins=1, n_ybins=1, x_min=-20.0, y_min=-20.0, dx=40.0, dy=40.0)
    host = torch.empty(n * RECORD_BYTES, dtype=torch.uint8, pin_memory=True)
    W.generate_into(w.gen, 0, n, host.data_ptr(), threads=os.cpu_count() or 1)
    host_chunks = [host[f * RECORD_BYTES:(f + c) * RECORD_BYTES] for f, c in chunks]
    ctx = P.PslContext(grid, w.geometry, P.MODE_ONTHEFLY, max_records=n, max_host_records=n, max_chunks=len(chunks) + 1,
                       flags=w.flags, device=0)
    beams = [ctx.beam(dict(b, roi=None)) for b in w.beams]
    K = grid["n_types"] * grid["n_ebins"]
    h_counts = torch.empty(K, dtype=torch.int32).pin_memory()
    h_offsets = torch.empty(K + 1, dtype=torch.int32).pin_memory()

    def step():
        surv = []
        for b in beams:
            ctx.reset()
            for c in host_chunks:
                ctx.load_chunk(c)
            ctx.build_batches(b)
            counts, offsets = ctx.get_tables()
            h_counts.copy_(counts, non_blocking=True)
            h_offsets.copy_(offsets, non_blocking=True)
            surv.append(ctx.get_stats()["n_survivors"])  # synchronises: the beam's result is on the host
        return surv

    land = torch.empty(max(c for _, c in chunks) * RECORD_BYTES, dtype=torch.uint8, device=dev)
    for _ in range(2):  # the host-link ceiling: plain pinned copies of the same chunks, same run
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for hc in host_chunks:
            land[:hc.numel()].copy_(hc, non_blocking=True)
        c1.record()
        torch.cuda.synchronize()
        h2d_peak = n * RECORD_BYTES / (c0.elapsed_time(c1) * 1e-3) / 1e9
    del land
    sampler = ClockSampler(0)
    sampler.start()
    surv = step()  # one step of warm-up is nine full streams
    steps = max(1, min(args.steps, 3))
    l0 = ctx.kernel_launches()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.region(True)
    e0.record()
    for _ in range(steps):
        surv = step()
    e1.record()
    torch.cuda.synchronize()
    sampler.region(False)
    ms = e0.elapsed_time(e1)
    launches = ctx.kernel_launches() - l0
    # the device side alone, brackets on: one beam's build over the chunks already in the landing zone
    ctx.profile_enable(True)
    ctx.profile_read()
    ctx.build_batches(beams[-1])
    prof = {k: v[0] for k, v in ctx.profile_read().items() if v[1]}
    ctx.profile_enable(False)
    clocks = sampler.finish()
    peak, peak_src = measured_peaks()
    h2d = len(beams) * n * RECORD_BYTES
    value = n * steps / (ms * 1e-3)
    cfg = describe(w, 1)
    cfg.update(variant="5b", keys=K, mode="onthefly", position_bins=[1, 1],
               l2_policy="every beam re-streams %.0f GB from pinned host memory" % (n * RECORD_BYTES / 1e9))
    count_gbs = RECORD_BYTES * n / (prof.get("count", 0.0) * 1e-3) / 1e9 if prof.get("count") else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": 1, "ms_per_step": ms / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": cfg, "workload_stats": {"survivors_per_beam": surv, "chunks_skipped": 0}, "clocks": clocks,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": len(beams) * ((2 * K + 1) * 4 + (K + 1) * 4 + 64),
                "h2d_gbs": h2d * steps / (ms * 1e-3) / 1e9, "h2d_peak_gbs": h2d_peak,
                "h2d_frac": h2d * steps / (ms * 1e-3) / 1e9 / h2d_peak,
                "source": "pinned host memory, %d chunk(s) x %d beams per step through psl_load_chunk(PSL_MEM_PINNED)"
                          % (len(chunks), len(beams))},
        "gpu_launches": int(launches),
        "per_phase": {"device_build_ms_one_beam": prof, "note": "kernel classes of one beam's build over the landed chunks"},
        "roofline": {"bound": "hbm", "kernel": "count", "achieved": count_gbs, "peak": peak, "unit": "GB/s",
                     "frac": None if count_gbs is None else count_gbs / peak, "peak_source": peak_src, "traffic": None,
                     "note": "the step itself is bound by the host link (e2e.h2d_frac), not by this kernel"},
    }
    print(json.dumps(line))
    ctx.destroy()
    return 0


def run_verify(ctx, w, host, beams, step, host_chunks):
    """--verify (outside every timed region): the full-size result of the configuration bench.py times, against
    the oracle.  The oracle classifies every record (all host cores, each on its own shard; no sort, no oracle
    output arrays) and np.bincount gives counts[K]: compared with the library's counts[] for the bare index (INDEX
    mode) or the build (ONTHEFLY) bit for bit, and per beam with the library's counts[], statistics and
    sum(counts) = offsets[K] = n_survivors."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor

    import workloads as W
    from oracle import psl_oracle as O

    t_start = time.perf_counter()
    rec = host.numpy().view(W.RECORD_DTYPE)
    n, K = len(rec), w.n_keys
    cores = os.cpu_count() or 1
    piece = 4_000_000
    shards = [(f, min(n, f + piece)) for f in range(0, n, piece)]
    names = ("n_invalid", "n_outside_grid", "n_roi_skipped", "n_jaw_rejected", "n_zero_weight", "n_survivors")
    cls_of = {O.INVALID: 0, O.OUTSIDE_GRID: 1, O.ROI_SKIPPED: 2, O.JAW_REJECTED: 3, O.ZERO_WEIGHT: 4, O.SURVIVOR: 5}

    def oracle_counts(beam):
        def one(se):
            o = O.Oracle(w.grid, w.geometry, flags=w.flags)
            cls, keys = o.classify(rec[se[0]:se[1]], beam)
            c = np.bincount(keys[cls == O.SURVIVOR], minlength=K).astype(np.int64)
            pop = np.bincount(cls, minlength=6)
            return c, np.array([pop[k] for k in sorted(cls_of, key=cls_of.get)], dtype=np.int64)
        counts, pops = np.zeros(K, np.int64), np.zeros(6, np.int64)
        with ThreadPoolExecutor(max_workers=cores) as ex:
            for c, p in ex.map(one, shards):
                counts += c
                pops += p
        return counts, pops

    checked = []
    step(host_chunks, False)  # the streamed path: pinned host chunks, as the e2e leg runs it
    targets = [None] + list(w.beams) if w.mode == 1 else list(w.beams)
    lib_beams = [None] + list(beams) if w.mode == 1 else list(beams)
    for i, (b, lb) in enumerate(zip(targets, lib_beams)):
        st = ctx.build_batches(lb, want_stats=True)
        c, o = ctx.get_tables()
        c = c.cpu().numpy().view(np.uint32).astype(np.int64)
        o = o.cpu().numpy().view(np.uint32).astype(np.int64)
        want, pops = oracle_counts(b)
        ok = bool(np.array_equal(c, want)) and bool(np.array_equal(np.diff(o), c)) and int(o[-1]) == st["n_survivors"] == int(c.sum())
        for k, name in enumerate(names):
            ok = ok and int(pops[k]) == st[name]
        ok = ok and sum(st[nm] for nm in names) == st["n_in"] == n
        checked.append({"build": "index" if b is None and w.mode == 1 else "beam %d" % (i - (1 if w.mode == 1 else 0)),
                        "ok": ok, "n_survivors": st["n_survivors"]})
        if not ok:
            break
    return {"ok": all(c["ok"] for c in checked) and len(checked) == len(targets), "records": n, "builds": checked,
            "how": "oracle classification of every record on %d host cores + bincount vs the library's counts[], "
                   "offsets[] and statistics, streamed from pinned host chunks" % cores,
            "seconds": time.perf_counter() - t_start}


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.variant == "5b":
        return run_restream(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
