#!/usr/bin/env python
"""bench.py — throughput of the LLOID hot path on B200 (contract: see DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--precision f16|f32] [--impl ours|reference]

A "step" is one pass of the whole hot path (A1 resample .. A6 trigger compaction)
over one batch of synthetic input: BASELINE.json config 2 (one BNS-like SVD bin of 1000 templates,
8 time slices 2048..64 Hz, L = 150, 2 detectors x 4096 s of N(0,1) whitened strain with 20
injections).  Prints ONE JSON line (rank 0).  metric = template*s of strain filtered per wall-second:
value = (templates x detectors x seconds of strain per detector, summed over ranks) / time.

  value     device-resident inputs, timed with CUDA events around lloid_filter (per step, L2 flushed
            between steps), max over ranks
  e2e       same metric through lloid_filter_host: pinned HOST strain in, triggers + count back to
            the host, copies inside the timed region
  roofline  the dominant kernel (stage times measured by the library's CUDA events on the stream)
  cpu_baseline  the float64 oracle timed on the host cores on a bounded sample of the same workload

--impl reference: times the oracle (oracle/lloid_oracle.py) as it stands on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "template_seconds_of_strain_filtered_per_second"
UNIT = "template*s/s"


_T0 = time.time()


def note(msg):
    """Progress to stderr (stdout carries the one JSON line only)."""
    print(f"[bench {time.time() - _T0:7.1f} s] {msg}", file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------------
def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")


def workload_flops(w):
    """Algorithmic flops per f0 sample of one detector, per stage."""
    fir = rec = up = 0.0
    for b in w.bins:
        for s in b.slices:
            fir += 2.0 * s.n_basis * s.n_taps / s.d
            rec += 2.0 * 2 * b.n_templates * s.n_basis / s.d
            if s.d > 1:
                up += 2.0 * 2 * b.n_templates * 2 * w.k_up
    return dict(fir=fir, recon=rec, upsample=up)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def mark_begin(self):
        self.i0 = len(self.rows)

    def mark_end(self):
        time.sleep(0.06)                       # let the sample that covers the end of the region arrive
        self.i1 = len(self.rows)

    def summary(self):
        sm, mx, reasons = [], [], set()
        rows = self.rows[getattr(self, "i0", 0):getattr(self, "i1", len(self.rows))] or self.rows
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
_ORACLE_W = None          # the workload of the oracle legs: forked workers inherit it (pickling 1000 bins per job would copy them)


def _oracle_stretch(args):
    """One oracle call: bin 0, detector 0, output samples [k0, k1).  Module-level so that a process pool can run it."""
    k0, k1 = args
    w = _ORACLE_W
    from oracle import lloid_oracle as oc
    b = w.bins[0]
    rho = oc.snr_series(w.strain[0].astype(np.float64), b.slices, b.basis, b.recon, k0, k1, w.k_down, w.k_up)
    return len(oc.triggers(rho, k0, w.peak_window, w.threshold))


def oracle_sample(w, seconds: float, all_cores: bool = False):
    """Time the float64 oracle AS IT STANDS (single-threaded numpy; BLAS pinned to one thread) on a bounded sample:
    bin 0, detector 0, `seconds` of output past the start-up transient, all templates, O1..O6.  all_cores: the same call
    in one process per host core, each on its own `seconds`-long stretch (the work is independent across time).
    Returns (template*s per wall-second, wall, cores actually used, description)."""
    from threadpoolctl import threadpool_limits          # in the image; the oracle leg must not silently use more threads
    b = w.bins[0]
    W = w.peak_window
    k0 = ((b.template_len + W - 1) // W + 1) * W
    span = max(1, int(round(seconds * w.f0)) // W) * W
    n_proc = 1
    if all_cores:
        n_proc = max(1, min(os.cpu_count() or 1, (w.n_samples - k0) // span))
    global _ORACLE_W
    _ORACLE_W = w
    jobs = [(k0 + i * span, k0 + (i + 1) * span) for i in range(n_proc)]
    with threadpool_limits(1):
        t0 = time.perf_counter()
        if n_proc == 1:
            n_trig = _oracle_stretch(jobs[0])
        else:
            import multiprocessing as mp
            with mp.get_context("fork").Pool(n_proc) as pool:
                n_trig = sum(pool.map(_oracle_stretch, jobs))
        wall = time.perf_counter() - t0
    ts = b.n_templates * n_proc * span / w.f0
    return ts / wall, wall, n_proc, (f"bin 0, detector 0, {b.n_templates} templates x {n_proc} x {span / w.f0:.0f} s of output "
                                    f"(from k = {k0}), {n_trig} triggers")


def make_workload(args, rank=0):
    from paper_2410_16416_b200 import workloads as wl
    if args.workload == "config3":                        # batching over bins (A7): the paper's throughput-vs-banks curve
        secs = args.seconds if args.seconds != 4096 else 256
        return wl.config3(n_bins=args.bins, seconds=secs, n_detectors=args.detectors)
    if args.workload == "config4":                        # heterogeneous L = 100 ... 300 (full-bank geometry, reduced bin count)
        secs = args.seconds if args.seconds != 4096 else 192
        return wl.config4(n_bins=args.bins, n_templates=args.templates, seconds=secs, n_detectors=3, n_distinct=2)
    w = wl.config2(n_templates=args.templates, seconds=args.seconds, n_detectors=args.detectors)
    if rank:
        w.strain = wl.make_strain(wl.SEED0 + 2000 + 10 * rank, w.n_detectors, w.n_samples, w.bins, w.injections, 15.0, 1024.0)
    return w


def workload_name(args):
    if args.workload == "config4":
        secs = args.seconds if args.seconds != 4096 else 192
        return (f"BASELINE config 4 geometry, {args.bins} of 1000 bins x {args.templates} templates (6 slices 2048..64 Hz, M = 64 s, "
                f"L(b, s) = 100 + ((37 b + 61 s) mod 201)), 3 det x {secs} s")
    if args.workload == "config3":
        secs = args.seconds if args.seconds != 4096 else 256
        return (f"BASELINE config 3 geometry, {args.bins} of 100 BBH-like bins x 500 templates batched "
                f"(3 slices 2048/512/128 Hz, L=64), {args.detectors} det x {secs} s")
    full = (args.templates, args.seconds, args.detectors) == (1000, 4096, 2)
    return "BASELINE config 2 (1 BNS bin: 1000 templates, 8 slices 2048..64 Hz, L=150, 2 det x 4096 s)" if full else \
        f"config-2 geometry reduced: {args.templates} templates, {args.detectors} det x {args.seconds} s"


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args)
    vals = []
    for i in range(args.warmup + args.steps):
        v, wall, cores, sample = oracle_sample(w, args.ref_seconds)
        if i >= args.warmup:
            vals.append((v, wall))
    value = float(np.mean([v for v, _ in vals]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean([t for _, t in vals])), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args), "sample_per_step": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def time_coincidence(bank, w, trig_dev, n_trig, stream, reps=5):
    """SURVEY.md section 8(f) NEXT-2 on the triggers of the last timed step: lloid_coincidence (same template, detectors a < b, within
    max_dt samples: 10 ms baselines + 10 samples of timing resolution at 2048 Hz).  HBM-bound integer work; bytes = the
    lookup table written once (memset) + the trigger list read by the scatter and by the match kernel + the partner
    look-ups (3 windows x 4 B per other detector)."""
    import torch
    from paper_2410_16416_b200 import binding as lb
    D, n = w.n_detectors, w.n_samples
    max_dt = np.zeros((D, D), dtype=np.int32)
    for a in range(D):
        for b in range(a + 1, D):
            max_dt[a, b] = 31
    sb = lb.lloid_coincidence_scratch_bytes(bank.handle, 0, n)
    scratch = torch.empty(sb, dtype=torch.uint8, device="cuda")
    cap = max(1, n_trig)
    pairs = torch.empty(cap * 16, dtype=torch.uint8, device="cuda")
    pcnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    times = []
    for i in range(reps + 1):
        e0.record()
        lb.lloid_coincidence(bank.handle, trig_dev.data_ptr(), n_trig, 0, n, max_dt, scratch.data_ptr(), sb, pairs.data_ptr(), cap, pcnt.data_ptr(), stream)
        e1.record()
        e1.synchronize()
        if i:
            times.append(e0.elapsed_time(e1))
    ms = float(np.median(times))
    nbytes = float(sb + n_trig * (32 + 32 + 12 * (D - 1)))
    peak = load_peaks()["hbm"]
    return {"what": "lloid_coincidence on the triggers of one step (PAPER.md:41 coincidence generator; max_dt = 31 samples)",
            "n_triggers": int(n_trig), "n_pairs": int(pcnt.item()), "ms": ms, "launches": 2,
            "roofline": {"bound": "hbm", "achieved": nbytes / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": nbytes / (ms * 1e-3) / 1e9 / peak, "algorithmic_bytes": nbytes}}


def time_bank(w, precision, steps, warmup, chunk, local=0, world=1, bins=None, want_e2e=True, flush=None):
    """Build a bank over `w` and time `steps` passes of the whole hot path.  Device leg: strain resident in HBM, CUDA
    events around lloid_filter on the launching stream, L2 flushed between steps, the library's per-stage events recorded
    DURING these steps.  e2e leg: lloid_filter_host from pinned host strain to host triggers.  Returns a dict; times are
    this rank's (the caller takes the max over ranks)."""
    import torch
    from paper_2410_16416_b200 import binding as lb
    note(f"uploading {len(w.bins) if bins is None else len(bins)} bins")
    bank = lb.Bank(w, precision, device=local, max_chunk=chunk, bins=bins)
    note(f"bank resident: {lb.lloid_device_bytes(bank.handle) / 2**30:.2f} GiB, chunk {lb.lloid_chunk_samples(bank.handle)} samples")
    n, D = w.n_samples, w.n_detectors
    ids = bank.bin_ids
    n_templates = sum(w.bins[b].n_templates for b in ids)
    cap = n_templates * D * (n // w.peak_window + 1)
    if cap * 32 > (4 << 30):                         # full-bank runs: room for a 0.35 trigger rate (0.11 measured); overflow is reported
        cap = int(0.35 * cap)
    strain_dev = torch.from_numpy(w.strain).cuda()
    trig_dev = torch.empty(cap * 32, dtype=torch.uint8, device="cuda")
    cnt_dev = torch.zeros(1, dtype=torch.int64, device="cuda")
    if flush is None:
        flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream().cuda_stream

    def step_device():
        lb.lloid_reset(bank.handle, stream)
        bank.filter(strain_dev, trig_dev, cnt_dev, stream)

    out = {"launches": 0, "times": []}
    stage_sum = np.zeros(6)
    with ClockSampler(local) as clocks:          # started before the warm-up: nvidia-smi needs a moment to come up
        for _ in range(warmup):
            step_device()
        torch.cuda.synchronize()
        lb.lloid_set_profiling(bank.handle, True)   # stage events on the stream, inside the timed steps (5 records per chunk)
        clocks.mark_begin()
        for _ in range(steps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            step_device()
            e1.record()
            e1.synchronize()
            out["times"].append(e0.elapsed_time(e1))
            out["launches"] += lb.lloid_last_launch_count(bank.handle)
            stage_sum += lb.lloid_last_stage_ms(bank.handle)
        torch.cuda.synchronize()
        clocks.mark_end()
        lb.lloid_set_profiling(bank.handle, False)
    out["clocks"] = clocks.summary()
    out["stage_ms"] = stage_sum / steps              # resample, FIR, recon (both kernels), merge, whole call, low-rate kernel
    out["n_trig"] = int(cnt_dev.item())
    out["trigger_capacity"] = int(cap)
    out["units"] = n_templates * D * (n / w.f0)      # template * detector * seconds of strain per step, this rank
    out["chunk"] = int(lb.lloid_chunk_samples(bank.handle))
    out["dev_bytes"] = int(lb.lloid_device_bytes(bank.handle))
    out["path"] = lb.lloid_path_info(bank.handle)
    out["n_templates"] = n_templates
    if D >= 2 and bins is None and out["n_trig"] <= cap:
        out["coincidence"] = time_coincidence(bank, w, trig_dev, out["n_trig"], stream)
    if want_e2e:
        strain_pin = torch.from_numpy(w.strain).pin_memory()
        trig_np = torch.empty(cap * 32, dtype=torch.uint8).pin_memory().numpy().view(lb.TRIGGER_DTYPE)
        strain_np = strain_pin.numpy()
        e2e_times, d2h = [], 0
        for i in range(1 + steps):
            lb.lloid_reset(bank.handle, stream)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            got, rc = bank.filter_host(strain_np, trig_np, stream)
            dt = time.perf_counter() - t0
            if i > 0:
                e2e_times.append(dt)
                d2h = 8 + 32 * min(got, cap)
        out["e2e_s"] = sum(e2e_times)
        out["d2h"] = int(d2h)
        out["h2d"] = int(w.strain.nbytes)
        out["last_triggers"] = trig_np[:min(got, cap)].copy()
    del strain_dev, trig_dev
    bank.close()
    return out


def load_traffic():
    """DRAM bytes per launch of the reconstruction / FIR kernels from the committed ncu capture (profiles/r2_traffic.json,
    written from `ncu --set full` by hand: dram__bytes_read.sum + dram__bytes_write.sum of one launch at the 131072-sample
    chunk of config 2).  None when the file is missing."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.json")
    try:
        return json.load(open(p))
    except Exception:
        return None


def roofline_f16(w, stage, n_chunks, chunk, args, peaks):
    """Roofline of the dominant kernel from the stage times of the TIMED steps.  Tensor credit is algorithmic flops only:
    the interpolation MMAs (A4) and the extra taps of the folded slices are work done on the tensor pipe that is not counted."""
    fl = workload_flops(w)
    samples = float(w.n_samples) * w.n_detectors
    # a slice at f0 / 2 is reconstructed by the f0 kernel (its interpolation is folded into the basis filters)
    f0_flops = sum(2.0 * 2 * b.n_templates * s.n_basis / s.d for b in w.bins for s in b.slices if s.d <= 2) * samples
    low_flops = fl["recon"] * samples - f0_flops
    f0_ms, low_ms = stage[2] - stage[5], stage[5]
    kernels = {"fir_f16_pers_kernel": (fl["fir"] * samples, stage[1]), "lowrate_pair_kernel": (low_flops, low_ms),
               "f0_pair_kernel": (f0_flops, f0_ms)}
    dom = max(kernels, key=lambda k: kernels[k][1])
    ach = kernels[dom][0] / (kernels[dom][1] * 1e-3) / 1e12
    path_ach = (fl["fir"] + fl["recon"]) * samples / ((stage[1] + stage[2]) * 1e-3) / 1e12
    pk = peaks["bf16_sustained"]
    tr = load_traffic()
    full_chunk = chunk == 131072 and (args.templates, args.detectors) == (1000, 2) and args.workload == "config2"
    traffic = tr["kernels"].get(dom) if (tr and full_chunk) else None
    roofline = {"bound": "tensor", "kernel": dom, "achieved": ach, "peak": pk, "unit": "TFLOP/s", "frac": ach / pk,
                "traffic": traffic,
                "traffic_source": (tr or {}).get("source") if traffic is not None else None,
                "peak_source": peaks["source"] + " (cuBLAS bf16 sustained; fp16 runs at the same rate)",
                "times_from": "CUDA events recorded by the library inside the timed steps (mean over the steps)",
                "launch_ms": kernels[dom][1] / n_chunks, "launches": n_chunks,
                "kernels": {k: {"algorithmic_tflop": v[0] / 1e12, "ms": v[1], "tflops": v[0] / (v[1] * 1e-3) / 1e12,
                                "frac": v[0] / (v[1] * 1e-3) / 1e12 / pk} for k, v in kernels.items() if v[1] > 0},
                "fused_tensor_path": {"achieved": path_ach, "frac": path_ach / pk, "frac_of_datasheet_2250": path_ach / 2250.0}}
    rates = sorted({s.d for b in w.bins for s in b.slices})
    res_bytes = samples * (4.0 + sum((6.0 / d) if d > 1 else 2.0 for d in rates))
    n_templates = sum(b.n_templates for b in w.bins)
    merge_bytes = (w.n_samples / w.peak_window) * n_templates * w.n_detectors * (16.0 + 32.0 * 0.1)   # one partial per template and window + triggers
    roofline["merge_hbm"] = {"achieved": merge_bytes / (stage[3] * 1e-3) / 1e9, "peak": peaks["hbm"], "unit": "GB/s",
                             "frac": merge_bytes / (stage[3] * 1e-3) / 1e9 / peaks["hbm"], "ms": stage[3],
                             "note": "one 16-byte partial per template and peak window since round 2: launch-latency bound, not bandwidth bound"}
    roofline["resample_hbm"] = {"achieved": res_bytes / (stage[0] * 1e-3) / 1e9, "peak": peaks["hbm"], "unit": "GB/s",
                                "frac": res_bytes / (stage[0] * 1e-3) / 1e9 / peaks["hbm"], "ms": stage[0]}
    res_flops = samples * sum(2.0 * (2 * w.k_down * d + 1) / d for d in rates if d > 1)
    alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
    roofline["resample_alu"] = {"achieved": res_flops / (stage[0] * 1e-3) / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
                                "frac": res_flops / (stage[0] * 1e-3) / 1e12 / alu_peak, "flop_per_byte": res_flops / res_bytes,
                                "note": "the direct-form decimator is ALU-bound (27 flop/B, 2.4x the machine balance): this is the bound it is judged against"}
    return roofline


def roofline_f32(w, stage):
    fl = workload_flops(w)
    samples = float(w.n_samples) * w.n_detectors
    alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12       # FFMA lanes x 2 flop x max SM clock
    dom = ("recon+upsample", (fl["recon"] + fl["upsample"]) * samples, stage[2]) if stage[2] >= stage[1] else ("fir", fl["fir"] * samples, stage[1])
    ach = dom[1] / (dom[2] * 1e-3) / 1e12
    return {"bound": "alu", "kernel": dom[0], "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
            "traffic": None, "peak_source": "derived: 148 SM x 128 FFMA/clk x 2 x 1.965 GHz"}


def stage_dict(stage):
    return {"resample": stage[0], "fir": stage[1], "recon_epilogue": stage[2], "merge_compact": stage[3], "total": stage[4],
            "recon_lowrate_part": stage[5]}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2410_16416_b200 import binding as lb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the LLOID library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    precision = lb.LLOID_F16 if args.precision == "f16" else lb.LLOID_F32

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    note("generating the workload")
    w = make_workload(args, rank)
    note("workload ready")                         # weak scaling: one replica of the workload per rank, own noise
    barrier()
    r = time_bank(w, precision, args.steps, args.warmup, args.chunk, local, world)
    barrier()
    t_dev = torch.tensor([sum(r["times"]), r["e2e_s"]], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t_dev, op=dist.ReduceOp.MAX)      # the slowest rank sets the time
    total_ms, e2e_s = float(t_dev[0].item()), float(t_dev[1].item())
    value = world * r["units"] * args.steps / (total_ms * 1e-3)
    e2e_value = world * r["units"] * args.steps / e2e_s
    stage = r["stage_ms"]
    n_chunks = max(1, -(-w.n_samples // r["chunk"]))
    peaks = load_peaks()
    roofline = roofline_f16(w, stage, n_chunks, r["chunk"], args, peaks) if precision == lb.LLOID_F16 else roofline_f32(w, stage)
    roofline["stage_ms"] = stage_dict(stage)

    extra = {}
    if r.get("coincidence"):
        extra["coincidence"] = r["coincidence"]
    if world > 1:
        extra["config3_sharded"] = sharded_config3(args, rank, world, local)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    note("device and e2e legs done; oracle legs")
    cpu_v, cpu_wall, cores, sample = oracle_sample(w, args.ref_seconds)
    cpu_all = oracle_sample(w, args.ref_seconds, all_cores=True)
    note("oracle legs done")
    if world == 1 and args.extras and args.workload == "config2" and precision == lb.LLOID_F16:
        extra.update(run_extras(args, w))
    D = w.n_detectors
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.precision, "data": "synthetic",
            "config": {"workload": workload_name(args), "units": "templates x detectors x seconds of strain per detector",
                       "per_detector_template_s_per_s": value / D, "l2": "flushed between steps (512 MiB write)",
                       "chunk_samples": r["chunk"], "bank_device_bytes": r["dev_bytes"], "triggers_per_step": r["n_trig"],
                       "kernels": r["path"], "parallelism": f"replica per rank x{world}"},
            "clocks": r["clocks"],
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"]},
            "gpu_launches": int(r["launches"]),
            "roofline": roofline,
            "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "wall_s": cpu_wall,
                             "nproc": os.cpu_count(),
                             "all_cores": {"value": cpu_all[0], "cores": cpu_all[2], "wall_s": cpu_all[1], "sample": cpu_all[3],
                                           "per_core": cpu_all[0] / cpu_all[2]}},
            "extra": extra,
            "context": "paper: up to 169x (A100, float16) over GstLAL on one EPYC 7313 core (PAPER.md:96)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def sharded_config3(args, rank, world, local):
    """N > 1: BASELINE config 3 (100 bins) with the bins sharded over the ranks (parallel.shard_bins, LPT), the same
    strain on every rank, triggers gathered over NCCL (parallel.gather_triggers): strong scaling of one bank."""
    import torch
    import torch.distributed as dist
    from paper_2410_16416_b200 import binding as lb, parallel as par, workloads as wl
    w = wl.config3(seconds=256)
    shards = par.shard_bins([par.bin_cost(b) for b in w.bins], world)
    dist.barrier(); torch.cuda.synchronize()
    r = time_bank(w, lb.LLOID_F16, 2, 1, 0, local, world, bins=shards[rank], want_e2e=True)
    t = torch.tensor([sum(r["times"])], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    allt = par.gather_triggers(par.to_global_bins(r["last_triggers"], shards[rank]), device="cuda")
    units = sum(b.n_templates for b in w.bins) * w.n_detectors * (w.n_samples / w.f0)
    return {"workload": "BASELINE config 3, 100 bins sharded over the ranks, 2 det x 256 s", "scaling": "strong",
            "value": units * 2 / (float(t.item()) * 1e-3), "unit": UNIT, "ms_per_step": float(t.item()) / 2,
            "bins_per_rank": [len(s) for s in shards], "triggers_gathered": int(len(allt))}


def run_extras(args, w2):
    """Sub-results carried in the same JSON line (N = 1): the fp32 path on config 2, config 3 (100 bins batched), config 5
    (1 s streaming buffers) and a reduced config 4 (full-bank geometry).  Each is a short run of the same library."""
    import torch
    from paper_2410_16416_b200 import binding as lb, workloads as wl
    ex = {}
    r = time_bank(w2, lb.LLOID_F32, 3, 1, 0, want_e2e=False)
    ex["config2_fp32"] = {"value": r["units"] * 3 / (sum(r["times"]) * 1e-3), "unit": UNIT, "ms_per_step": sum(r["times"]) / 3, "steps": 3,
                          "dtype": "f32", "stage_ms": stage_dict(r["stage_ms"]), "roofline": roofline_f32(w2, r["stage_ms"])}
    w3 = wl.config3(seconds=2048)
    r = time_bank(w3, lb.LLOID_F16, 3, 1, 0, want_e2e=False)
    ex["config3_100bins"] = {"workload": "BASELINE config 3: 100 bins x 500 templates, 2 det x 2048 s", "value": r["units"] * 3 / (sum(r["times"]) * 1e-3),
                             "unit": UNIT, "ms_per_step": sum(r["times"]) / 3, "steps": 3, "dtype": "f16", "stage_ms": stage_dict(r["stage_ms"]),
                             "kernels": r["path"], "chunk_samples": r["chunk"]}
    ex["config5_stream"] = stream_measure(wl.config3(seconds=600), lb.LLOID_F16, 0)
    if args.extra_config4_bins > 0:
        nb = args.extra_config4_bins
        w4 = wl.config4(n_bins=nb, n_templates=1000, seconds=192, n_detectors=3, n_distinct=2)
        r = time_bank(w4, lb.LLOID_F16, 2, 1, 0, want_e2e=False)
        ex["config4_reduced"] = {"workload": f"BASELINE config 4 geometry: {nb} of 1000 bins x 1000 templates, L = 100 ... 300, 3 det x 192 s "
                                             "(the full 1000-bin run is profiles/r2_bench_config4_1000bins.json)",
                                 "value": r["units"] * 2 / (sum(r["times"]) * 1e-3), "unit": UNIT, "ms_per_step": sum(r["times"]) / 2, "steps": 2,
                                 "dtype": "f16", "stage_ms": stage_dict(r["stage_ms"]), "kernels": r["path"], "chunk_samples": r["chunk"]}
    return ex


def stream_measure(w, precision, chunk):
    """BASELINE config 5: 1 s buffers with history carried, back to back, stream-synchronised per call; per-buffer device
    latency from CUDA events around each lloid_filter call.  The calls are replayed from ONE captured CUDA graph."""
    import torch
    from paper_2410_16416_b200 import binding as lb
    secs = w.n_samples // w.f0
    bank = lb.Bank(w, precision, max_chunk=chunk)
    D, f0 = w.n_detectors, w.f0
    n_templates = sum(b.n_templates for b in w.bins)
    strain = torch.from_numpy(w.strain).cuda()
    cap = n_templates * D * 2
    trig = torch.empty(cap * 32, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    buf = torch.empty((D, f0), dtype=torch.float32, device="cuda")           # the graph's fixed input buffer
    side = torch.cuda.Stream()
    graph = None
    with torch.cuda.stream(side):
        for i in range(min(8, secs)):                                        # warm-up calls (eager)
            buf.copy_(strain[:, i * f0:(i + 1) * f0])
            bank.filter(buf, trig, cnt, side.cuda_stream)
        side.synchronize()
        if lb.lloid_graph_safe(bank.handle, f0):
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                bank.filter(buf, trig, cnt, side.cuda_stream)
        lb.lloid_reset(bank.handle, side.cuda_stream)
        side.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(secs)]
        n_trig = 0
        with ClockSampler(0) as clocks:
            t0 = time.perf_counter()
            for i in range(secs):
                buf.copy_(strain[:, i * f0:(i + 1) * f0])
                ev[i][0].record(side)
                if graph is not None:
                    lb.lloid_graph_advance(bank.handle, f0)                  # host-side sample counter of the replayed call
                    graph.replay()
                else:
                    bank.filter(buf, trig, cnt, side.cuda_stream)
                ev[i][1].record(side)
                ev[i][1].synchronize()                                       # a live search reads the count after every buffer
                n_trig += int(cnt.item())
            wall = time.perf_counter() - t0
    lat = np.array([a.elapsed_time(b) for a, b in ev])
    units = n_templates * D * secs
    out = {"workload": f"BASELINE config 5 (config-3 bank: {len(w.bins)} bins x 500 templates, {D} det; {secs} x 1 s buffers, history carried)",
           "value": units / (lat.sum() * 1e-3), "unit": UNIT, "ms_per_buffer": float(lat.mean()),
           "latency_ms": {"p50": float(np.percentile(lat, 50)), "p99": float(np.percentile(lat, 99)), "max": float(lat.max())},
           "value_including_host_sync": units / wall, "triggers": n_trig, "cuda_graph": graph is not None,
           "chunk_samples": int(lb.lloid_chunk_samples(bank.handle)), "launches_per_buffer": int(lb.lloid_last_launch_count(bank.handle)),
           "clocks": clocks.summary()}
    bank.close()
    return out


def run_stream(args):
    """--workload config5: the streaming line on its own."""
    import torch
    from paper_2410_16416_b200 import binding as lb, workloads as wl
    torch.cuda.set_device(0)
    secs = args.seconds if args.seconds != 4096 else 600
    r = stream_measure(wl.config3(seconds=secs), lb.LLOID_F16 if args.precision == "f16" else lb.LLOID_F32, args.chunk)
    line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": 1, "steps": secs, "warmup": 8, "ms_per_step": r["ms_per_buffer"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
            "config": {k: r[k] for k in ("workload", "latency_ms", "value_including_host_sync", "triggers", "cuda_graph", "chunk_samples", "launches_per_buffer")},
            "clocks": r["clocks"], "gpu_launches": r["launches_per_buffer"] * secs}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default="f16", choices=["f16", "f32"])
    ap.add_argument("--templates", type=int, default=1000)
    ap.add_argument("--seconds", type=int, default=4096)
    ap.add_argument("--detectors", type=int, default=2)
    ap.add_argument("--workload", default="config2", choices=["config2", "config3", "config4", "config5"],
                    help="config2: the headline bench line; config3: --bins BBH-like bins batched offline (throughput vs number of "
                         "bins, PAPER.md:96); config5: 1 s streaming buffers on the config-3 bank (p50/p99 latency)")
    ap.add_argument("--bins", type=int, default=100, help="number of SVD bins batched (--workload config3 / config4: full-bank geometry with heterogeneous L)")
    ap.add_argument("--chunk", type=int, default=0, help="library time-chunk length in samples (0 = automatic)")
    ap.add_argument("--ref-seconds", type=float, default=2.0, help="seconds of output the oracle sample covers")
    ap.add_argument("--no-extras", dest="extras", action="store_false", help="skip the sub-results (fp32, config 3, 5, reduced 4) of the default line")
    ap.add_argument("--extra-config4-bins", type=int, default=16, help="bins of the reduced config-4 sub-result (0: skip)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU, NCCL), rank 0 prints the line
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = max(args.warmup, 1)
    if args.workload == "config5":
        run_stream(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
