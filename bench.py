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
def oracle_sample(w, seconds: float):
    """Time the float64 oracle on a bounded sample: bin 0, detector 0, `seconds` of output past the
    start-up transient, all templates, O1..O6.  Returns (template*s per wall-second, wall, cores)."""
    from oracle import lloid_oracle as oc
    try:
        from threadpoolctl import threadpool_limits
        limiter = threadpool_limits(1)
        cores = 1
    except Exception:
        limiter, cores = None, os.cpu_count()
    b = w.bins[0]
    W = w.peak_window
    k0 = ((b.template_len + W - 1) // W + 1) * W
    k1 = min(w.n_samples, k0 + max(1, int(round(seconds * w.f0)) // W) * W)
    x = w.strain[0].astype(np.float64)
    t0 = time.perf_counter()
    rho = oc.snr_series(x, b.slices, b.basis, b.recon, k0, k1, w.k_down, w.k_up)
    trig = oc.triggers(rho, k0, W, w.threshold)
    wall = time.perf_counter() - t0
    if limiter is not None:
        limiter.restore_original_limits()
    ts = b.n_templates * (k1 - k0) / w.f0
    return ts / wall, wall, cores, f"bin 0, detector 0, {b.n_templates} templates x {(k1 - k0) / w.f0:.0f} s of output (k in [{k0},{k1})), {len(trig)} triggers"


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

    w = make_workload(args, rank)                         # weak scaling: one config-2 replica per rank
    bank = lb.Bank(w, precision, device=local, max_chunk=args.chunk)
    n, D = w.n_samples, w.n_detectors
    n_templates = sum(b.n_templates for b in w.bins)
    cap = n_templates * D * (n // w.peak_window + 1)
    strain_dev = torch.from_numpy(w.strain).cuda()
    trig_dev = torch.empty(cap * 32, dtype=torch.uint8, device="cuda")
    cnt_dev = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream().cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        lb.lloid_reset(bank.handle, stream)
        bank.filter(strain_dev, trig_dev, cnt_dev, stream)

    # ---- device-resident throughput -----------------------------------------------------------
    launches = 0
    times = []
    with ClockSampler(local) as clocks:          # started before the warm-up: nvidia-smi needs a moment to come up
        for _ in range(args.warmup):
            step_device()
        barrier()
        clocks.mark_begin()
        for _ in range(args.steps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            step_device()
            e1.record()
            e1.synchronize()
            times.append(e0.elapsed_time(e1))
            launches += lb.lloid_last_launch_count(bank.handle)
        barrier()
        clocks.mark_end()
    n_trig = int(cnt_dev.item())
    t_dev = torch.tensor([sum(times)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t_dev, op=dist.ReduceOp.MAX)
    total_ms = float(t_dev.item())
    units = n_templates * D * (n / w.f0)                  # template * seconds of strain, this rank
    value = world * units * args.steps / (total_ms * 1e-3)

    # ---- stage times -> roofline of the dominant kernel ------------------------------------------
    lb.lloid_set_profiling(bank.handle, True)
    step_device()
    torch.cuda.synchronize()
    stage = lb.lloid_last_stage_ms(bank.handle)          # resample, FIR, recon+epilogue, merge, total
    lb.lloid_set_profiling(bank.handle, False)
    fl = workload_flops(w)
    peaks = load_peaks()
    samples = float(n) * D
    launches_per_step = max(1, int(lb.lloid_last_launch_count(bank.handle)))
    n_chunks = max(1, -(-n // int(lb.lloid_chunk_samples(bank.handle))))
    if precision == lb.LLOID_F16:
        # dominant kernel = f0_kernel (A3 of the full-rate slices + A4 + A5); its tensor credit is ONLY the algorithmic
        # reconstruction flops of the d = 1 slices -- the interpolation MMAs (A4) are ALU-equivalent work done on the
        # tensor pipe and are not counted.  The whole fused tensor path (A2 + A3, three kernels) is reported beside it.
        f0_flops = sum(2.0 * 2 * b.n_templates * s.n_basis for b in w.bins for s in b.slices if s.d == 1) * samples
        low_flops = fl["recon"] * samples - f0_flops
        f0_ms, low_ms = stage[2] - stage[5], stage[5]
        kernels = {"fir_f16_pers_kernel": (fl["fir"] * samples, stage[1]), "lowrate_recon_kernel": (low_flops, low_ms),
                   "f0_kernel": (f0_flops, f0_ms)}
        dom = max(kernels, key=lambda k: kernels[k][1])
        ach = kernels[dom][0] / (kernels[dom][1] * 1e-3) / 1e12
        path_ach = (fl["fir"] + fl["recon"]) * samples / ((stage[1] + stage[2]) * 1e-3) / 1e12
        pk = peaks["bf16_sustained"]
        # DRAM bytes (read + write) of ONE launch at the 131072-sample chunk, from the committed ncu --set full capture
        ncu_traffic = {"f0_kernel": 1.167e9, "lowrate_recon_kernel": 1.115e9, "fir_f16_pers_kernel": 0.127e9}
        full_chunk = (int(lb.lloid_chunk_samples(bank.handle)) == 131072 and (args.templates, args.detectors) == (1000, 2)
                      and args.workload == "config2")
        roofline = {"bound": "tensor", "kernel": dom, "achieved": ach, "peak": pk, "unit": "TFLOP/s", "frac": ach / pk,
                    "traffic": ncu_traffic.get(dom) if full_chunk else None,
                    "traffic_source": "profiles/r1_04_ncu_full.md (dram__bytes_read.sum + dram__bytes_write.sum, one launch)", "peak_source": peaks["source"] + " (cuBLAS bf16 sustained; fp16 runs at the same rate)",
                    "launch_ms": kernels[dom][1] / n_chunks, "launches": n_chunks,
                    "kernels": {k: {"algorithmic_tflop": v[0] / 1e12, "ms": v[1], "tflops": v[0] / (v[1] * 1e-3) / 1e12,
                                    "frac": v[0] / (v[1] * 1e-3) / 1e12 / pk} for k, v in kernels.items()},
                    "fused_tensor_path": {"achieved": path_ach, "frac": path_ach / pk,
                                          "frac_of_datasheet_2250": path_ach / 2250.0}}
        # A1 resampler against HBM: bytes = read x (4 B) + write every rate stream (fp32 + fp16) per f0 sample
        rates = sorted({s.d for b in w.bins for s in b.slices})
        res_bytes = samples * (4.0 + sum((6.0 / d) if d > 1 else 2.0 for d in rates))
        merge_bytes = (n / 128.0) * n_templates * D * 16.0          # one 16-byte partial peak per template and 128-sample tile
        roofline["merge_hbm"] = {"achieved": merge_bytes / (stage[3] * 1e-3) / 1e9, "peak": peaks["hbm"], "unit": "GB/s",
                                 "frac": merge_bytes / (stage[3] * 1e-3) / 1e9 / peaks["hbm"], "ms": stage[3]}
        roofline["resample_hbm"] = {"achieved": res_bytes / (stage[0] * 1e-3) / 1e9, "peak": peaks["hbm"], "unit": "GB/s",
                                    "frac": res_bytes / (stage[0] * 1e-3) / 1e9 / peaks["hbm"], "ms": stage[0]}
        # the direct-form decimator does 2 (2 K_dn d + 1) / d flop per input sample and rate: 27 flop per byte moved,
        # 2.4 times the machine balance (74.4 TFLOP/s / 6.5 TB/s = 11.5 flop/B) -- its bound is the FP32 ALUs
        res_flops = samples * sum(2.0 * (2 * w.k_down * d + 1) / d for d in rates if d > 1)
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
        roofline["resample_alu"] = {"achieved": res_flops / (stage[0] * 1e-3) / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
                                    "frac": res_flops / (stage[0] * 1e-3) / 1e12 / alu_peak,
                                    "flop_per_byte": res_flops / res_bytes}
    else:
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12       # FFMA lanes x 2 flop x max SM clock
        dom = ("recon+upsample", (fl["recon"] + fl["upsample"]) * samples, stage[2]) if stage[2] >= stage[1] else ("fir", fl["fir"] * samples, stage[1])
        ach = dom[1] / (dom[2] * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": dom[0], "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
                    "traffic": None, "peak_source": "derived: 148 SM x 128 FFMA/clk x 2 x 1.965 GHz"}
    roofline["stage_ms"] = {"resample": stage[0], "fir": stage[1], "recon_epilogue": stage[2], "merge_compact": stage[3], "total": stage[4],
                            "recon_lowrate_part": stage[5]}

    # ---- end to end: pinned host strain in, triggers out ---------------------------------------
    strain_pin = torch.from_numpy(w.strain).pin_memory()
    trig_pin = torch.empty(cap * 32, dtype=torch.uint8).pin_memory()
    trig_np = trig_pin.numpy().view(lb.TRIGGER_DTYPE)
    strain_np = strain_pin.numpy()
    e2e_times, d2h = [], 0
    for i in range(1 + args.steps):
        lb.lloid_reset(bank.handle, stream)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        got, rc = bank.filter_host(strain_np, trig_np, stream)
        dt = time.perf_counter() - t0
        if i > 0:
            e2e_times.append(dt)
            d2h = 8 + 32 * min(got, cap)
    t_e2e = torch.tensor([sum(e2e_times)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
    e2e_value = world * units * args.steps / float(t_e2e.item())

    chunk = int(lb.lloid_chunk_samples(bank.handle))
    dev_bytes = int(lb.lloid_device_bytes(bank.handle))
    bank.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    cpu_v, cpu_wall, cores, sample = oracle_sample(w, args.ref_seconds)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.precision, "data": "synthetic",
            "config": {"workload": workload_name(args), "units": "templates x detectors x seconds of strain per detector",
                       "per_detector_template_s_per_s": value / D, "l2": "flushed between steps (512 MiB write)",
                       "chunk_samples": chunk, "bank_device_bytes": dev_bytes, "triggers_per_step": n_trig,
                       "parallelism": f"replica per rank x{world}"},
            "clocks": clocks.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(w.strain.nbytes), "d2h_bytes_per_step": int(d2h)},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "wall_s": cpu_wall},
            "context": "paper: up to 169x (A100, float16) over GstLAL on one EPYC 7313 core (PAPER.md:96)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_stream(args):
    """BASELINE config 5: the config-3 bank (100 BBH-like bins x 500 templates, 2 detectors) fed 1 s buffers with
    history carried, back to back; per-buffer device latency (CUDA events around each lloid_filter call) and
    throughput.  Not the default bench line (config 2 is); run with --workload config5."""
    import torch
    from paper_2410_16416_b200 import binding as lb, workloads as wl
    torch.cuda.set_device(0)
    secs = args.seconds if args.seconds != 4096 else 600
    w = wl.config3(seconds=secs)
    precision = lb.LLOID_F16 if args.precision == "f16" else lb.LLOID_F32
    bank = lb.Bank(w, precision, max_chunk=args.chunk)
    D, f0 = w.n_detectors, w.f0
    n_templates = sum(b.n_templates for b in w.bins)
    strain = torch.from_numpy(w.strain).cuda()
    bufs = [strain[:, i * f0:(i + 1) * f0].contiguous() for i in range(secs)]
    cap = n_templates * D * 2
    trig = torch.empty(cap * 32, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    for i in range(min(8, secs)):                                  # warm-up calls
        bank.filter(bufs[i], trig, cnt, stream)
    lb.lloid_reset(bank.handle, stream)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(secs)]
    n_trig = 0
    with ClockSampler(0) as clocks:
        t0 = time.perf_counter()
        for i in range(secs):
            ev[i][0].record()
            bank.filter(bufs[i], trig, cnt, stream)
            ev[i][1].record()
            ev[i][1].synchronize()                                 # stream-synchronised per call (a live search reads the count)
            n_trig += int(cnt.item())
        wall = time.perf_counter() - t0
    lat = np.array([a.elapsed_time(b) for a, b in ev])
    units = n_templates * D * secs
    line = {"metric": METRIC, "value": units / (lat.sum() * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": secs, "warmup": 8,
            "ms_per_step": float(lat.mean()), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.precision, "data": "synthetic",
            "config": {"workload": f"BASELINE config 5 (config-3 bank: 100 bins x 500 templates, 2 det; {secs} x 1 s buffers, history carried)",
                       "latency_ms": {"p50": float(np.percentile(lat, 50)), "p99": float(np.percentile(lat, 99)), "max": float(lat.max())},
                       "value_including_host_sync": units / wall, "triggers": n_trig,
                       "chunk_samples": int(lb.lloid_chunk_samples(bank.handle)), "launches_per_buffer": int(lb.lloid_last_launch_count(bank.handle))},
            "clocks": clocks.summary(), "gpu_launches": int(lb.lloid_last_launch_count(bank.handle)) * secs}
    bank.close()
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
    args = ap.parse_args()
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
