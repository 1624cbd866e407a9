"""Helpers for the GPU-vs-oracle parity tests: drive the C ABI, and apply SURVEY.md §8(c)'s
comparison rule (dense tolerance; trigger existence / index / value rules with margins)."""
from __future__ import annotations

import math
from typing import Optional, Sequence, Tuple

import numpy as np

from oracle import lloid_oracle as oc
from paper_2410_16416_b200 import binding as lb

TOL = {lb.LLOID_F32: 1e-3, lb.LLOID_F16: 5e-2}     # BASELINE.json north_star, sigma units, absolute


def run_gpu(w, precision, pieces: Optional[Sequence[int]] = None, capture: Optional[Tuple[int, int, int, int]] = None,
            max_chunk: int = 0, capacity: Optional[int] = None, host_path: bool = False):
    """Feed workload ``w`` through lloid_filter (optionally in ``pieces``), return (triggers, snr, bank_info).
    capture = (bin, det, k_begin, n) arms lloid_debug_capture and returns the dense SNR [2N, n]."""
    import torch
    bank = lb.Bank(w, precision, max_chunk=max_chunk)
    try:
        n = w.n_samples
        n_win = n // w.peak_window + 1
        if capacity is None:
            capacity = sum(b.n_templates for b in w.bins) * w.n_detectors * n_win + 16
        strain = torch.from_numpy(w.strain).cuda()
        trig = torch.zeros(max(1, capacity) * 32, dtype=torch.uint8, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        snr = None
        if capture is not None:
            cb, cd, k0, cn = capture
            rows = 2 * w.bins[cb].n_templates
            snr = torch.full((rows, cn), float("nan"), dtype=torch.float32, device="cuda")
            lb.lloid_debug_capture(bank.handle, cb, cd, k0, cn, snr.data_ptr())
        out, counts, launches = [], [], 0
        pieces = [n] if pieces is None else list(pieces)
        assert sum(pieces) == n
        a = 0
        for c in pieces:
            if host_path:
                hbuf = np.zeros(max(1, capacity), dtype=lb.TRIGGER_DTYPE)
                got, rc = bank.filter_host(np.ascontiguousarray(w.strain[:, a:a + c]), hbuf)
                counts.append(got)
                out.append(hbuf[:min(got, capacity)].copy())
            else:
                bank.filter(strain[:, a:a + c].contiguous(), trig, cnt)
                torch.cuda.synchronize()
                got = int(cnt.item())
                counts.append(got)
                out.append(trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:min(got, capacity)].copy())
            launches += lb.lloid_last_launch_count(bank.handle)
            a += c
        info = dict(counts=counts, launches=launches, chunk=lb.lloid_chunk_samples(bank.handle),
                    consumed=lb.lloid_samples_consumed(bank.handle), bytes=lb.lloid_device_bytes(bank.handle),
                    path=lb.lloid_path_info(bank.handle))
        trigs = np.concatenate(out) if out else np.zeros(0, dtype=lb.TRIGGER_DTYPE)
        return trigs, (None if snr is None else snr.cpu().numpy()), info
    finally:
        bank.close()


def oracle_snr(w, bin_: int, det: int, k_begin: int, k_end: int) -> np.ndarray:
    b = w.bins[bin_]
    return oc.snr_series(w.strain[det].astype(np.float64), b.slices, b.basis, b.recon, k_begin, k_end,
                         w.k_down, w.k_up)


def check_triggers(trigs: np.ndarray, rho: np.ndarray, k_begin: int, w, bin_: int, det: int, tol: float):
    """Apply rules (ii)-(iv) to every complete window inside rho's range.  Returns stats dict."""
    W, theta = w.peak_window, w.threshold
    re, im = rho[0::2], rho[1::2]
    amp = np.sqrt(re * re + im * im)
    N = amp.shape[0]
    k_end = k_begin + rho.shape[1]
    sel = trigs[(trigs["bin"] == bin_) & (trigs["detector"] == det)]
    by_key = {}
    for t in sel:
        key = (int(t["template_idx"]), int(t["sample"]) // W)
        assert key not in by_key, f"duplicate trigger for template/window {key}"
        by_key[key] = t
    w_first = -((-k_begin) // W)
    w_last = k_end // W
    n_checked = n_trig = n_exact = 0
    for wi in range(w_first, w_last):
        lo = wi * W - k_begin
        seg = amp[:, lo:lo + W]
        kstar = np.argmax(seg, axis=1)
        best = seg[np.arange(N), kstar]
        tmp = seg.copy()
        tmp[np.arange(N), kstar] = -1.0
        margin = best - tmp.max(axis=1)
        for p in range(N):
            t = by_key.get((p, wi))
            n_checked += 1
            if abs(best[p] - theta) > tol:                       # (ii) existence
                assert (t is not None) == (best[p] > theta), \
                    f"trigger existence mismatch p={p} window={wi}: oracle peak {best[p]:.4f}, gpu {'has' if t is not None else 'lacks'} a trigger"
            if t is None:
                continue
            n_trig += 1
            kg = int(t["sample"]) - wi * W
            assert 0 <= kg < W
            if margin[p] > 2 * tol:                              # (iii) index
                assert kg == kstar[p], f"argmax mismatch p={p} window={wi}: gpu {kg} oracle {kstar[p]} margin {margin[p]:.4g}"
            else:
                assert seg[p, kg] >= best[p] - 2 * tol, f"gpu index not a near-maximum p={p} window={wi}"
            n_exact += int(kg == kstar[p])
            assert abs(float(t["snr_re"]) - re[p, lo + kg]) <= tol, f"Re mismatch p={p} window={wi}"   # (iv)
            assert abs(float(t["snr_im"]) - im[p, lo + kg]) <= tol, f"Im mismatch p={p} window={wi}"
            assert math.hypot(float(t["snr_re"]), float(t["snr_im"])) > theta
    # no triggers outside complete windows of the range that we did not account for
    for (p, wi), t in by_key.items():
        assert 0 <= p < N
    return dict(checked=n_checked, triggers=n_trig, exact_index=n_exact)
