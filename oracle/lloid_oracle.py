"""float64 CPU oracle for the LLOID filter + trigger generator.   TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import this module.  It shares no code with the CUDA path under
``paper_2410_16416_b200/`` and imports nothing from it (the seeded input *data* is handed in by
the caller).  Plain numpy, float64, direct sums; no FFT, no blocking, no fusion.

What it follows.  The paper names the four LLOID operations and the trigger rule and defers the
details to its refs. [17], [24] (not available):
  PAPER.md:41  (§II.A) "the LLOID algorithm ... downsamples the conditioned data, cross-correlates
               it with orthogonal templates, performs matrix multiplication of the orthogonal SNR
               time series with SVD coefficients, and finally up-samples and sums the physical SNR
               segments.  ... identifies peaks in the SNR time series with SNR > 4 ... 'triggers'."
  PAPER.md:53  (§II.B) "cross-correlation, matrix multiplication, resampling, and addition".
  PAPER.md:73  no sub-sample interpolation in the adaptation.
LLOID is an approximation (SVD truncation + multirate) to the exact matched filter, so the oracle
follows the algorithm step by step (O1..O6 below); the exact correlation is the
second-level brute force (``snr_exact``).  Every free choice is a DESIGN.md reading (R1..R12).

Pins (tests/test_oracle_pins.py): every function below is pinned by closed forms, invariants,
special cases that reduce to numpy.correlate / pure-Python brute force, the singular-value error
bound and injected-chirp recovery.  Conventions that the paper does not fix at all — the resampling
kernels' window/half-widths (R1), the strict '>' (R6), the window alignment (R7) — are
"parity unpinned": they are this build's conventions, right iff oracle and GPU agree.

Notation: f0 full rate; k absolute f0 sample index, x[k] = 0 for k < 0; slice s has
rate f_s = f0/d_s, n_s taps, L_s basis filters U^s [L_s, n_s], reconstruction R^s [2N, L_s] and
end delay Delta_s (f0 samples).  Row 2p / 2p+1 of R^s = cos / sin quadrature of template p.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

import numpy as np


# ------------------------------------------------------------------------------------------------
# O1  resampling kernels and decimation                                   ("downsamples")
# ------------------------------------------------------------------------------------------------
def lowpass_taps(d: int, K: int) -> np.ndarray:
    """lp_{d,K}[n], n = -K d .. K d  (returned array index n + K d).

    lp[n] = (1/d) sinc(n/d) * (1/2)(1 + cos(pi n / (K d))), then divided by sum_n lp[n]
    (exact unit DC gain).  Hann-windowed sinc, zero phase, cutoff at the low-rate Nyquist
    (R1).  d = 1 gives the unit impulse.
    """
    n = np.arange(-K * d, K * d + 1, dtype=np.float64)
    lp = (1.0 / d) * np.sinc(n / d) * 0.5 * (1.0 + np.cos(np.pi * n / (K * d)))
    return lp / lp.sum()


def _x_at(x: np.ndarray, k: np.ndarray) -> np.ndarray:
    """x[k] with x = 0 outside [0, len(x))  (stream starts at k = 0: DESIGN.md R10)."""
    k = np.asarray(k)
    ok = (k >= 0) & (k < len(x))
    out = np.zeros(k.shape, dtype=np.float64)
    out[ok] = x[k[ok]]
    return out


def decimate(x: np.ndarray, d: int, K: int, j_lo: int, j_hi: int) -> np.ndarray:
    """x^s[j] = sqrt(d) * sum_{n=-K d}^{K d} lp_{d,K}[n] * x[d j - n]   for j in [j_lo, j_hi).

    Decimation phase locked to absolute k = 0; the sqrt(d) keeps unit white noise near unit
    variance (R2).  d = 1: identity.
    """
    x = np.asarray(x, dtype=np.float64)
    j = np.arange(j_lo, j_hi, dtype=np.int64)
    if d == 1:
        return _x_at(x, j)
    lp = lowpass_taps(d, K)
    out = np.zeros(len(j), dtype=np.float64)
    for n in range(-K * d, K * d + 1):
        out += lp[n + K * d] * _x_at(x, d * j - n)
    return math.sqrt(d) * out


# ------------------------------------------------------------------------------------------------
# O2  basis FIR                                  ("cross-correlates it with orthogonal templates")
# ------------------------------------------------------------------------------------------------
def basis_fir(xs_seg: np.ndarray, U: np.ndarray) -> np.ndarray:
    """y_l[j] = sum_{t=0}^{n_s-1} U[l, t] * x^s[j - n_s + t]      (end-exclusive: uses x^s[< j]).

    ``xs_seg`` holds x^s[j_first - n_s .. j_last - 1]; returns y[l, j] for j = j_first..j_last.
    numpy.correlate(a, v, 'valid')[i] = sum_t a[i + t] v[t] is exactly this sum.
    """
    L, n = U.shape
    out = np.empty((L, len(xs_seg) - n + 1), dtype=np.float64)
    for l in range(L):
        out[l] = np.correlate(xs_seg, U[l], mode="valid")
    return out


# ------------------------------------------------------------------------------------------------
# O3  reconstruction                    ("matrix multiplication ... with SVD coefficients")
# ------------------------------------------------------------------------------------------------
def reconstruct(R: np.ndarray, y: np.ndarray) -> np.ndarray:
    """rho^s_i[j] = sum_l R[i, l] * y_l[j]."""
    return R @ y


# ------------------------------------------------------------------------------------------------
# O4  up-sample, delay, sum                  ("up-samples and sums the physical SNR segments")
# ------------------------------------------------------------------------------------------------
def upsample_add(acc: np.ndarray, k_begin: int, rho_s: np.ndarray, j_first: int, d: int, K: int,
                 delay: int) -> None:
    """acc[:, k - k_begin] += c^s[k],  c^s[k] = sum_j rho^s[j] * d * lp_{d,K}[k - delay - d j].

    Direct interpolation to f0 (zero-phase windowed sinc, gain d), delayed by Delta_s (R3).
    d = 1: c[k] = rho^s[k - delay].  ``rho_s[:, c]`` is rho^s[j_first + c]; samples outside the array
    are the caller's responsibility (``snr_series`` passes every j that can contribute).
    The sum runs over j and tap offset n = k - delay - d j, skipping nothing but out-of-range k.
    """
    n_out = acc.shape[1]
    if d == 1:
        for c in range(rho_s.shape[1]):
            k = j_first + c + delay
            if k_begin <= k < k_begin + n_out:
                acc[:, k - k_begin] += rho_s[:, c]
        return
    h = d * lowpass_taps(d, K)
    Kd = K * d
    for c in range(rho_s.shape[1]):
        centre = delay + d * (j_first + c)            # k at which tap n = 0 lands
        lo = max(centre - Kd, k_begin)
        hi = min(centre + Kd, k_begin + n_out - 1)
        if lo > hi:
            continue
        acc[:, lo - k_begin:hi - k_begin + 1] += np.outer(rho_s[:, c], h[lo - centre + Kd:hi - centre + Kd + 1])


# ------------------------------------------------------------------------------------------------
# O1..O4 chained: the SNR time series of one (bin, detector)
# ------------------------------------------------------------------------------------------------
def slice_j_range(k_begin: int, k_end: int, d: int, K_up: int, delay: int) -> Tuple[int, int]:
    """All low-rate indices j with |k - delay - d j| <= K_up d for some k in [k_begin, k_end)."""
    if d == 1:
        return k_begin - delay, k_end - 1 - delay
    j_first = -((-(k_begin - delay - K_up * d)) // d)      # ceil
    j_last = (k_end - 1 - delay + K_up * d) // d           # floor
    return j_first, j_last


def snr_series(x: np.ndarray, slices: Sequence, basis: Sequence[np.ndarray], recon: Sequence[np.ndarray],
               k_begin: int, k_end: int, k_down: int, k_up: int) -> np.ndarray:
    """rho_i[k] for i < 2N, k in [k_begin, k_end)  — LLOID, steps O1..O4, float64.

    ``slices[s]`` needs attributes d, n_taps, end_delay.  rho_i[k] depends only on x[k' < k]
    provided Delta_s >= (K_dn + K_up) d_s for every slice with d_s > 1 (checked).
    """
    rows = recon[0].shape[0]
    acc = np.zeros((rows, k_end - k_begin), dtype=np.float64)
    for sl, U, R in zip(slices, basis, recon):
        d, n_s, delay = sl.d, sl.n_taps, sl.end_delay
        if d > 1 and delay < (k_down + k_up) * d:
            raise ValueError("slice violates causality: Delta_s < (K_dn + K_up) d_s")
        j_first, j_last = slice_j_range(k_begin, k_end, d, k_up, delay)
        xs_seg = decimate(x, d, k_down, j_first - n_s, j_last)             # O1
        y = basis_fir(xs_seg, U)                                           # O2  [L, j_first..j_last]
        rho_s = reconstruct(R, y)                                          # O3
        upsample_add(acc, k_begin, rho_s, j_first, d, k_up, delay)         # O4
    return acc


# ------------------------------------------------------------------------------------------------
# O5, O6  windowed peaks and triggers              ("peaks ... with SNR > 4 ... triggers")
# ------------------------------------------------------------------------------------------------
def window_peaks(rho: np.ndarray, k_begin: int, W: int):
    """Per complex template p and complete window w (samples [wW, (w+1)W)): the first index k*
    attaining max_k q_p[k], q_p[k] = rho_2p[k]^2 + rho_2p+1[k]^2.   (R7, R8)

    Returns (windows [nw], kstar [N, nw] absolute, re [N, nw], im [N, nw]).
    """
    re, im = rho[0::2], rho[1::2]
    q = re * re + im * im
    k_end = k_begin + rho.shape[1]
    w_first = -((-k_begin) // W)
    w_last = k_end // W                       # exclusive
    ws = np.arange(w_first, max(w_first, w_last))
    N = q.shape[0]
    kstar = np.zeros((N, len(ws)), dtype=np.int64)
    pre = np.zeros((N, len(ws)))
    pim = np.zeros((N, len(ws)))
    for c, w in enumerate(ws):
        lo = w * W - k_begin
        a = np.argmax(q[:, lo:lo + W], axis=1)          # numpy argmax returns the first maximum
        kstar[:, c] = w * W + a
        pre[:, c] = re[np.arange(N), lo + a]
        pim[:, c] = im[np.arange(N), lo + a]
    return ws, kstar, pre, pim


def triggers(rho: np.ndarray, k_begin: int, W: int, theta: float) -> List[Tuple[int, int, float, float]]:
    """(p, k*, Re, Im) for every (template, complete window) whose peak has |rho| > theta (strict)."""
    ws, kstar, pre, pim = window_peaks(rho, k_begin, W)
    out = []
    for p in range(kstar.shape[0]):
        for c in range(len(ws)):
            if math.hypot(pre[p, c], pim[p, c]) > theta:
                out.append((p, int(kstar[p, c]), float(pre[p, c]), float(pim[p, c])))
    return out


# ------------------------------------------------------------------------------------------------
# second-level brute force (tiny banks)
# ------------------------------------------------------------------------------------------------
def snr_untruncated(x, slices, slice_filters, k_begin, k_end, k_down, k_up) -> np.ndarray:
    """BF-1: time-sliced multirate filter with the un-truncated slice filters G^s in place of
    R^s U^s (isolates the SVD truncation).  rho^s_i[j] = sum_t G^s[i,t] x^s[j - n_s + t]."""
    rows = slice_filters[0].shape[0]
    acc = np.zeros((rows, k_end - k_begin), dtype=np.float64)
    for sl, G in zip(slices, slice_filters):
        j_first, j_last = slice_j_range(k_begin, k_end, sl.d, k_up, sl.end_delay)
        xs_seg = decimate(x, sl.d, k_down, j_first - sl.n_taps, j_last)
        rho_s = basis_fir(xs_seg, G)
        upsample_add(acc, k_begin, rho_s, j_first, sl.d, k_up, sl.end_delay)
    return acc


def snr_exact(x, templates, k_begin, k_end) -> np.ndarray:
    """BF-2: the exact matched filter at f0, rho_i[k] = sum_m h_i[m] x[k - M + m]."""
    x = np.asarray(x, dtype=np.float64)
    rows, M = templates.shape
    seg = _x_at(x, np.arange(k_begin - M, k_end - 1))
    out = np.empty((rows, k_end - k_begin))
    for i in range(rows):
        out[i] = np.correlate(seg, templates[i], mode="valid")
    return out
