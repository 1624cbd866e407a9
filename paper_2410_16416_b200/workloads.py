"""Seeded synthetic inputs for the LLOID hot path: SVD banks and whitened strain.

This module is the *input generator* (the paper's "setup stage",
PAPER.md:33 — "templates are split into different time slices, which then undergo
singular value decomposition ... referred to as an SVD bank"). It serves both the CPU
oracle (``oracle/``) and the CUDA path (``paper_2410_16416_b200.binding``) with the same
arrays, and it holds **none of the method's arithmetic**: no resampling, no FIR, no
reconstruction, no peak finding.  It only
  * evaluates the closed-form Newtonian chirp of BASELINE.json's configs at integer
    sample positions, tapers and normalises it,
  * takes strided samples of those templates per time slice (a time slice of rate
    f_s = f0/d keeps every d-th template sample, times sqrt(d); reading R3),
  * calls LAPACK's SVD (numpy) per slice and truncates to the top L vectors,
  * draws seeded N(0,1) strain and adds template injections.

numpy only; importing this module never touches torch or the CUDA extension.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

F0 = 2048            # full sample rate of the whitened strain, Hz (every config in BASELINE.json)
PEAK_WINDOW = 2048   # W: 1 s peak windows
SNR_THRESHOLD = 4.0  # theta ("SNR > 4")
K_DOWN = 16          # half-width (zero crossings at the low rate) of the decimation kernel
K_UP = 8             # half-width of the interpolation kernel
TAPER_SAMPLES = F0 // 16   # Tukey tapers are 1/16 s at each end (reading R9)


# --------------------------------------------------------------------------------------
# data model
# --------------------------------------------------------------------------------------
@dataclass
class SliceSpec:
    """Geometry of one time slice (SURVEY.md §8.0 notation)."""
    rate: int        # f_s
    d: int           # f0 / f_s, a power of two
    a: int           # slice span [a, b) in template sample coordinates at f0
    b: int
    n_taps: int      # n_s = (b - a) / d
    n_basis: int     # L_s
    end_delay: int   # Delta_s = M - b


@dataclass
class BinData:
    """One SVD bin: N complex templates (2N real rows, 2p = cos, 2p+1 = sin)."""
    n_templates: int
    template_len: int                      # M, f0 samples
    slices: List[SliceSpec]
    basis: List[np.ndarray]                # U^s  [L_s, n_s] float64, rows orthonormal
    recon: List[np.ndarray]                # R^s  [2N, L_s]  float64  (= V * sigma, truncated)
    sigma: List[np.ndarray]                # all singular values per slice (for the P2/P5 pins)
    slice_filters: Optional[List[np.ndarray]] = None   # G^s [2N, n_s] (tiny banks only: BF-1)
    templates: Optional[np.ndarray] = None             # h [2N, M] at f0 (tiny banks only: BF-2)
    mchirp: Optional[np.ndarray] = None


@dataclass
class Injection:
    bin: int
    template: int    # p
    amplitude: float # A (expected SNR for a lossless bank)
    phase: float     # phi
    end: int         # e: template occupies x[e-M, e)


@dataclass
class Workload:
    name: str
    bins: List[BinData]                    # bank[b] is used for every detector of bin b
    n_detectors: int
    strain: np.ndarray                     # [D, n] float32
    injections: List[Injection] = field(default_factory=list)
    f0: int = F0
    peak_window: int = PEAK_WINDOW
    threshold: float = SNR_THRESHOLD
    k_down: int = K_DOWN
    k_up: int = K_UP

    @property
    def n_samples(self) -> int:
        return int(self.strain.shape[1])

    def template_seconds(self) -> float:
        """sum_bins N * D * T_strain  (template * detector * seconds of strain)."""
        t = self.n_samples / self.f0
        return float(sum(b.n_templates for b in self.bins) * self.n_detectors * t)


# --------------------------------------------------------------------------------------
# waveforms (closed form; BASELINE.json configs)
# --------------------------------------------------------------------------------------
def chirp_coefficient(mchirp: np.ndarray) -> np.ndarray:
    """A in f(tau) = A * tau^(-3/8):  134 Hz * (1.21 Msun / Mc)^(5/8)   [BASELINE.json configs]."""
    return 134.0 * (1.21 / np.asarray(mchirp, dtype=np.float64)) ** (5.0 / 8.0)


def template_rows(mchirp: Sequence[float], M: int, f_low: float, f_high: float,
                  m: np.ndarray, f0: int = F0) -> Tuple[np.ndarray, np.ndarray]:
    """Un-normalised cos and sin rows at integer template sample positions ``m`` (0 <= m < M).

    Sample m sits tau_m = (M - m)/f0 seconds before the template end.  f(tau) = A tau^(-3/8),
    phase Phi(tau) = 2 pi (8/5) A tau^(5/8) (the integral of f), amplitude tau^(-1/4).
    Support = {m : f_low <= f(tau_m) <= f_high}, clipped to [0, M).  A Tukey window with
    TAPER_SAMPLES-long cosine ramps covers the support.  Returns ([n_mc, len(m)], same).
    """
    mc = np.asarray(mchirp, dtype=np.float64)[:, None]
    A = chirp_coefficient(mc)
    m = np.asarray(m, dtype=np.float64)[None, :]
    tau = (M - m) / f0
    tau_hi = (A / f_high) ** (8.0 / 3.0)            # f reaches f_high at this tau (end of support)
    tau_lo = (A / f_low) ** (8.0 / 3.0)             # f equals f_low at this tau (start of support)
    m_first = np.maximum(0.0, np.ceil(M - tau_lo * f0))
    m_last = np.minimum(M - 1.0, np.floor(M - tau_hi * f0))
    u = m - m_first
    v = m_last - m
    inside = (u >= 0) & (v >= 0)
    edge = np.minimum(np.minimum(u, v), TAPER_SAMPLES).clip(min=0.0)
    w = np.where(inside, 0.5 * (1.0 - np.cos(np.pi * edge / TAPER_SAMPLES)), 0.0)
    tau_safe = np.where(inside, tau, 1.0)
    amp = w * tau_safe ** (-0.25)
    phi = 2.0 * np.pi * (8.0 / 5.0) * A * tau_safe ** (5.0 / 8.0)
    return amp * np.cos(phi), amp * np.sin(phi)


def slice_layout(M: int, spans: Sequence[Tuple[int, float, float]], n_basis,
                 f0: int = F0) -> List[SliceSpec]:
    """Build SliceSpecs from (rate, tau_lo_seconds, tau_hi_seconds) triples, latest slice first."""
    out = []
    if isinstance(n_basis, int):
        n_basis = [n_basis] * len(spans)
    for (rate, tlo, thi), L in zip(spans, n_basis):
        d = f0 // rate
        assert d * rate == f0 and d & (d - 1) == 0, "rate must divide f0 by a power of two"
        b = M - int(round(tlo * f0))
        a = M - int(round(thi * f0))
        assert a % d == 0 and b % d == 0 and 0 <= a < b <= M
        out.append(SliceSpec(rate=rate, d=d, a=a, b=b, n_taps=(b - a) // d, n_basis=int(L),
                             end_delay=M - b))
    assert out[0].b == M and out[-1].a == 0
    for s0, s1 in zip(out[:-1], out[1:]):
        assert s0.a == s1.b, "slices must tile [0, M) without gaps"
    return out


def make_bin(mchirp: Sequence[float], M: int, f_low: float, f_high: float,
             spans: Sequence[Tuple[int, float, float]], n_basis, keep_dense: bool = False,
             row_chunk: int = 128) -> BinData:
    """Templates -> per-slice strided samples -> SVD -> (U^s, R^s).

    Each real row is divided by its own l2 norm at f0 (sum_m h[m]^2 = 1).  Slice filters are
    G^s[i, t] = sqrt(d_s) * h_i[a_s + d_s t]; G^s = V diag(sigma) W^T; U^s = W^T[:L],
    R^s = (V sigma)[:, :L].
    """
    mchirp = np.asarray(mchirp, dtype=np.float64)
    N = len(mchirp)
    slices = slice_layout(M, spans, n_basis)
    G = [np.empty((2 * N, s.n_taps)) for s in slices]
    H = np.empty((2 * N, M)) if keep_dense else None
    m_all = np.arange(M)
    for p0 in range(0, N, row_chunk):
        p1 = min(N, p0 + row_chunk)
        c, s_ = template_rows(mchirp[p0:p1], M, f_low, f_high, m_all)
        c /= np.sqrt(np.sum(c * c, axis=1, keepdims=True))
        s_ /= np.sqrt(np.sum(s_ * s_, axis=1, keepdims=True))
        for sl, g in zip(slices, G):
            g[2 * p0:2 * p1:2] = math.sqrt(sl.d) * c[:, sl.a:sl.b:sl.d]
            g[2 * p0 + 1:2 * p1:2] = math.sqrt(sl.d) * s_[:, sl.a:sl.b:sl.d]
        if keep_dense:
            H[2 * p0:2 * p1:2] = c
            H[2 * p0 + 1:2 * p1:2] = s_
    basis, recon, sigma = [], [], []
    for sl, g in zip(slices, G):
        V, sg, Wt = np.linalg.svd(g, full_matrices=False)
        L = min(sl.n_basis, len(sg))
        sl.n_basis = L
        basis.append(np.ascontiguousarray(Wt[:L]))
        recon.append(np.ascontiguousarray(V[:, :L] * sg[None, :L]))
        sigma.append(sg)
    return BinData(n_templates=N, template_len=M, slices=slices, basis=basis, recon=recon,
                   sigma=sigma, slice_filters=G if keep_dense else None,
                   templates=H, mchirp=mchirp)


def retruncate(bin_: BinData, n_basis: Sequence[int]) -> BinData:
    """Same SVD, different L per slice (config 4's L heterogeneity: SURVEY.md §8(c) O0.5)."""
    slices, basis, recon = [], [], []
    for sl, U, R, L in zip(bin_.slices, bin_.basis, bin_.recon, n_basis):
        L = min(int(L), U.shape[0])
        slices.append(SliceSpec(sl.rate, sl.d, sl.a, sl.b, sl.n_taps, L, sl.end_delay))
        basis.append(U[:L])                    # views: 1000 re-truncated bins share the base bins' memory
        recon.append(R[:, :L])
    return BinData(bin_.n_templates, bin_.template_len, slices, basis, recon, bin_.sigma,
                   None, None, bin_.mchirp)


# --------------------------------------------------------------------------------------
# strain
# --------------------------------------------------------------------------------------
def template_at_f0(bin_: BinData, p: int, f_low: float, f_high: float) -> Tuple[np.ndarray, np.ndarray]:
    """Unit-norm cos/sin rows of template p at f0 (for injections into big banks)."""
    c, s = template_rows(bin_.mchirp[p:p + 1], bin_.template_len, f_low, f_high,
                         np.arange(bin_.template_len))
    return c[0] / np.linalg.norm(c[0]), s[0] / np.linalg.norm(s[0])


def make_strain(seed: int, n_detectors: int, n_samples: int, bins: Sequence[BinData],
                injections: Sequence[Injection], f_low: float, f_high: float,
                noise: bool = True) -> np.ndarray:
    """Seeded N(0,1) strain per detector (seed + detector), injections added in float64,
    result stored as float32.   x[e-M:e] += A (cos(phi) h_2p + sin(phi) h_2p+1)."""
    out = np.empty((n_detectors, n_samples), dtype=np.float32)
    for det in range(n_detectors):
        if noise:
            rng = np.random.Generator(np.random.PCG64(seed + det))
            x = rng.standard_normal(n_samples)
        else:
            x = np.zeros(n_samples)
        for inj in injections:
            b = bins[inj.bin]
            M = b.template_len
            if b.templates is not None:
                c, s = b.templates[2 * inj.template], b.templates[2 * inj.template + 1]
            else:
                c, s = template_at_f0(b, inj.template, f_low, f_high)
            lo, hi = inj.end - M, inj.end
            assert 0 <= lo and hi <= n_samples, "injection must lie inside the strain"
            x[lo:hi] += inj.amplitude * (math.cos(inj.phase) * c + math.sin(inj.phase) * s)
        out[det] = x.astype(np.float32)
    return out


# --------------------------------------------------------------------------------------
# BASELINE.json configs (SURVEY.md §8(d) "Concrete inputs")
# --------------------------------------------------------------------------------------
SEED0 = 20241016

CONFIG1_SPANS = [(2048, 0.0, 0.5), (512, 0.5, 4.0)]
CONFIG2_SPANS = [(2048, 0.0, 0.25), (1024, 0.25, 1.0), (512, 1.0, 4.0), (256, 4.0, 8.0),
                 (256, 8.0, 16.0), (128, 16.0, 32.0), (128, 32.0, 48.0), (64, 48.0, 64.0)]
CONFIG3_SPANS = {
    16384: [(2048, 0.0, 0.5), (512, 0.5, 2.5), (128, 2.5, 8.0)],
    8192: [(2048, 0.0, 0.5), (512, 0.5, 1.5), (128, 1.5, 4.0)],
    4096: [(2048, 0.0, 0.25), (512, 0.25, 0.75), (128, 0.75, 2.0)],
}
CONFIG4_SPANS = [(2048, 0.0, 0.25), (1024, 0.25, 1.0), (512, 1.0, 4.0), (256, 4.0, 16.0),
                 (128, 16.0, 40.0), (64, 40.0, 64.0)]


def config1(lossless: bool = False, noise: bool = True, seconds: int = 16,
            n_templates: int = 64, n_basis: int = 32) -> Workload:
    """Config 1 (tiny): 64 templates, Mc 1.0-1.5 (1c: 1.20-1.25), 30-1024 Hz, M = 8192, 2 slices,
    L = 32, 16 s of strain, one injection p=32, A=12, phi=0, e=19209."""
    mc = np.linspace(1.20, 1.25, n_templates) if lossless else np.linspace(1.0, 1.5, n_templates)
    b = make_bin(mc, 8192, 30.0, 1024.0, CONFIG1_SPANS, n_basis, keep_dense=True)
    inj = [Injection(0, n_templates // 2, 12.0, 0.0, 19209)]
    x = make_strain(SEED0 + 1000 * 1, 1, seconds * F0, [b], inj, 30.0, 1024.0, noise=noise)
    return Workload("config1c" if lossless else "config1", [b], 1, x, inj)


def config2(n_templates: int = 1000, seconds: int = 4096, n_detectors: int = 2,
            n_basis: int = 150, n_injections: int = 20, mc_lo: float = 1.1,
            mc_hi: float = 1.3) -> Workload:
    """Config 2 (one BNS-like SVD bin): 1000 templates, Mc 1.1-1.3, 15-1024 Hz, M = 131072 (64 s),
    8 slices 2048...64 Hz, L = 150, 2 detectors x 4096 s, 20 injections SNR 8-20.
    ``n_templates``/``seconds`` scale it down for parity tests (same geometry)."""
    M = 131072
    mc = np.linspace(mc_lo, mc_hi, n_templates)
    b = make_bin(mc, M, 15.0, 1024.0, CONFIG2_SPANS, n_basis)
    n = seconds * F0
    inj = []
    if n > 2 * M + 64:
        for i in range(n_injections):
            e = M + (i + 1) * ((n - 2 * M) // (n_injections + 1)) + 13 * i
            inj.append(Injection(0, (37 * i) % n_templates, 8.0 + 12.0 * i / max(1, n_injections - 1),
                                 2.0 * math.pi * i / n_injections, e))
    x = make_strain(SEED0 + 1000 * 2, n_detectors, n, [b], inj, 15.0, 1024.0)
    return Workload("config2", [b], n_detectors, x, inj)


def config3(n_bins: int = 100, n_templates: int = 500, seconds: int = 2048, n_detectors: int = 2,
            n_basis: int = 64, distinct_per_class: int = 1) -> Workload:
    """Config 3 (100 BBH-like bins batched): 500 templates each, Mc_b = 5*8^(b/100), 20-1024 Hz,
    three shape classes (8 s / 4 s / 2 s templates), 3 slices 2048/512/128 Hz, L = 64.
    As the paper replicates its bank, only ``distinct_per_class`` bins per shape
    class are generated; the others reuse those arrays."""
    classes = [(0, 34, 16384), (34, 67, 8192), (67, 100, 4096)]
    cache = {}
    bins = []
    for b in range(n_bins):
        bb = b * 100 // n_bins                 # position on the 100-bin mass ladder
        M = next(Mc for lo, hi, Mc in classes if lo <= bb < hi)
        lo = next(lo for lo, hi, Mc in classes if lo <= bb < hi)
        key = (M, (bb - lo) % distinct_per_class)
        if key not in cache:
            src = lo + key[1]
            mc = np.linspace(5.0 * 8.0 ** (src / 100.0), 5.0 * 8.0 ** ((src + 1) / 100.0), n_templates)
            cache[key] = make_bin(mc, M, 20.0, 1024.0, CONFIG3_SPANS[M], n_basis)
        bins.append(cache[key])
    rng_n = seconds * F0
    x = make_strain(SEED0 + 1000 * 3, n_detectors, rng_n, bins, [], 20.0, 1024.0)
    return Workload("config3", bins, n_detectors, x, [])


def config4(n_bins: int = 1000, n_templates: int = 1000, seconds: int = 3600, n_detectors: int = 3,
            n_distinct: int = 4) -> Workload:
    """Config 4 (full-bank scale): 1000 bins x 1000 templates, M = 131072, 6 slices 2048...64 Hz,
    L(b, s) = 100 + ((37 b + 61 s) mod 201); ``n_distinct`` generated bins (Mc sub-ranges of
    1.1-1.3) replicated, L heterogeneity by re-truncating the same SVD."""
    M = 131072
    base = []
    edges = np.linspace(1.1, 1.3, n_distinct + 1)
    for i in range(n_distinct):
        base.append(make_bin(np.linspace(edges[i], edges[i + 1], n_templates), M, 15.0, 1024.0,
                             CONFIG4_SPANS, 300))
    bins = []
    for b in range(n_bins):
        L = [100 + ((37 * b + 61 * s) % 201) for s in range(len(CONFIG4_SPANS))]
        bins.append(retruncate(base[b % n_distinct], L))
    # 100 injections (BASELINE config 4): injection i -> bin 10 i, template 37 i mod N, A = 8 ... 20, phase
    # 2 pi i / 100, the same in every detector; those whose bin exists in a reduced bank are kept.  End times are spread
    # over the strain past the start-up transient, off every decimation grid.
    n = seconds * F0
    inj = []
    if n > 2 * M + 64:
        n_inj = min(100, (n_bins + 9) // 10)
        for i in range(n_inj):
            e = M + (i + 1) * ((n - 2 * M) // (n_inj + 1)) + 13 * i + 777
            inj.append(Injection(10 * i, (37 * i) % n_templates, 8.0 + 12.0 * i / 99.0, 2.0 * math.pi * i / 100.0, int(e)))
    x = make_strain(SEED0 + 1000 * 4, n_detectors, n, bins, inj, 15.0, 1024.0)
    return Workload("config4", bins, n_detectors, x, inj)


def toy(n_templates: int = 4, M: int = 256, spans=((2048, 0.0, 0.0625), (1024, 0.0625, 0.125)),
        n_basis=None, seconds: float = 1.0, seed: int = 7, mc=(1.0, 1.4), f_low: float = 40.0,
        noise: bool = True, injections: Sequence[Injection] = ()) -> Workload:
    """A bank small enough for pure-Python brute force (pins P3-P5, P9)."""
    mcs = np.linspace(mc[0], mc[1], n_templates)
    slices = slice_layout(M, spans, 1)
    if n_basis is None:
        n_basis = [min(2 * n_templates, s.n_taps) for s in slices]
    b = make_bin(mcs, M, f_low, 1024.0, spans, n_basis, keep_dense=True)
    n = int(seconds * F0)
    x = make_strain(seed, 1, n, [b], list(injections), f_low, 1024.0, noise=noise)
    return Workload("toy", [b], 1, x, list(injections))
