"""Pins for the float64 oracle (oracle/lloid_oracle.py) against what the paper and the mathematics
fix — closed forms, invariants, special cases that reduce to a library routine, the singular-value
error bound, pure-Python brute force on tiny inputs, injected-chirp recovery.
The paper prints no worked LLOID example (PAPER.md has no numeric SNR series), so there are no
paper-value fixtures; tests/golden/ holds oracle-written regression values only.

None of these tests touches the CUDA path.
"""
import math

import numpy as np
import pytest

from oracle import lloid_oracle as oc
from paper_2410_16416_b200 import workloads as wl

KD, KU = wl.K_DOWN, wl.K_UP


# ---------------------------------------------------------------------------------- P1: O1 resample
@pytest.mark.parametrize("d", [2, 4, 8, 16, 32])
@pytest.mark.parametrize("K", [8, 16])
def test_lowpass_taps_closed_form(d, K):
    lp = oc.lowpass_taps(d, K)
    assert len(lp) == 2 * K * d + 1
    assert abs(lp.sum() - 1.0) < 1e-14                       # exact unit DC gain
    assert np.allclose(lp, lp[::-1], atol=0, rtol=0)         # zero phase
    centre = K * d
    nz = [i for i in range(-K, K + 1) if i != 0]
    assert max(abs(lp[centre + d * i]) for i in nz) < 1e-15  # sinc zero crossings (Nyquist filter)
    assert abs(lp[0]) < 1e-15 and abs(lp[-1]) < 1e-15        # Hann reaches zero at +-K d
    # white-noise power gain of the sqrt(d)-scaled decimator (independent survey probe)
    assert abs(d * np.sum(lp ** 2) - (0.9745 if K == 16 else 0.9487)) < 2e-4


def test_decimate_identity_and_constant():
    rng = np.random.default_rng(1)
    x = rng.standard_normal(500)
    assert np.array_equal(oc.decimate(x, 1, KD, 0, 500), x)
    assert np.array_equal(oc.decimate(x, 1, KD, -3, 2), np.r_[0, 0, 0, x[:2]])
    for d in (2, 8, 32):
        c = 0.7 * np.ones(4096)
        y = oc.decimate(c, d, KD, KD + 1, 4096 // d - KD - 1)       # away from both edges
        assert np.allclose(y, math.sqrt(d) * 0.7, atol=1e-13)


@pytest.mark.parametrize("d", [2, 4, 16])
def test_decimate_sinusoid_passband_stopband_and_phase(d):
    n = 16384
    k = np.arange(n)
    nyq = 0.5 / d                                  # cycles per f0 sample
    j = np.arange(KD + 2, n // d - KD - 2)
    for frac, tol in ((0.3, 2e-3), (0.8, 2e-3)):
        f = frac * nyq
        y = oc.decimate(np.cos(2 * np.pi * f * k + 0.4), d, KD, j[0], j[-1] + 1)
        ref = math.sqrt(d) * np.cos(2 * np.pi * f * d * j + 0.4)       # zero phase: same argument
        assert np.max(np.abs(y - ref)) < tol * math.sqrt(d)
    f = 1.2 * nyq                                  # beyond Nyquist: <= -50 dB (survey: -56 dB)
    y = oc.decimate(np.cos(2 * np.pi * f * k), d, KD, j[0], j[-1] + 1)
    assert np.max(np.abs(y)) < math.sqrt(d) * 10 ** (-50 / 20)


def test_decimate_pure_python_brute_force():
    rng = np.random.default_rng(2)
    x = rng.standard_normal(300)
    d, K = 4, 3
    lp = oc.lowpass_taps(d, K)
    got = oc.decimate(x, d, K, -2, 80)
    for idx, jj in enumerate(range(-2, 80)):
        acc = 0.0
        for n in range(-K * d, K * d + 1):
            kk = d * jj - n
            if 0 <= kk < len(x):
                acc += lp[n + K * d] * x[kk]
        assert abs(got[idx] - math.sqrt(d) * acc) < 1e-13


def test_decimate_white_noise_variance():
    rng = np.random.default_rng(3)
    x = rng.standard_normal(1 << 20)
    for d in (2, 8):
        y = oc.decimate(x, d, KD, KD, (1 << 20) // d - KD)
        v = d * np.sum(oc.lowpass_taps(d, KD) ** 2)
        assert abs(y.var() / v - 1.0) < 4.0 * math.sqrt(2.0 / len(y)) * 1.5


# ---------------------------------------------------------------------------------- O4 upsample
def _upsample_literal(rho_s, j_first, d, K, delay, k_begin, k_end):
    """c[k] = sum_j rho[j] d lp[k - delay - d j] by zero-stuffing + numpy.convolve (the definition)."""
    h = d * oc.lowpass_taps(d, K)
    nj = rho_s.shape[1]
    stuffed = np.zeros((rho_s.shape[0], (nj - 1) * d + 1))
    stuffed[:, ::d] = rho_s
    out = np.zeros((rho_s.shape[0], k_end - k_begin))
    for r in range(rho_s.shape[0]):
        full = np.convolve(stuffed[r], h)                  # index 0 <-> k = delay + d j_first - K d
        k0 = delay + d * j_first - K * d
        for c in range(k_end - k_begin):
            i = k_begin + c - k0
            if 0 <= i < len(full):
                out[r, c] = full[i]
    return out


@pytest.mark.parametrize("d,K,delay", [(2, 8, 32), (4, 3, 24), (8, 8, 256)])
def test_upsample_add_matches_literal_definition(d, K, delay):
    rng = np.random.default_rng(4)
    rho_s = rng.standard_normal((3, 40))
    j_first, k_begin, k_end = -5, 10, 10 + 200
    acc = np.zeros((3, k_end - k_begin))
    oc.upsample_add(acc, k_begin, rho_s, j_first, d, K, delay)
    assert np.allclose(acc, _upsample_literal(rho_s, j_first, d, K, delay, k_begin, k_end), atol=1e-13)


def test_upsample_d1_is_pure_delay():
    rho_s = np.arange(12.0).reshape(2, 6)
    acc = np.zeros((2, 10))
    oc.upsample_add(acc, 100, rho_s, 95, 1, KU, 7)        # k = j + 7, j = 95..100 -> k = 102..107
    assert np.array_equal(acc[:, 2:8], rho_s) and not acc[:, :2].any() and not acc[:, 8:].any()


@pytest.mark.parametrize("d", [2, 8, 32])
def test_decimate_then_upsample_returns_band_limited_input(d):
    """Closed form for O1+O4 gains and alignment: for x band-limited well below the low-rate
    Nyquist, upsample(decimate(x)) = sqrt(d) * x(k - delay), no other shift (zero phase both ways)."""
    n = 8192
    k = np.arange(n)
    f = 0.25 * (0.5 / d)
    x = np.cos(2 * np.pi * f * k + 1.1)
    delay = 5 * d
    kb, ke = 3000, 3500
    j0, j1 = oc.slice_j_range(kb, ke, d, KU, delay)
    xs = oc.decimate(x, d, KD, j0, j1 + 1)[None, :]
    acc = np.zeros((1, ke - kb))
    oc.upsample_add(acc, kb, xs, j0, d, KU, delay)
    ref = math.sqrt(d) * np.cos(2 * np.pi * f * (np.arange(kb, ke) - delay) + 1.1)
    assert np.max(np.abs(acc[0] - ref)) < 3e-3 * math.sqrt(d)


# ---------------------------------------------------------------------------------- P2: bank invariants
def test_svd_bank_invariants(cfg1):
    b = cfg1.bins[0]
    for sl, U, R, G, sg in zip(b.slices, b.basis, b.recon, b.slice_filters, b.sigma):
        assert np.allclose(U @ U.T, np.eye(U.shape[0]), atol=1e-12)        # orthonormal basis
        err = G - R @ U
        assert abs(np.linalg.norm(err, 2) - sg[sl.n_basis]) < 1e-10       # = sigma_{L+1}
        assert abs(np.linalg.norm(err, "fro") ** 2 - np.sum(sg[sl.n_basis:] ** 2)) < 1e-10
    full = wl.make_bin(b.mchirp[:8], 8192, 30.0, 1024.0, wl.CONFIG1_SPANS, 16, keep_dense=True)
    for U, R, G in zip(full.basis, full.recon, full.slice_filters):
        assert np.allclose(R @ U, G, atol=1e-12)                           # L = rank: lossless
    assert np.allclose(np.sum(b.templates ** 2, axis=1), 1.0, atol=1e-12)  # unit-normalised rows


# ---------------------------------------------------------------------------------- P3: reduces to numpy.correlate
def test_single_full_rate_slice_equals_numpy_correlate():
    w = wl.toy(n_templates=3, M=128, spans=((2048, 0.0, 128 / 2048),), seconds=0.5)
    b = w.bins[0]
    x = w.strain[0].astype(np.float64)
    rho = oc.snr_series(x, b.slices, b.basis, b.recon, 0, len(x), KD, KU)
    xp = np.r_[np.zeros(128), x]
    for i in range(6):
        ref = np.correlate(xp, b.templates[i], mode="valid")[:len(x)]      # ref[k] = sum_m h[m] x[k-M+m]
        assert np.allclose(rho[i], ref, atol=1e-11)
    # and against pure-Python loops (independent of numpy.correlate, which O2 itself calls)
    for i, kk in ((0, 0), (1, 5), (4, 130), (5, 700)):
        acc = sum(b.templates[i][m] * x[kk - 128 + m] for m in range(128) if 0 <= kk - 128 + m)
        assert abs(rho[i, kk] - acc) < 1e-11


# ---------------------------------------------------------------------------------- P4: L = rank  =>  == BF-1
def test_full_rank_lloid_equals_untruncated_time_sliced_filter():
    w = wl.toy(n_templates=4, M=512, spans=((2048, 0.0, 0.0625), (1024, 0.0625, 0.125), (512, 0.125, 0.25)),
               seconds=1.0, f_low=60.0)
    b = w.bins[0]
    x = w.strain[0].astype(np.float64)
    rho = oc.snr_series(x, b.slices, b.basis, b.recon, 0, 2048, KD, KU)
    bf1 = oc.snr_untruncated(x, b.slices, b.slice_filters, 0, 2048, KD, KU)
    assert np.max(np.abs(rho - bf1)) < 1e-10


def test_bf1_pure_python_one_sample():
    """BF-1 itself against nested Python loops at a handful of (row, k) — pins index conventions
    (end-exclusive FIR, delay, interpolation taps) without any numpy routine."""
    w = wl.toy(n_templates=2, M=256, spans=((2048, 0.0, 0.0625), (512, 0.0625, 0.125)), seconds=0.5,
               f_low=60.0)
    b = w.bins[0]
    x = w.strain[0].astype(np.float64)
    Kd, Ku = 4, 2                      # (Delta_1 = 128 >= (4 + 2) * 4)
    bf1 = oc.snr_untruncated(x, b.slices, b.slice_filters, 0, 1024, Kd, Ku)

    def xat(kk):
        return x[kk] if 0 <= kk < len(x) else 0.0

    def xs(sl, j):
        if sl.d == 1:
            return xat(j)
        lp = oc.lowpass_taps(sl.d, Kd)
        return math.sqrt(sl.d) * sum(lp[n + Kd * sl.d] * xat(sl.d * j - n) for n in range(-Kd * sl.d, Kd * sl.d + 1))

    def rho_s(sl, G, i, j):
        return sum(G[i, t] * xs(sl, j - sl.n_taps + t) for t in range(sl.n_taps))

    for i, kk in ((0, 301), (3, 777), (2, 130)):
        total = 0.0
        for sl, G in zip(b.slices, b.slice_filters):
            if sl.d == 1:
                total += rho_s(sl, G, i, kk - sl.end_delay)
            else:
                h = sl.d * oc.lowpass_taps(sl.d, Ku)
                for j in range((kk - sl.end_delay) // sl.d - Ku - 1, (kk - sl.end_delay) // sl.d + Ku + 2):
                    n = kk - sl.end_delay - sl.d * j
                    if abs(n) <= Ku * sl.d:
                        total += rho_s(sl, G, i, j) * h[n + Ku * sl.d]
        assert abs(bf1[i, kk] - total) < 1e-11


# ---------------------------------------------------------------------------------- P5: truncation bound
def test_truncation_error_bounded_by_discarded_singular_values(cfg1):
    b = cfg1.bins[0]
    x = cfg1.strain[0].astype(np.float64)
    kb, ke = 9000, 9000 + 1024
    rho = oc.snr_series(x, b.slices, b.basis, b.recon, kb, ke, KD, KU)
    bf1 = oc.snr_untruncated(x, b.slices, b.slice_filters, kb, ke, KD, KU)
    diff = rho - bf1
    bound = 0.0
    for sl, sg in zip(b.slices, b.sigma):
        j0, j1 = oc.slice_j_range(kb, ke, sl.d, KU, sl.end_delay)
        seg = oc.decimate(x, sl.d, KD, j0 - sl.n_taps, j1)
        win = np.sqrt(np.convolve(seg ** 2, np.ones(sl.n_taps), mode="valid"))     # ||x^s window||_2
        gamma = 1.0
        if sl.d > 1:
            h = sl.d * oc.lowpass_taps(sl.d, KU)
            gamma = max(np.sum(np.abs(h[phi::sl.d])) for phi in range(sl.d))
        bound += gamma * sg[sl.n_basis] * win.max()
    assert 1e-3 < np.max(np.abs(diff)) <= bound          # config 1 literal truncates a lot (DESIGN R14)
    # residual variance in unit white noise, row by row:  sum_s v_s sum_{l>L} (V_il sigma_l)^2
    pred = np.zeros(diff.shape[0])
    for sl, G, U, R in zip(b.slices, b.slice_filters, b.basis, b.recon):
        v = 1.0 if sl.d == 1 else sl.d * np.sum(oc.lowpass_taps(sl.d, KD) ** 2)
        pred += v * np.sum((G - R @ U) ** 2, axis=1)
    rows = [i for i in range(diff.shape[0]) if i // 2 != 32]       # injected template excluded
    assert abs(np.sqrt(np.mean(diff[rows] ** 2)) / np.sqrt(np.mean(pred[rows])) - 1.0) < 0.15


# ---------------------------------------------------------------------------------- P6: injected chirp
@pytest.mark.parametrize("phase", [0.0, 1.0])
def test_injection_recovered_at_injected_snr_and_time(phase):
    for lossless in (True, False):
        mc = np.linspace(1.20, 1.25, 64) if lossless else np.linspace(1.0, 1.5, 64)
        b = wl.make_bin(mc, 8192, 30.0, 1024.0, wl.CONFIG1_SPANS, 32, keep_dense=True)
        p, A, e = 32, 12.0, 19209                           # e is off every decimation grid
        x = wl.make_strain(0, 1, 24576, [b], [wl.Injection(0, p, A, phase, e)], 30.0, 1024.0, noise=False)[0]
        rho = oc.snr_series(x.astype(np.float64), b.slices, b.basis, b.recon, e - 300, e + 300, KD, KU)
        q = rho[0::2] ** 2 + rho[1::2] ** 2
        assert np.argmax(q[p]) + e - 300 == e               # end-exclusive: peak exactly at k = e
        kc = sum(np.sum(R[2 * p] ** 2) for R in b.recon)    # retained power kappa_p (cos row)
        ks = sum(np.sum(R[2 * p + 1] ** 2) for R in b.recon)
        assert abs(rho[2 * p, 300] - A * math.cos(phase) * kc) < 0.005 * A
        assert abs(rho[2 * p + 1, 300] - A * math.sin(phase) * ks) < 0.005 * A
        if lossless:
            assert abs(math.hypot(rho[2 * p, 300], rho[2 * p + 1, 300]) - A) < 0.003 * A    # survey: 11.987
    # exact matched filter recovers exactly A at exactly e
    ex = oc.snr_exact(x.astype(np.float64), b.templates[2 * p:2 * p + 2], e - 3, e + 3)
    assert abs(math.hypot(ex[0, 3], ex[1, 3]) - A) < 1e-5


def _eight_slice_bin(mc_lo, mc_hi, n, L):
    return wl.make_bin(np.linspace(mc_lo, mc_hi, n), 131072, 15.0, 1024.0, wl.CONFIG2_SPANS, L)


@pytest.mark.parametrize("phase", [0.0, 1.0])
def test_injection_recovered_on_eight_slice_bank(phase):
    """P6 on config 2's geometry (8 slices, d = 1 ... 32, M = 131072) with chirp masses whose frequency stays
    below 0.75 of every slice's Nyquist (Mc 2.0-2.1: 23 Hz at tau = 48 s against 32 Hz), so the resamplers are in
    their pass band and the noise-free peak is A times the retained power, at exactly k = e."""
    b = _eight_slice_bin(2.0, 2.1, 48, 16)
    p, A, e = 29, 12.0, 131072 + 40019                     # e is off every decimation grid
    x = wl.make_strain(0, 1, 2 * 131072 + 65536, [b], [wl.Injection(0, p, A, phase, e)], 15.0, 1024.0, noise=False)[0]
    rho = oc.snr_series(x.astype(np.float64), b.slices, b.basis, b.recon, e - 200, e + 200, KD, KU)
    q = rho[0::2] ** 2 + rho[1::2] ** 2
    assert np.argmax(q[p]) + e - 200 == e
    kc = sum(np.sum(R[2 * p] ** 2) for R in b.recon)
    ks = sum(np.sum(R[2 * p + 1] ** 2) for R in b.recon)
    kx = sum(np.sum(R[2 * p] * R[2 * p + 1]) for R in b.recon)      # cos/sin rows are not exactly orthogonal
    assert 0.5 < kc < 0.97 and 0.5 < ks < 0.97                      # L = 16 truncates for real
    assert abs(rho[2 * p, 200] - A * (math.cos(phase) * kc + math.sin(phase) * kx)) < 0.003 * A
    assert abs(rho[2 * p + 1, 200] - A * (math.sin(phase) * ks + math.cos(phase) * kx)) < 0.003 * A
    # a neighbouring template responds with the truncated overlap  sum_s R_p'. R_p  (U^s orthonormal)
    p2 = p + 3
    o = sum(np.sum(R[2 * p2] * (math.cos(phase) * R[2 * p] + math.sin(phase) * R[2 * p + 1])) for R in b.recon)
    assert abs(rho[2 * p2, 200] - A * o) < 0.003 * A


def _taps_gain(d, K, f):
    lp = oc.lowpass_taps(d, K)
    i = np.arange(len(lp)) - K * d
    return np.sum(lp[None, :] * np.cos(2 * np.pi * f[:, None] * i[None, :]), axis=1)


def test_config2_band_loses_power_in_its_64_hz_slice():
    """Config 2's own chirp masses (1.1-1.3) sweep 28-33 Hz inside the 64 Hz slice: the noise-free
    peak is A kappa times the resamplers' gain there.  Stationary phase predicts the gain: the power-weighted mean
    (weight tau^-1/2) of H_down(f(tau)) H_up(f(tau)) over the support; good to a few per cent at the band edge."""
    b = _eight_slice_bin(1.18, 1.22, 32, 64)
    p, A, e = 17, 12.0, 131072 + 40019
    x = wl.make_strain(0, 1, 2 * 131072 + 65536, [b], [wl.Injection(0, p, A, 0.0, e)], 15.0, 1024.0, noise=False)[0]
    rho = oc.snr_series(x.astype(np.float64), b.slices, b.basis, b.recon, e - 8, e + 8, KD, KU)
    q = rho[0::2] ** 2 + rho[1::2] ** 2
    assert np.argmax(q[p]) == 8
    kc = sum(np.sum(R[2 * p] ** 2) for R in b.recon)
    assert abs(kc - 1.0) < 1e-3                                     # L = 64 keeps the whole narrow bank
    a_c = wl.chirp_coefficient(np.array([b.mchirp[p]]))[0]
    tau_end, tau_start = (a_c / 1024.0) ** (8 / 3), min(64.0, (a_c / 15.0) ** (8 / 3))
    num = den = 0.0
    for rate, tlo, thi in wl.CONFIG2_SPANS:
        d = wl.F0 // rate
        t = np.linspace(max(tlo, tau_end), min(thi, tau_start), 4001)
        f = a_c * t ** (-3 / 8) / wl.F0
        g = np.ones_like(t) if d == 1 else _taps_gain(d, KD, f) * _taps_gain(d, KU, f)
        w = t ** -0.5
        num += np.sum(0.5 * (w[1:] * g[1:] + w[:-1] * g[:-1]) * np.diff(t))
        den += np.sum(0.5 * (w[1:] + w[:-1]) * np.diff(t))
    got = rho[2 * p, 8] / A
    assert 0.90 < got < 0.96 and abs(got - num / den) < 0.035, (got, num / den)


# ---------------------------------------------------------------------------------- P7: white-noise normalisation
def test_white_noise_snr_is_chi2_two_dof():
    b = wl.make_bin(np.linspace(1.20, 1.25, 64), 8192, 30.0, 1024.0, wl.CONFIG1_SPANS, 32)
    x = wl.make_strain(99, 1, 24 * 2048, [b], [], 30.0, 1024.0)[0].astype(np.float64)
    skip = 8192 + (KD + KU) * 4
    rho = oc.snr_series(x, b.slices, b.basis, b.recon, skip, len(x), KD, KU)
    q = rho[0::2] ** 2 + rho[1::2] ** 2
    pred = 0.0
    for sl, R in zip(b.slices, b.recon):
        v = 1.0 if sl.d == 1 else sl.d * np.sum(oc.lowpass_taps(sl.d, KD) ** 2)
        pred += v * np.sum(R ** 2) / 64.0                    # mean over templates of sum of both rows
    assert 1.90 < pred < 2.0                                 # "chi^2 with 2 dof", minus resampler loss
    assert abs(q.mean() / pred - 1.0) < 0.03
    for t in (2.0, 6.0):                                     # exponential tail P(q > t) = exp(-t/mean)
        assert abs(np.mean(q > t) / math.exp(-t / pred) - 1.0) < 0.12


def test_white_noise_single_slice_mean_is_exactly_two():
    w = wl.toy(n_templates=3, M=128, spans=((2048, 0.0, 128 / 2048),), seconds=32.0, seed=5)
    b = w.bins[0]
    rho = oc.snr_series(w.strain[0].astype(np.float64), b.slices, b.basis, b.recon, 128, 65536, KD, KU)
    q = rho[0::2] ** 2 + rho[1::2] ** 2
    assert abs(q.mean() - 2.0) < 0.05


# ---------------------------------------------------------------------------------- P8: multirate vs exact
def test_multirate_close_to_exact_matched_filter(cfg1):
    b = cfg1.bins[0]
    x = cfg1.strain[0].astype(np.float64)
    bf1 = oc.snr_untruncated(x, b.slices, b.slice_filters, 10000, 12048, KD, KU)
    bf2 = oc.snr_exact(x, b.templates, 10000, 12048)
    assert np.sqrt(np.mean((bf1 - bf2) ** 2)) < 0.03          # survey probe: rms 0.019


# ---------------------------------------------------------------------------------- P9: peaks and triggers
def test_window_peaks_and_triggers_brute_force():
    rng = np.random.default_rng(6)
    W, kb = 64, 40                      # first window is partial -> skipped; last partial -> skipped
    rho = 2.2 * rng.standard_normal((6, 300))
    rho[0, 100] = rho[0, 110] = 9.0     # exact tie inside window 1 -> lowest k wins
    rho[1, 100] = rho[1, 110] = 0.0
    rho[2, 200 - kb] = 4.0              # |rho| == theta exactly -> no trigger (strict >)
    rho[3, 200 - kb] = 0.0
    rho[2, 192 - kb:256 - kb][np.arange(64) != 8] *= 0.1
    rho[3, 192 - kb:256 - kb] *= 0.1
    rho[3, 200 - kb] = 0.0
    ws, ks, re, im = oc.window_peaks(rho, kb, W)
    assert list(ws) == [1, 2, 3, 4]     # complete windows inside [40, 340)
    for p in range(3):
        for c, w in enumerate(ws):
            best, bk = -1.0, None
            for kk in range(w * W, (w + 1) * W):
                qq = rho[2 * p, kk - kb] ** 2 + rho[2 * p + 1, kk - kb] ** 2
                if qq > best:
                    best, bk = qq, kk
            assert ks[p, c] == bk and re[p, c] == rho[2 * p, bk - kb] and im[p, c] == rho[2 * p + 1, bk - kb]
    assert ks[0, 1] == kb + 100
    trig = oc.triggers(rho, kb, W, 4.0)
    assert (0, kb + 100, 9.0, 0.0) in trig
    assert not any(p == 1 and 192 <= kk < 256 for p, kk, _, _ in trig)
    for p, kk, r, i in trig:
        assert math.hypot(r, i) > 4.0


# ---------------------------------------------------------------------------------- P10: streaming invariants
def test_range_evaluation_shift_and_linearity(cfg1):
    b = cfg1.bins[0]
    x = cfg1.strain[0].astype(np.float64)[:16384]
    whole = oc.snr_series(x, b.slices, b.basis, b.recon, 8000, 9000, KD, KU)
    parts = np.concatenate([oc.snr_series(x, b.slices, b.basis, b.recon, a, c, KD, KU)
                            for a, c in ((8000, 8100), (8100, 8101), (8101, 9000))], axis=1)
    assert np.max(np.abs(whole - parts)) < 1e-12
    shift = 4                                              # lcm of the decimation factors
    xs = np.r_[np.zeros(shift), x]
    shifted = oc.snr_series(xs, b.slices, b.basis, b.recon, 8000 + shift, 9000 + shift, KD, KU)
    assert np.max(np.abs(whole - shifted)) < 1e-12
    y = np.random.default_rng(8).standard_normal(len(x))
    lin = oc.snr_series(2.0 * x - 3.0 * y, b.slices, b.basis, b.recon, 8000, 8200, KD, KU)
    ry = oc.snr_series(y, b.slices, b.basis, b.recon, 8000, 8200, KD, KU)
    assert np.max(np.abs(lin - (2.0 * whole[:, :200] - 3.0 * ry))) < 1e-11


def test_causality_output_ignores_future_samples(cfg1):
    b = cfg1.bins[0]
    x = cfg1.strain[0].astype(np.float64)[:16384].copy()
    a = oc.snr_series(x, b.slices, b.basis, b.recon, 9990, 10000, KD, KU)
    x[9999:] = 123.0                                       # rho[k] uses x[k' < k] only
    c = oc.snr_series(x, b.slices, b.basis, b.recon, 9990, 10000, KD, KU)
    assert np.array_equal(a, c)
    bad = [wl.SliceSpec(512, 4, 0, 64, 16, 2, 8)]
    with pytest.raises(ValueError):
        oc.snr_series(x, bad, [np.zeros((2, 16))], [np.zeros((2, 2))], 0, 8, KD, KU)


# ---------------------------------------------------------------------------------- golden regression
def test_golden_regression_values(cfg1):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "config1_oracle_snr.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    b = cfg1.bins[0]
    x = cfg1.strain[0].astype(np.float64)
    for i, k, val in rows:
        got = oc.snr_series(x, b.slices, b.basis, b.recon, int(k), int(k) + 1, KD, KU)[int(i), 0]
        assert abs(got - float(val)) < 1e-9


# ---------------------------------------------------------------------------------- NEXT-2: coincidence oracle
def _trigs(rows):
    from paper_2410_16416_b200.binding import TRIGGER_DTYPE
    t = np.zeros(len(rows), dtype=TRIGGER_DTYPE)
    for i, (b, d, p, k) in enumerate(rows):
        t[i]["bin"], t[i]["detector"], t[i]["template_idx"], t[i]["sample"] = b, d, p, k
    return t


def test_coincidence_oracle_hand_built_cases():
    from oracle import coinc_oracle as co
    dt = np.array([[0, 30, 50], [0, 0, 40], [0, 0, 0]])
    rows = [(0, 0, 5, 10000),      # 0
            (0, 1, 5, 10030),      # 1: exactly at the 0-1 tolerance         -> (0, 1)
            (0, 1, 6, 10000),      # 2: other template                         -> nothing
            (1, 1, 5, 10000),      # 3: other bin                              -> nothing
            (0, 0, 7, 20000),      # 4
            (0, 1, 7, 20031),      # 5: one sample outside                     -> nothing with 4
            (0, 2, 7, 20049),      # 6: inside 0-2 (49 <= 50), inside 1-2 (18) -> (4, 6), (5, 6)
            (0, 0, 9, 30000),      # 7
            (0, 0, 9, 30005),      # 8: same detector twice                    -> nothing between 7 and 8
            (0, 2, 9, 29960)]      # 9: 40 and 45 before                       -> (7, 9), (8, 9)
    got = co.coincidences(_trigs(rows), dt)
    assert got == {(0, 1), (4, 6), (5, 6), (7, 9), (8, 9)}
    assert co.coincidences(_trigs([]), dt) == set()
    assert co.coincidences(_trigs(rows), np.zeros((3, 3), dtype=int)) == set()          # nothing is simultaneous to the sample


def test_coincidence_oracle_equals_double_loop_on_random_lists():
    from oracle import coinc_oracle as co
    rng = np.random.Generator(np.random.PCG64(5))
    dt = [[0, 21, 35], [0, 0, 28], [0, 0, 0]]
    for n in (1, 40, 300):
        rows = [(int(rng.integers(0, 2)), int(rng.integers(0, 3)), int(rng.integers(0, 4)), int(rng.integers(0, 600))) for _ in range(n)]
        t = _trigs(rows)
        want = set()
        for i, (bi, di, pi, ki) in enumerate(rows):            # the definition, pair by pair, no grouping
            for j, (bj, dj, pj, kj) in enumerate(rows):
                if bi == bj and pi == pj and di < dj and abs(ki - kj) <= dt[di][dj]:
                    want.add((i, j))
        assert co.coincidences(t, dt) == want
        if n == 300:
            assert len(want) > 20
