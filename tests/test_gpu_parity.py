"""GPU-vs-oracle parity through the C ABI (include/lloid.h), element by element on the same seeded
inputs.  Tolerances are BASELINE.json's: |SNR_gpu - SNR_oracle| <= 1e-3 (fp32 path) / 5e-2 (fp16 path)
absolute in sigma units; trigger template/sample indices identical wherever the oracle's peak margin
exceeds the tolerance (SURVEY.md §8(c) comparison rule, implemented in tests/parity_util.py).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2410_16416_b200 import binding as lb          # noqa: E402
from paper_2410_16416_b200 import workloads as wl        # noqa: E402
import parity_util as pu                                 # noqa: E402

PRECISIONS = [pytest.param(lb.LLOID_F32, id="fp32"), pytest.param(lb.LLOID_F16, id="fp16")]


def _dense_check(w, precision, k0, k1, bin_=0, det=0, **kw):
    tol = pu.TOL[precision]
    trigs, snr, info = pu.run_gpu(w, precision, capture=(bin_, det, k0, k1 - k0), **kw)
    rho = pu.oracle_snr(w, bin_, det, k0, k1)
    assert not np.isnan(snr).any(), "capture left samples unwritten"
    err = np.abs(snr - rho)
    assert err.max() <= tol, f"dense SNR error {err.max():.3e} > {tol} at {np.unravel_index(err.argmax(), err.shape)}"
    stats = pu.check_triggers(trigs, rho, k0, w, bin_, det, tol)
    return trigs, snr, rho, info, stats


# ------------------------------------------------------------------------------------------------
# small banks spanning several tiles and ragged tails (odd N, odd L, taps not a multiple of 32)
# ------------------------------------------------------------------------------------------------
TOYS = {
    "one_slice": dict(n_templates=3, M=128, spans=((2048, 0.0, 128 / 2048),), seconds=1.0),
    "two_rates": dict(n_templates=5, M=1024, spans=((2048, 0.0, 0.125), (512, 0.125, 0.5)), seconds=2.0,
                      n_basis=[7, 9], f_low=40.0),
    "five_rates": dict(n_templates=37, M=16384,
                       spans=((2048, 0.0, 0.25), (1024, 0.25, 0.5), (256, 0.5, 2.0), (128, 2.0, 4.0), (64, 4.0, 8.0)),
                       seconds=12.0, n_basis=[33, 20, 40, 17, 5], f_low=20.0, mc=(1.2, 1.3)),
    # taps 520 / 300 / 100: not multiples of the kernels' K blocks; N = 70 -> 140 rows (ragged row tile)
    "ragged_taps": dict(n_templates=70, M=1520,
                        spans=((2048, 0.0, 520 / 2048), (1024, 520 / 2048, 1120 / 2048), (512, 1120 / 2048, 1520 / 2048)),
                        seconds=3.0, n_basis=[50, 30, 12], f_low=30.0, mc=(1.0, 1.1)),
}


@pytest.mark.parametrize("precision", PRECISIONS)
@pytest.mark.parametrize("name", list(TOYS))
def test_toy_banks_dense_and_triggers(name, precision):
    kw = dict(TOYS[name])
    w = wl.toy(**kw)
    w.peak_window = 256                      # many windows, even on short strain
    n = w.n_samples
    _, _, _, info, stats = _dense_check(w, precision, 0, n)
    assert stats["checked"] == w.bins[0].n_templates * (n // 256)
    assert info["consumed"] == n


@pytest.mark.parametrize("precision", PRECISIONS)
def test_one_tile_windows_and_chunks(precision):
    """peak_window = 128 and max_chunk = 128: one tile per window, per chunk and per partial-peak granule (the smallest values
    include/lloid.h allows)."""
    w = wl.toy(**TOYS["two_rates"])
    w.peak_window = 128
    n = w.n_samples
    _, _, _, info, stats = _dense_check(w, precision, 0, n, max_chunk=128)
    assert info["chunk"] == 128 and stats["checked"] == w.bins[0].n_templates * (n // 128)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config1_dense_snr_and_triggers(cfg1, precision):
    """BASELINE config 1 in full: 16 s, 64 templates, 2 slices, L = 32, injection at k = 19209."""
    w = cfg1
    trigs, snr, rho, info, stats = _dense_check(w, precision, 0, w.n_samples)
    assert stats["checked"] == 64 * 16 and stats["triggers"] > 0
    inj = w.injections[0]
    hit = trigs[(trigs["template_idx"] == inj.template) & (trigs["sample"] // w.peak_window == inj.end // w.peak_window)]
    assert len(hit) == 1 and abs(int(hit[0]["sample"]) - inj.end) <= 2  # recovered at the injected time (noise moves the
    k_or = int(np.argmax(rho[2 * inj.template] ** 2 + rho[2 * inj.template + 1] ** 2)) # peak by a sample; exact vs oracle)
    assert int(hit[0]["sample"]) == k_or
    assert stats["exact_index"] >= 0.98 * stats["triggers"]


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config1c_lossless_bank_recovers_injected_snr(cfg1c, precision):
    w = cfg1c
    trigs, _, _ = pu.run_gpu(w, precision)
    inj = w.injections[0]
    hit = trigs[(trigs["template_idx"] == inj.template) & (np.abs(trigs["sample"] - inj.end) <= 2)]
    assert len(hit) == 1
    amp = float(np.hypot(hit[0]["snr_re"], hit[0]["snr_im"]))
    assert abs(amp - inj.amplitude) < 1.5          # 12 sigma signal + unit noise


# ------------------------------------------------------------------------------------------------
# streaming (A8): pieces == one shot; chunking inside the library; host path; reset
# ------------------------------------------------------------------------------------------------
def _as_set(trigs):
    return sorted((int(t["bin"]), int(t["detector"]), int(t["template_idx"]), int(t["sample"]),
                   float(t["snr_re"]), float(t["snr_im"])) for t in trigs)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_streaming_pieces_equal_one_shot(cfg1, precision):
    w = cfg1
    n = w.n_samples
    one, _, info1 = pu.run_gpu(w, precision)
    pieces = [2048] * 4 + [4, 60, 1984, 4096, 8, 8192 - 8, 10240]
    assert sum(pieces) == n
    many, _, info2 = pu.run_gpu(w, precision, pieces=pieces)
    assert _as_set(one) == _as_set(many)
    small, _, info3 = pu.run_gpu(w, precision, max_chunk=512)           # library-internal chunking
    assert info3["chunk"] == 512 and _as_set(one) == _as_set(small)
    assert info2["consumed"] == n
    odd, _, info4 = pu.run_gpu(w, precision, max_chunk=1920)            # 15 tiles: chunks cut the 16-tile peak windows anywhere
    assert info4["chunk"] == 1920 and _as_set(one) == _as_set(odd)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_host_path_equals_device_path_and_overflow_is_reported(cfg1, precision):
    w = cfg1
    dev, _, _ = pu.run_gpu(w, precision)
    host, _, _ = pu.run_gpu(w, precision, host_path=True)
    assert _as_set(dev) == _as_set(host)
    few, _, info = pu.run_gpu(w, precision, capacity=5)
    assert info["counts"][0] == len(dev) and len(few) == 5
    assert lb.lloid_check_count(info["counts"][0], 5) == lb.LLOID_EOVERFLOW
    got = set(_as_set(few))
    assert got <= set(_as_set(dev))


def test_reset_restarts_the_stream(cfg1):
    import torch
    w = cfg1
    bank = lb.Bank(w, lb.LLOID_F32)
    strain = torch.from_numpy(w.strain).cuda()
    trig = torch.zeros(64 * 17 * 32, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    outs = []
    for _ in range(2):
        bank.filter(strain, trig, cnt)
        torch.cuda.synchronize()
        outs.append(_as_set(trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:int(cnt.item())]))
        lb.lloid_reset(bank.handle)
        assert lb.lloid_samples_consumed(bank.handle) == 0
    bank.close()
    assert outs[0] == outs[1] and len(outs[0]) > 0


def test_filter_argument_errors(cfg1):
    import torch
    bank = lb.Bank(cfg1, lb.LLOID_F32)
    strain = torch.zeros(1, 4096, device="cuda")
    trig = torch.zeros(32 * 8, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    with pytest.raises(lb.LloidError) as e:
        lb.lloid_filter(bank.handle, strain.data_ptr(), 4095, trig.data_ptr(), 8, cnt.data_ptr())
    assert e.value.code == lb.LLOID_EINVAL
    with pytest.raises(lb.LloidError):
        lb.lloid_filter(bank.handle, 0, 4096, trig.data_ptr(), 8, cnt.data_ptr())
    with pytest.raises(lb.LloidError) as e:
        lb.lloid_bank_upload_slice(bank.handle, 0, 0, 0, cfg1.bins[0].basis[0], cfg1.bins[0].recon[0])
    assert e.value.code == lb.LLOID_ESTATE
    bank.close()


# ------------------------------------------------------------------------------------------------
# several bins x detectors in one bank (A7), heterogeneous geometry, aliasing of replicated bins
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", PRECISIONS)
def test_multi_bin_multi_detector_bank(precision):
    w3 = wl.config3(n_bins=6, n_templates=24, seconds=12, n_detectors=2, n_basis=16)
    assert len({b.template_len for b in w3.bins}) == 3          # all three shape classes present
    w3.threshold = 3.0                                          # enough noise triggers in 12 s to compare
    tol = pu.TOL[precision]
    k0, k1 = 16384, 16384 + 4096
    for bin_, det in ((0, 1), (3, 0), (5, 1)):
        trigs, snr, info = pu.run_gpu(w3, precision, capture=(bin_, det, k0, k1 - k0))
        rho = pu.oracle_snr(w3, bin_, det, k0, k1)
        assert np.abs(snr - rho).max() <= tol
        pu.check_triggers(trigs, rho, k0, w3, bin_, det, tol)
    # replicated bins (same BinData object) give identical triggers up to the bin index
    a = trigs[trigs["bin"] == 0]
    b = trigs[trigs["bin"] == 1]
    assert w3.bins[0] is w3.bins[1] and len(a) == len(b) > 0
    strip = lambda t: sorted((int(x["detector"]), int(x["template_idx"]), int(x["sample"]), float(x["snr_re"])) for x in t)
    assert strip(a) == strip(b)


# ------------------------------------------------------------------------------------------------
# BASELINE config 2 geometry (8 slices 2048..64 Hz, M = 64 s, L = 150) at reduced template count
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", PRECISIONS)
def test_config2_geometry_excerpt(precision):
    w = wl.config2(n_templates=120, seconds=160, n_detectors=2, n_basis=150, n_injections=2)
    assert len(w.injections) == 2
    tol = pu.TOL[precision]
    inj = w.injections[1]
    k0 = (inj.end // 2048) * 2048 - 2048
    k1 = k0 + 3 * 2048
    trigs, snr, info = pu.run_gpu(w, precision, capture=(0, 1, k0, k1 - k0))
    rho = pu.oracle_snr(w, 0, 1, k0, k1)
    assert np.abs(snr - rho).max() <= tol
    stats = pu.check_triggers(trigs, rho, k0, w, 0, 1, tol)
    hit = trigs[(trigs["detector"] == 1) & (trigs["template_idx"] == inj.template) & (np.abs(trigs["sample"] - inj.end) <= 2)]
    assert len(hit) == 1
    assert stats["triggers"] > 0


# ------------------------------------------------------------------------------------------------
# edge cases: other decimation half-widths (odd K_dn runs the generic resampler), degenerate banks,
# minimal buffers, count-only calls
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", PRECISIONS)
@pytest.mark.parametrize("k_down", [7, 8, 24])
def test_other_decimation_half_widths(k_down, precision):
    w = wl.toy(n_templates=6, M=4096, spans=((2048, 0.0, 0.25), (512, 0.25, 1.0), (128, 1.0, 2.0)), seconds=6.0,
               n_basis=[10, 12, 9], f_low=25.0, mc=(1.2, 1.3))
    w.k_down = k_down
    w.peak_window = 512
    _, _, _, _, stats = _dense_check(w, precision, 0, w.n_samples)
    assert stats["checked"] == 6 * (w.n_samples // 512)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_single_template_single_basis_vector(precision):
    w = wl.toy(n_templates=1, M=512, spans=((2048, 0.0, 0.125), (1024, 0.125, 0.25)), seconds=2.0, n_basis=[1, 1], f_low=40.0)
    w.peak_window = 256
    w.threshold = 1.0
    _, _, _, info, stats = _dense_check(w, precision, 0, w.n_samples)
    assert stats["checked"] == w.n_samples // 256 and stats["triggers"] > 0


@pytest.mark.parametrize("precision", PRECISIONS)
def test_minimal_buffers_and_count_only_calls(cfg1, precision):
    """Buffers of exactly the largest decimation factor (4 samples here) for a stretch of the stream, and a call
    with capacity 0 / no trigger buffer: the count is still exact and overflow is reported by lloid_check_count."""
    import torch
    w = cfg1
    n = w.n_samples
    one, _, _ = pu.run_gpu(w, precision)
    pieces = [8192] + [4] * 64 + [n - 8192 - 256]
    many, _, info = pu.run_gpu(w, precision, pieces=pieces)
    assert _as_set(one) == _as_set(many) and info["consumed"] == n
    bank = lb.Bank(w, precision)
    strain = torch.from_numpy(w.strain).cuda()
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    lb.lloid_filter(bank.handle, strain.data_ptr(), n, 0, 0, cnt.data_ptr())
    torch.cuda.synchronize()
    assert int(cnt.item()) == len(one)
    assert lb.lloid_check_count(int(cnt.item()), 0) == lb.LLOID_EOVERFLOW
    bank.close()


def test_fp16_bank_outside_the_tensor_limits_runs_the_cuda_core_reconstruction():
    """Three 512 Hz slices with L_pad = 320 each: K = 960 at one rate, more than the tensor reconstruction kernels hold.
    The bin's FIR still runs on tcgen05; its reconstruction falls back, inside the library and on the GPU, to the FFMA
    kernels reading the packed fp16 operands.  Same tolerance as every fp16 test."""
    w = wl.toy(n_templates=150, M=5120, spans=((2048, 0.0, 0.25), (512, 0.25, 1.0), (512, 1.0, 1.75), (512, 1.75, 2.5)),
               seconds=7.0, n_basis=[40, 290, 290, 290], f_low=20.0, mc=(1.0, 1.4))
    w.peak_window = 512
    n = w.n_samples
    _, _, _, info, stats = _dense_check(w, lb.LLOID_F16, 6144, n)
    assert info["path"]["cuda_core_bds"] == 1, info["path"]
    assert stats["checked"] == 150 * ((n - 6144) // 512)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_non_finite_strain_silences_one_detector_for_one_history_length(precision):
    """include/lloid.h: the strain must be finite and is not checked.  What a NaN does is stated there and pinned here: every
    SNR value whose filter span covers it is NaN, a NaN never wins the peak comparison, so that detector emits nothing
    until the sample has left the carried history; the other detector is untouched and the first one recovers."""
    import copy
    w = wl.config3(n_bins=2, n_templates=24, seconds=40, n_detectors=2, n_basis=16)
    w.threshold = 3.0
    clean, _, _ = pu.run_gpu(w, precision)
    bad = copy.copy(w)
    bad.strain = w.strain.copy()
    k_nan = 20 * 2048 + 77
    bad.strain[0, k_nan] = np.nan
    got, _, info = pu.run_gpu(bad, precision)
    assert info["consumed"] == w.n_samples
    assert np.isfinite(got["snr_re"]).all() and np.isfinite(got["snr_im"]).all()          # no NaN ever reaches a trigger
    M = max(b.template_len for b in w.bins)
    key = lambda t: sorted((int(x["bin"]), int(x["template_idx"]), int(x["sample"])) for x in t)   # noqa: E731
    assert key(got[got["detector"] == 1]) == key(clean[clean["detector"] == 1])           # the other detector: identical
    d0, c0 = got[got["detector"] == 0], clean[clean["detector"] == 0]
    before = lambda t: t[t["sample"] < (k_nan // 2048) * 2048]                            # noqa: E731
    after = lambda t: t[t["sample"] >= ((k_nan + M + 4096) // 2048 + 1) * 2048]           # noqa: E731
    assert key(before(d0)) == key(before(c0)) and len(before(c0)) > 0
    assert key(after(d0)) == key(after(c0)) and len(after(c0)) > 0                        # recovered
    dead = d0[(d0["sample"] > k_nan + 64) & (d0["sample"] < k_nan + min(b.template_len for b in w.bins) - 64)]
    assert len(dead) == 0                                                                # silent while every template covers the NaN
