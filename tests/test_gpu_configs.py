"""GPU-vs-oracle parity at BASELINE.json's sizes and shapes, through the C ABI, in the launch configuration
bench.py times (automatic chunking, whole strain in one lloid_filter call).  The oracle cannot run a full config,
so outputs are SAMPLED: the dense SNR of one peak window around an injection (all templates, one detector) is
compared element by element, the triggers of that window go through the comparison rule of tests/parity_util.py,
and properties that hold at any size are checked on everything else (one trigger per (bin, detector, template,
window) at most, every injection recovered in every detector at its injected time, replicated bins identical).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2410_16416_b200 import binding as lb          # noqa: E402
from paper_2410_16416_b200 import workloads as wl        # noqa: E402
import parity_util as pu                                 # noqa: E402

PRECISIONS = [pytest.param(lb.LLOID_F32, id="fp32"), pytest.param(lb.LLOID_F16, id="fp16")]


def _unique_keys(trigs, W):
    keys = np.stack([trigs["bin"].astype(np.int64), trigs["detector"].astype(np.int64),
                     trigs["template_idx"].astype(np.int64), trigs["sample"] // W], axis=1)
    return len(np.unique(keys, axis=0)) == len(keys)


def _noise_free_peak(w, inj) -> float:
    """|rho_p[e]| of the injection alone, from the oracle, on a short noise-free strain whose injection end has the
    same phase on every decimation grid as in the full-size strain."""
    b = w.bins[inj.bin]
    M = b.template_len
    e = M + 8192 + inj.end % 64
    x = wl.make_strain(0, 1, e + 4096, [b], [wl.Injection(inj.bin, inj.template, inj.amplitude, inj.phase, e)],
                       15.0, 1024.0, noise=False)[0].astype(np.float64)
    rows = [R[2 * inj.template:2 * inj.template + 2] for R in b.recon]
    rho = pu.oc.snr_series(x, b.slices, b.basis, rows, e, e + 1, w.k_down, w.k_up)
    return float(np.hypot(rho[0, 0], rho[1, 0]))


@pytest.fixture(scope="module")
def cfg2_full():
    return wl.config2()          # 1000 templates, 8 slices, L = 150, 2 detectors x 4096 s, 20 injections


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config2_full_size_sampled(cfg2_full, precision):
    w = cfg2_full
    W, tol = w.peak_window, pu.TOL[precision]
    inj = w.injections[13]
    det = 1
    k0 = (inj.end // W) * W                       # the peak window that holds injection 13
    trigs, snr, info = pu.run_gpu(w, precision, capture=(0, det, k0, W))
    assert info["consumed"] == w.n_samples and info["counts"][0] == len(trigs)
    rho = pu.oracle_snr(w, 0, det, k0, k0 + W)
    assert not np.isnan(snr).any()
    err = np.abs(snr - rho)
    assert err.max() <= tol, f"dense SNR error {err.max():.3e} > {tol}"
    stats = pu.check_triggers(trigs, rho, k0, w, 0, det, tol)
    assert stats["checked"] == 1000 and stats["triggers"] > 0
    # properties at full size
    assert _unique_keys(trigs, W)
    amp = np.hypot(trigs["snr_re"], trigs["snr_im"])
    assert (amp > w.threshold).all() and np.isfinite(amp).all()
    assert trigs["sample"].min() >= 0 and trigs["sample"].max() < w.n_samples
    dev = []
    for i in w.injections:                        # every injection, both detectors, at its injected time
        a0 = _noise_free_peak(w, i)               # A kappa_p times the resamplers' gain (oracle pins P6)
        assert 0.85 * i.amplitude < a0 < 1.001 * i.amplitude
        for d in range(w.n_detectors):
            hit = trigs[(trigs["detector"] == d) & (trigs["template_idx"] == i.template) & (np.abs(trigs["sample"] - i.end) <= 2)]
            assert len(hit) == 1, f"injection p={i.template} e={i.end} det={d} not recovered"
            a = float(np.hypot(hit[0]["snr_re"], hit[0]["snr_im"]))
            assert abs(a - a0) < 3.5, (a, a0, i.amplitude)        # unit noise on the peak: 40 draws stay inside 3.5 sigma
            dev.append(a - a0)
    # a 10 % gain error moves this mean by 1.3 (mean A kappa = 13); its noise is 1/sqrt(40) = 0.16, its bias
    # (Rice, peak picking over +-2 samples) under 0.1
    assert abs(np.mean(dev)) < 0.45, np.mean(dev)
    # noise trigger rate: chi^2_2 tail over ~2000 independent samples per window (0.1 - 0.5)
    rate = len(trigs) / (1000 * w.n_detectors * (w.n_samples // W))
    assert 0.05 < rate < 0.6, rate


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config3_hundred_bins_batched(precision):
    """BASELINE config 3 shape: 100 bins x 500 templates x 2 detectors, 3 slices 2048/512/128 Hz, L = 64, three
    template-length classes; shortened to 40 s of strain (cost is linear in duration)."""
    w = wl.config3(n_bins=100, n_templates=500, seconds=40, n_detectors=2, n_basis=64)
    tol = pu.TOL[precision]
    W = w.peak_window
    bin_, det = 57, 1                              # 4 s class
    k0 = 10 * W
    trigs, snr, info = pu.run_gpu(w, precision, capture=(bin_, det, k0, 2 * W))
    rho = pu.oracle_snr(w, bin_, det, k0, k0 + 2 * W)
    assert np.abs(snr - rho).max() <= tol
    pu.check_triggers(trigs, rho, k0, w, bin_, det, tol)
    assert _unique_keys(trigs, W)
    assert set(np.unique(trigs["bin"])) == set(range(100)) and set(np.unique(trigs["detector"])) == {0, 1}
    # bins of one shape class share their arrays (the paper replicates one bank): identical triggers
    strip = lambda t: sorted((int(x["detector"]), int(x["template_idx"]), int(x["sample"]), float(x["snr_re"])) for x in t)
    assert w.bins[34] is w.bins[57]
    assert strip(trigs[trigs["bin"] == 34]) == strip(trigs[trigs["bin"] == 57])
    assert strip(trigs[trigs["bin"] == 0]) != strip(trigs[trigs["bin"] == 57])


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config3_ten_bins_units_between_half_and_all_sms(precision):
    """10 bins x 2 detectors x 4 template blocks = 80 reconstruction units: more than half of the 148 SMs, fewer than
    all.  The f0 kernel then deals tiles over all SMs and most CTAs replace their stationary R mid-way (the
    whole-CTAs-per-unit rule would idle 68 SMs); same checks as the 100-bin case."""
    w = wl.config3(n_bins=10, n_templates=500, seconds=40, n_detectors=2, n_basis=64)
    tol = pu.TOL[precision]
    W = w.peak_window
    k0 = 10 * W
    for bin_, det in ((4, 1), (9, 0)):
        trigs, snr, info = pu.run_gpu(w, precision, capture=(bin_, det, k0, 2 * W))
        rho = pu.oracle_snr(w, bin_, det, k0, k0 + 2 * W)
        assert np.abs(snr - rho).max() <= tol
        pu.check_triggers(trigs, rho, k0, w, bin_, det, tol)
    assert _unique_keys(trigs, W)
    assert set(np.unique(trigs["bin"])) == set(range(10))
    strip = lambda t: sorted((int(x["detector"]), int(x["template_idx"]), int(x["sample"]), float(x["snr_re"])) for x in t)
    assert w.bins[0] is w.bins[1]                   # bins of one shape class share their arrays: identical triggers
    assert strip(trigs[trigs["bin"] == 0]) == strip(trigs[trigs["bin"] == 1])


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config4_geometry_heterogeneous_L(precision):
    """BASELINE config 4 shape: 6 slices 2048..64 Hz, M = 64 s, L(b, s) = 100 + ((37 b + 61 s) mod 201) in
    [100, 300], 3 detectors; reduced to 5 bins x 160 templates x 100 s."""
    w = wl.config4(n_bins=5, n_templates=160, seconds=100, n_detectors=3, n_distinct=2)
    Ls = sorted({s.n_basis for b in w.bins for s in b.slices})
    assert Ls[0] >= 100 and Ls[-1] > 256, Ls       # spans the L_pad <= 256 and > 256 code paths
    tol = pu.TOL[precision]
    W = w.peak_window
    k0 = 66 * W                                    # past the 64 s start-up transient
    # fp16: bins 0-3 (L_pad <= 224 on the full-rate slice) run on the tensor reconstruction kernels, bin 4 (L_pad = 256)
    # is outside their shared-memory limit and is reconstructed by the FFMA kernels in the same call
    for bin_, det in ((3, 2), (0, 0), (4, 1)):
        trigs, snr, info = pu.run_gpu(w, precision, capture=(bin_, det, k0, W))
        rho = pu.oracle_snr(w, bin_, det, k0, k0 + W)
        assert np.abs(snr - rho).max() <= tol
        pu.check_triggers(trigs, rho, k0, w, bin_, det, tol)
    assert _unique_keys(trigs, W)


@pytest.fixture(scope="module")
def cfg4_64():
    return wl.config4(n_bins=64, n_templates=1000, seconds=160, n_detectors=3, n_distinct=2)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config4_64_bins_full_template_count_chunk_2048(cfg4_64, precision):
    """BASELINE config 4 at its per-bin size: 64 bins x 1000 templates x 3 detectors, L(b, s) in [100, 300], with the chunk
    length forced to 2048 samples -- the clamp the 1000-bin bank runs into (less than one 128-row tile per chunk at
    d = 32) -- 1536 reconstruction units per detector set, injections in bins 0, 10, ..., 60.  Dense window + trigger rules
    on bin 5 (L = 285 on the full-rate slice), bin 10 (injected) and bin 63."""
    w = cfg4_64
    assert len(w.injections) == 7 and w.bins[5].slices[0].n_basis == 285
    tol = pu.TOL[precision]
    W = w.peak_window
    inj = w.injections[1]
    assert inj.bin == 10
    k0 = (inj.end // W) * W
    for bin_, det in ((5, 2), (10, 1), (63, 0)):
        trigs, snr, info = pu.run_gpu(w, precision, capture=(bin_, det, k0, W), max_chunk=2048)
        assert info["chunk"] == 2048 and info["consumed"] == w.n_samples
        rho = pu.oracle_snr(w, bin_, det, k0, k0 + W)
        assert not np.isnan(snr).any()
        assert np.abs(snr - rho).max() <= tol
        pu.check_triggers(trigs, rho, k0, w, bin_, det, tol)
        if precision == lb.LLOID_F16:
            assert info["path"]["tensor_recon"] and info["path"]["cuda_core_bds"] == 0, info["path"]   # no bin leaves tcgen05
            assert info["path"]["r_in_tmem"]                                                          # L = 285 + folded 1024 Hz slice
    assert _unique_keys(trigs, W)
    # every injection in every detector.  At SNR 8 in unit noise the peak of a 64 s chirp (most of its power below 100 Hz)
    # moves by a few samples (measured: up to 5), so the time is checked to +-8 samples here; exact indices are checked
    # against the oracle above.
    for i in w.injections:
        for d in range(w.n_detectors):
            hit = trigs[(trigs["bin"] == i.bin) & (trigs["detector"] == d) & (trigs["template_idx"] == i.template) & (np.abs(trigs["sample"] - i.end) <= 8)]
            assert len(hit) >= 1, f"injection bin={i.bin} p={i.template} e={i.end} det={d} not recovered"
            assert abs(float(np.hypot(hit["snr_re"], hit["snr_im"]).max()) - i.amplitude) < 4.5   # unit noise on an SNR-8 peak


def _as_set(trigs):
    return sorted((int(t["bin"]), int(t["detector"]), int(t["template_idx"]), int(t["sample"]),
                   float(t["snr_re"]), float(t["snr_im"])) for t in trigs)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config5_one_second_buffers_equal_one_shot(precision):
    """BASELINE config 5: the config-3 bank fed 1 s buffers with history carried (A8).  12 bins, 24 s."""
    w = wl.config3(n_bins=12, n_templates=500, seconds=24, n_detectors=2, n_basis=64)
    one, _, _ = pu.run_gpu(w, precision)
    many, _, info = pu.run_gpu(w, precision, pieces=[w.f0] * 24)
    assert info["consumed"] == w.n_samples and len(info["counts"]) == 24
    assert _as_set(one) == _as_set(many) and len(one) > 0


def test_config5_cuda_graph_replay_equals_one_shot():
    """BASELINE config 5 through a CUDA graph: ONE captured 1 s-buffer lloid_filter call, replayed for every following
    buffer (lloid_graph_safe / lloid_graph_advance), gives the triggers of the one-shot call."""
    import torch
    w = wl.config3(n_bins=12, n_templates=500, seconds=24, n_detectors=2, n_basis=64)
    one, _, _ = pu.run_gpu(w, lb.LLOID_F16)
    bank = lb.Bank(w, lb.LLOID_F16)
    try:
        f0, D = w.f0, w.n_detectors
        cap = sum(b.n_templates for b in w.bins) * D * 2
        strain = torch.from_numpy(w.strain).cuda()
        buf = torch.empty((D, f0), dtype=torch.float32, device="cuda")
        trig = torch.zeros(cap * 32, dtype=torch.uint8, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        side = torch.cuda.Stream()
        out = []
        with torch.cuda.stream(side):
            # buffer 0 eagerly (builds the work list of this buffer length), then capture a call and replay it 23 times
            buf.copy_(strain[:, :f0])
            bank.filter(buf, trig, cnt, side.cuda_stream)
            side.synchronize()
            out.append(trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:int(cnt.item())].copy())
            assert lb.lloid_graph_safe(bank.handle, f0) and not lb.lloid_graph_safe(bank.handle, f0 // 2)
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                bank.filter(buf, trig, cnt, side.cuda_stream)
            assert lb.lloid_samples_consumed(bank.handle) == f0          # the captured call has not run
            for i in range(1, 24):
                buf.copy_(strain[:, i * f0:(i + 1) * f0])
                lb.lloid_graph_advance(bank.handle, f0)
                g.replay()
                side.synchronize()
                out.append(trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:int(cnt.item())].copy())
        assert lb.lloid_samples_consumed(bank.handle) == 24 * f0
        many = np.concatenate(out)
        assert _as_set(one) == _as_set(many) and len(one) > 0
    finally:
        bank.close()


def test_two_banks_alive_and_interleaved_precisions():
    """Opt-in shared memory is a per-device function attribute: a large fp16 bank must keep working while a small bank and
    an fp32 bank are created and used next to it."""
    import torch
    big = wl.config2(n_templates=120, seconds=72, n_detectors=2, n_basis=150, n_injections=0)
    small = wl.toy(n_templates=5, M=1024, spans=((2048, 0.0, 0.125), (512, 0.125, 0.5)), seconds=2.0, n_basis=[7, 9], f_low=40.0)
    ref_big, _, _ = pu.run_gpu(big, lb.LLOID_F16)
    ref_small16, _, _ = pu.run_gpu(small, lb.LLOID_F16)
    ref_small32, _, _ = pu.run_gpu(small, lb.LLOID_F32)

    def run(bank, w):
        n = w.n_samples
        cap = sum(b.n_templates for b in w.bins) * w.n_detectors * (n // w.peak_window + 1) + 16
        strain = torch.from_numpy(w.strain).cuda()
        trig = torch.zeros(cap * 32, dtype=torch.uint8, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        lb.lloid_reset(bank.handle)
        bank.filter(strain, trig, cnt)
        torch.cuda.synchronize()
        return trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:int(cnt.item())].copy()

    b_big = lb.Bank(big, lb.LLOID_F16)
    try:
        b_s16 = lb.Bank(small, lb.LLOID_F16)        # created while the large bank is alive
        b_s32 = lb.Bank(small, lb.LLOID_F32)
        try:
            for _ in range(2):                      # interleaved
                assert _as_set(run(b_s16, small)) == _as_set(ref_small16)
                assert _as_set(run(b_big, big)) == _as_set(ref_big)
                assert _as_set(run(b_s32, small)) == _as_set(ref_small32)
        finally:
            b_s16.close(); b_s32.close()
    finally:
        b_big.close()


def _canon(t):
    return t[np.lexsort((t["sample"], t["template_idx"], t["detector"], t["bin"]))]


def test_split_bank_equals_whole_bank(monkeypatch):
    """A bank whose chunk-local intermediates would not fit a long chunk is cut at finalize into parts (ranges of bins
    that share one set of chunk buffers and run one after the other: lloid_api.cu).  Forced here with LLOID_PARTS on a
    5-bin config-4 bank: same triggers, record for record, same captured SNR, in one call and in pieces."""
    w = wl.config4(n_bins=5, n_templates=160, seconds=100, n_detectors=3, n_distinct=2)
    W = w.peak_window
    k0 = 66 * W
    monkeypatch.setenv("LLOID_NO_SPLIT", "1")
    whole, snr_w, info_w = pu.run_gpu(w, lb.LLOID_F16, capture=(3, 1, k0, W))
    monkeypatch.delenv("LLOID_NO_SPLIT")
    monkeypatch.setenv("LLOID_PARTS", "3")
    parts, snr_p, info_p = pu.run_gpu(w, lb.LLOID_F16, capture=(3, 1, k0, W))
    assert info_p["consumed"] == w.n_samples and info_p["counts"] == info_w["counts"], (info_p, info_w)
    assert info_p["path"] == info_w["path"] and info_p["launches"] > info_w["launches"]
    assert sorted(set(parts["bin"].tolist())) == [0, 1, 2, 3, 4]
    assert _canon(parts).tobytes() == _canon(whole).tobytes()
    assert np.array_equal(snr_p, snr_w)
    host, _, _ = pu.run_gpu(w, lb.LLOID_F16, host_path=True)
    assert _canon(host).tobytes() == _canon(whole).tobytes()
    n = w.n_samples
    pieces = [W * 30, 2048 * 7 + 64, n - W * 30 - 2048 * 7 - 64]        # history, window state and counters are per part
    streamed, _, _ = pu.run_gpu(w, lb.LLOID_F16, pieces=pieces)
    monkeypatch.delenv("LLOID_PARTS")
    monkeypatch.setenv("LLOID_NO_SPLIT", "1")
    streamed_whole, _, _ = pu.run_gpu(w, lb.LLOID_F16, pieces=pieces)
    assert len(streamed) == len(whole)
    assert _canon(streamed).tobytes() == _canon(streamed_whole).tobytes()


def test_repeated_runs_are_bit_identical():
    """The same bank on the same strain gives the same trigger records, bit for bit, run after run, in both reconstruction
    modes (R in TMEM: the config-4 bank; R in shared memory: the config-2 bank).  Regression test for a race in the f0
    kernel: an interpolation issuer waited for its own tile's window rows but not for the previous tile's (which the
    other issuing thread had waited for), so about one SNR value in 10^8 was built from rows still in flight and a
    handful of near-threshold triggers came and went between identical runs."""
    banks = (wl.config4(n_bins=5, n_templates=160, seconds=100, n_detectors=3, n_distinct=2),
             wl.config2(n_templates=256, seconds=200, n_detectors=2, n_basis=150, n_injections=2))
    for w, rt in zip(banks, (True, False)):
        first = None
        for _ in range(5):
            t, _, info = pu.run_gpu(w, lb.LLOID_F16)
            assert info["path"]["r_in_tmem"] == rt
            c = _canon(t).tobytes()
            first = c if first is None else first
            assert c == first
