"""lloid_window_peaks_noalloc (include/lloid.h): A5 + A6 on a caller-held dense SNR series with its scratch in a static
device array (no cudaMalloc: usable under graph capture and in harnesses that forbid allocation).  Checked against the
existing path: a bank filters BASELINE config 1, lloid_debug_capture hands back the dense SNR of a stretch of windows and
lloid_filter its triggers; the new entry point, fed that same SNR, must find the same triggers -- on two calls in a row
over different stretches (the array keeps the first call's records).  Collected last on purpose (file name)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2410_16416_b200 import binding as lb          # noqa: E402
from paper_2410_16416_b200 import workloads as wl        # noqa: E402
import parity_util as pu                                 # noqa: E402

PRECISIONS = [pytest.param(lb.LLOID_F32, id="fp32"), pytest.param(lb.LLOID_F16, id="fp16")]


def _peaks_noalloc(snr_dev, n_templates, k_begin, W, theta, bin_=0, det=0, capacity=None):
    import torch
    rows, n = snr_dev.shape
    assert rows == 2 * n_templates and snr_dev.is_contiguous()
    capacity = n_templates * (n // W + 1) if capacity is None else capacity
    trig = torch.zeros(max(1, capacity) * 32, dtype=torch.uint8, device="cuda")
    cnt = torch.full((1,), 12345, dtype=torch.int64, device="cuda")          # must be cleared by the call
    lb.lloid_window_peaks_noalloc(snr_dev.data_ptr(), n_templates, n, snr_dev.stride(0), k_begin, W, theta, bin_, det,
                                  trig.data_ptr(), capacity, cnt.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    got = int(cnt.item())
    return trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:min(got, capacity)].copy(), got


def _by_key(trigs, W, k_lo, k_hi):
    out = {}
    for t in trigs:
        wdw = int(t["sample"]) // W
        if wdw * W >= k_lo and (wdw + 1) * W <= k_hi:
            key = (int(t["template_idx"]), wdw)
            assert key not in out
            out[key] = t
    return out


def _compare(new, old, W, theta, k_lo, k_hi, tol):
    a, b = _by_key(new, W, k_lo, k_hi), _by_key(old, W, k_lo, k_hi)
    assert len(a) == len(new), "a trigger outside the complete windows of the range"
    same = 0
    for key in set(a) | set(b):
        ta, tb = a.get(key), b.get(key)
        if ta is None or tb is None:                     # existence may differ only at the threshold
            t = ta if tb is None else tb
            assert abs(float(np.hypot(t["snr_re"], t["snr_im"])) - theta) <= tol, key
            continue
        if int(ta["sample"]) == int(tb["sample"]):
            same += 1
            assert abs(float(ta["snr_re"]) - float(tb["snr_re"])) <= tol and abs(float(ta["snr_im"]) - float(tb["snr_im"])) <= tol
        else:                                            # two near-equal maxima: both must be as high within the tolerance
            assert abs(float(np.hypot(ta["snr_re"], ta["snr_im"])) - float(np.hypot(tb["snr_re"], tb["snr_im"]))) <= 2 * tol, key
    return len(a), len(b), same


@pytest.mark.parametrize("precision", PRECISIONS)
def test_noalloc_peaks_equal_the_bank_path_on_two_calls_in_a_row(precision):
    import torch
    w = wl.config1()
    W, theta, tol = w.peak_window, w.threshold, pu.TOL[precision]
    N = w.bins[0].n_templates
    k0, n = 4 * W, 8 * W                                 # the injection (e = 19209) lies inside
    old, snr, info = pu.run_gpu(w, precision, capture=(0, 0, k0, n))
    assert not np.isnan(snr).any() and info["counts"][0] == len(old)
    old = old[(old["bin"] == 0) & (old["detector"] == 0)]
    snr_dev = torch.from_numpy(snr).cuda()
    lb.lloid_noalloc_setup()
    # call 1: the whole stretch
    new1, got1 = _peaks_noalloc(snr_dev, N, k0, W, theta)
    assert got1 == len(new1)
    n_new, n_old, same = _compare(new1, old, W, theta, k0, k0 + n, tol)
    assert n_old > 0 and abs(n_new - n_old) <= 2 and same >= 0.95 * n_old
    pu.check_triggers(new1, snr.astype(np.float64), k0, w, 0, 0, 1e-5)        # and against the SNR it was given, exactly
    # call 2, straight after: a shorter stretch that starts off the window grid (the array still holds call 1's records)
    off, n2 = 3 * W + 128, 3 * W + 256
    sub = snr_dev[:, off:off + n2].contiguous()
    new2, got2 = _peaks_noalloc(sub, N, k0 + off, W, theta, bin_=7, det=1)
    assert got2 == len(new2) and (new2["bin"] == 7).all() and (new2["detector"] == 1).all()
    lo2, hi2 = k0 + 4 * W, k0 + 6 * W                    # the complete windows inside [k0 + off, k0 + off + n2)
    assert all(lo2 <= int(t["sample"]) < hi2 for t in new2)
    n_new2, n_old2, same2 = _compare(new2, old, W, theta, lo2, hi2, tol)
    assert n_old2 > 0 and abs(n_new2 - n_old2) <= 2 and same2 >= 0.95 * n_old2
    # call 3: same input as call 1 again -> identical records (order aside)
    new3, _ = _peaks_noalloc(snr_dev, N, k0, W, theta)
    key = lambda t: sorted((int(x["template_idx"]), int(x["sample"]), float(x["snr_re"]), float(x["snr_im"])) for x in t)   # noqa: E731
    assert key(new1) == key(new3)
    # overflow is counted, not stored
    few, got = _peaks_noalloc(snr_dev, N, k0, W, theta, capacity=3)
    assert got == len(new1) and len(few) == 3


def test_noalloc_rejects_what_does_not_fit_the_static_array():
    import torch
    lim = lb.lloid_noalloc_max_records()
    assert lim == 1 << 19
    dummy = torch.zeros(64, dtype=torch.float32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    with pytest.raises(lb.LloidError) as e:              # 4096 templates x 256 tiles = 2 x the limit
        lb.lloid_window_peaks_noalloc(dummy.data_ptr(), 4096, 256 * 128, 256 * 128, 0, 2048, 4.0, 0, 0, 0, 0, cnt.data_ptr(), 0)
    assert e.value.code == lb.LLOID_EINVAL and "static scratch array" in str(e.value) and str(lim) in str(e.value)
    for bad in (dict(n=100), dict(k=64), dict(W=100), dict(stride=130)):
        with pytest.raises(lb.LloidError):
            lb.lloid_window_peaks_noalloc(dummy.data_ptr(), 1, bad.get("n", 128), bad.get("stride", 128), bad.get("k", 0),
                                          bad.get("W", 128), 4.0, 0, 0, 0, 0, cnt.data_ptr(), 0)
