"""lloid_coincidence (include/lloid.h) against the oracle's all-pairs definition
(oracle/coinc_oracle.py), on the trigger list of a real lloid_filter pass: a 3-detector config-4-shaped bank with noise
(random coincidences) and a config-2-shaped bank with the same injections in both detectors (true coincidences).
Integer work: the sets of index pairs must be equal."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import coinc_oracle as co                    # noqa: E402
from paper_2410_16416_b200 import binding as lb          # noqa: E402
from paper_2410_16416_b200 import workloads as wl        # noqa: E402


def _filter_and_match(w, max_dt, capacity=None, k_split=None):
    import torch
    bank = lb.Bank(w, lb.LLOID_F16)
    try:
        n = w.n_samples
        cap = sum(b.n_templates for b in w.bins) * w.n_detectors * (n // w.peak_window + 1)
        strain = torch.from_numpy(w.strain).cuda()
        trig = torch.zeros(cap * 32, dtype=torch.uint8, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        bank.filter(strain, trig, cnt)
        torch.cuda.synchronize()
        n_trig = int(cnt.item())
        assert 0 < n_trig <= cap
        sb = lb.lloid_coincidence_scratch_bytes(bank.handle, 0, n)
        assert sb > 0
        scratch = torch.empty(sb, dtype=torch.uint8, device="cuda")
        pcap = n_trig * 4 if capacity is None else capacity
        pairs = torch.zeros(max(1, pcap) * 16, dtype=torch.uint8, device="cuda")
        pcnt = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        for _ in range(2):                                # twice in a row: the scratch table is rebuilt by every call
            lb.lloid_coincidence(bank.handle, trig.data_ptr(), n_trig, 0, n, max_dt, scratch.data_ptr(), sb, pairs.data_ptr(), pcap,
                                 pcnt.data_ptr(), torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
        got_n = int(pcnt.item())
        t = trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:n_trig].copy()
        p = pairs.cpu().numpy().view(lb.COINC_DTYPE)[:min(got_n, pcap)].copy()
        return t, p, got_n
    finally:
        bank.close()


def test_coincidences_of_noise_triggers_three_detectors():
    w = wl.config4(n_bins=3, n_templates=96, seconds=128, n_detectors=3, n_distinct=2)
    max_dt = np.array([[0, 31, 66], [0, 0, 45], [0, 0, 0]], dtype=np.int32)        # 10, 27, 17 ms baselines + 10 samples
    t, p, got_n = _filter_and_match(w, max_dt)
    want = co.coincidences(t, max_dt)
    got = {(int(x["a"]), int(x["b"])) for x in p}
    assert got_n == len(p) == len(got)
    assert got == want and len(want) >= 10
    for a, b in got:                                       # what the records say
        assert t[a]["bin"] == t[b]["bin"] and t[a]["template_idx"] == t[b]["template_idx"] and t[a]["detector"] < t[b]["detector"]


def test_injections_are_coincident_and_overflow_is_counted():
    w = wl.config2(n_templates=120, seconds=200, n_detectors=2, n_basis=150, n_injections=4)
    max_dt = np.array([[0, 31], [0, 0]], dtype=np.int32)
    t, p, got_n = _filter_and_match(w, max_dt)
    want = co.coincidences(t, max_dt)
    got = {(int(x["a"]), int(x["b"])) for x in p}
    assert got == want
    for inj in w.injections:                               # the same signal in both detectors: one coincident pair at its end time
        hits = [(a, b) for a, b in got if t[a]["template_idx"] == inj.template and abs(int(t[a]["sample"]) - inj.end) <= 2
                and abs(int(t[b]["sample"]) - inj.end) <= 2]
        assert len(hits) == 1, inj
    few_t, few_p, few_n = _filter_and_match(w, max_dt, capacity=2)
    # (the trigger order of a second pass differs: its indices are compared with the oracle on ITS list)
    assert few_n == len(want) and len(few_p) == 2 and {(int(x["a"]), int(x["b"])) for x in few_p} <= co.coincidences(few_t, max_dt)
    with pytest.raises(lb.LloidError):                     # tolerance beyond one peak window
        _filter_and_match(w, np.array([[0, w.peak_window + 1], [0, 0]], dtype=np.int32))
