"""CPU oracle for the coincidence step.   TEST INFRASTRUCTURE ONLY.

Only ``tests/`` and the ``cpu_baseline`` leg of ``bench.py`` may import this module; it shares no code with the CUDA path.

PAPER.md:41: "These triggers are passed to the coincidence generator, which identifies coincidences between triggers
detected with the same template and within the light travel time between detectors."  The result has a plain
definition, so the oracle is that definition written out: every pair of triggers (i, j) with the same bin and template,
detectors a < b, and |k_i - k_j| <= max_dt[a][b] -- all pairs, checked one by one.  ``max_dt`` (light travel time plus
timing resolution, in f0 samples) is an input: the paper gives no number (reading R17).

Pins (tests/test_oracle_pins.py): hand-built cases whose answer is known by construction (a pair exactly at, one sample
inside and one sample outside the tolerance; same time but other template / other bin / same detector; three detectors)
and an independent pure-Python double loop on random small lists.
"""
from __future__ import annotations

import numpy as np


def coincidences(triggers: np.ndarray, max_dt) -> set:
    """Set of (i, j) index pairs into ``triggers`` (structured array with fields bin, detector, template_idx, sample),
    i the trigger of the lower-numbered detector.  Grouping by (bin, template) first only skips pairs that the definition
    rejects anyway; inside a group every pair is tested."""
    max_dt = np.asarray(max_dt)
    out = set()
    key = np.stack([triggers["bin"].astype(np.int64), triggers["template_idx"].astype(np.int64)], axis=1)
    order = np.lexsort((key[:, 1], key[:, 0]))
    k = key[order]
    starts = np.flatnonzero(np.r_[True, np.any(k[1:] != k[:-1], axis=1)]) if len(k) else np.zeros(0, dtype=np.int64)
    ends = np.r_[starts[1:], len(k)]
    det = triggers["detector"]
    smp = triggers["sample"]
    for s, e in zip(starts, ends):
        idx = order[s:e]
        for x in range(len(idx)):
            for y in range(len(idx)):
                i, j = int(idx[x]), int(idx[y])
                a, b = int(det[i]), int(det[j])
                if a < b and abs(int(smp[i]) - int(smp[j])) <= int(max_dt[a][b]):
                    out.add((i, j))
    return out
