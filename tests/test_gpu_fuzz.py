"""Seeded fuzz of the CUDA path against the oracle: random shapes (window, integration, channels, stations),
storage types, threshold-set counts, footprints and kernel variants; every case through the same comparators and
tolerances as the hand-picked parity tests."""
import math
import random

import pytest

from paper_2412_14775_b200 import synth
from tests.test_gpu_parity import check

pytestmark = pytest.mark.gpu


def _case(i):
    rnd = random.Random(1000 + i)
    F = rnd.choice([1, 1, 1, 2, 4, 8])
    n_chan = rnd.choice([c for c in (1, 3, 8, 13, 16, 24, 32, 40, 64, 96) if c % F == 0])
    T = rnd.choice([2, 3, 4, 5, 6, 7, 8, 10, 12, 16, 20, 32, 64])
    wpo = rnd.choice([1, 2, 3, 5, 16, 17, 33])
    n_out = rnd.choice([1, 2, 3])
    n_st = rnd.choice([2, 3, 5, 7])
    autos = rnd.random() < 0.6
    fp16 = rnd.random() < 0.35
    K = rnd.choice([1, 1, 2, 5, 16, 17, 40])
    variant = rnd.choice(["auto", "direct", "tma"]) if K == 1 else "auto"
    w = synth.Workload(f"fuzz{i}", n_st, autos, n_chan, T * wpo * n_out, T, T * wpo, fp16=fp16, window_F=F,
                       channel_gain=rnd.random() < 0.5, burst_cell_frac=rnd.choice([0.0, 0.1, 0.4]),
                       tone_chan_frac=rnd.choice([0.0, 0.0, 0.1]))
    # reading G6 as data faults: NaN / +-Inf samples and all-zero cells at seeded positions
    faults = []
    if rnd.random() < 0.45:
        for _ in range(rnd.choice([1, 3, 8])):
            faults.append((rnd.randrange(w.n_time), rnd.randrange(w.n_cells), rnd.randrange(4), rnd.randrange(2),
                           rnd.choice([float("nan"), float("inf"), float("-inf")])))
        if rnd.random() < 0.5:
            faults.append((None, rnd.randrange(w.n_cells), None, None, 0.0))      # an all-zero cell
    return w, K, variant, faults


@pytest.mark.parametrize("i", range(48))
def test_fuzz_case(i):
    w, K, variant, faults = _case(i)

    def mutate(vis):
        v = vis.view(w.n_time, w.n_cells, 4, 2)
        for t, c, p, ri, val in faults:
            if t is None:
                v[:, c] = val
            else:
                v[t, c, p, ri] = val
    if variant == "tma" and (not w.fp16) and w.n_cells % 4:
        variant = "direct"
    W = w.window_M * w.window_F
    if K == 1:
        thr = synth.default_thresholds(W, d=0.5 + 0.5 * ((i * 7) % 10) / 10)
    else:
        thr = synth.sweep_thresholds(W, K, seed=i)
    if W < 8:   # tiny windows: the approximated null quantiles are poor, use wide hand thresholds around them
        c = (W * 1.0 + 1) / (W - 1)
        thr = [[1.0, 0.01 * c * (k + 1) / len(thr), c * (0.6 + 0.3 * k / len(thr)), 0.97 - 0.02 * k / len(thr)] for k in range(len(thr))]
    rep, out, _ = check(w, thr, variant, seed=5000 + i, mutate=mutate if faults else None)
    assert rep["K"] == len(thr)
    import numpy as np
    assert np.isfinite(out["avg"]).all()
    for t, c, p, ri, val in faults:
        if t is not None:                                 # the window holding a non-finite sample is flagged by every set
            cells = range(c - c % w.window_F, c - c % w.window_F + w.window_F)     # ... for its whole T x F footprint
            assert all(out["flags"][k][t // w.window_M, cc] for k in range(len(thr)) for cc in cells)
    assert rep["flag_mismatch_unexplained"] == 0 or w.fp16
