"""Writes the null quantiles that paper_2412_14775_b200/synth.py carries as `_NULL_Q_AUTO` (used only to PLACE the
class-1 thresholds of the auto-correlations; parity never depends on them).  Imports only oracle/ and the shared
seeded generator; run it as `python -m tests.golden.make_null_quantiles [n_stations]` and paste the printed dict.

Per window size W: the (0.1, 1, 5, 95, 99, 99.9) % quantiles of x = W S2/S1^2 - 1 = tau / c (Eq.(4)) and
the (95, 99, 99.9) % quantiles of max(r_re, r_im) (Eq.(9)) over the auto-correlation cells of RFI-free
`synth.make_chunk` output (Hermitian Sigma + H / sqrt(n_acc) noise model)."""
import sys

import numpy as np

from oracle import rfi_oracle as orc
from paper_2412_14775_b200 import synth


def null_quantiles_auto(W: int, n_stations: int = 40, n_windows: int = 512, seed: int = 77):
    w = synth.Workload("nullq", n_stations, True, 16, W * n_windows, W, W * n_windows, channel_gain=False)
    vis, _ = synth.make_chunk(w, seed=seed)
    autos = np.repeat(synth.auto_baseline_mask(w).numpy(), w.n_chan)
    v = vis.numpy().reshape(w.n_time, w.n_cells, 4, 2)[:, autos]
    res = orc.process(v, W, w.n_int, np.array([[1.0, -np.inf, np.inf, np.inf]]))
    c = (W * 1.0 + 1) / (W - 1)
    x = (res.tau[0] / c).ravel()
    r = np.maximum(res.r_re, res.r_im).ravel()
    xq = tuple(round(float(q), 4) for q in np.quantile(x, [0.001, 0.01, 0.05, 0.95, 0.99, 0.999]))
    rq = tuple(round(float(q), 3) for q in np.quantile(r, [0.95, 0.99, 0.999]))
    return xq, rq, x.size


if __name__ == "__main__":
    ns = int(sys.argv[1]) if len(sys.argv) > 1 else 40
    print("_NULL_Q_AUTO = {")
    for W in (16, 20, 32, 64):
        xq, rq, n = null_quantiles_auto(W, ns)
        print(f"    {W}: ({xq}, {rq}),   # {n} windows")
    print("}")
