"""Oracle of the on-line threshold adaptation: TEST INFRASTRUCTURE, not the product.

The paper names the problem and gives no algorithm: the hyper-parameters come from a desired false-alarm probability
("0.05"), "some fine-tuning for each data stream is necessary ... also in an online manner"
 and future work is "the dynamic adaptation of the threshold levels depending on the data streams"
(PAPER.md:275).  The reading built here (A1-A6) is a constant-false-alarm-rate rule by rank:

  A1  per baseline class (stream kind: e.g. cross / auto correlations) and per chunk, histogram tau (Eq.(4), with the
      class's d) and r_max = max(r_re, r_im) (Eq.(9)) of EVERY window with finite statistics;
  A2  bins are geometric with 64 linear sub-bins per octave, read straight off the float32 bit pattern of the value
      (index = (bits >> 17) - offset): tau in [2^-8, 2^4) -> 768 bins, r_max in [2^-6, 2^0) -> 384 bins, values below
      (incl. negative and zero) go to bin 0, values above to the last bin; relative bin width <= 1/64;
  A3  the running histogram is  acc <- forget * acc + chunk  (forget in [0,1): exponential forgetting over chunks);
  A4  quantile Q(q) of a histogram with total N: the bin where the cumulative count first reaches q N, linear
      interpolation between the bin's edges;
  A5  per-detector rate beta = 1 - sqrt(1 - alpha), so that two independent detectors OR-ed give alpha;
      s_low = Q_tau(beta/2), s_high = Q_tau(1 - beta/2) (Eq.(5) has two tails), gamma = Q_r(1 - beta) (Eq.(10));
  A6  a class with fewer than n_min counted windows keeps its thresholds; the thresholds of chunk n+1 are those
      computed after chunk n (the first chunk runs with the thresholds given a priori).

  A7  scope: the functions below serve ONE stream kind; the product keeps one state per baseline class or, with
      RFI_ADAPT_PER_BASELINE, one per baseline ("fine-tuning for each data stream") -- the tests then call
      them baseline by baseline.

  A8  (optional, off by default) loosening bound.  A1 histograms every finite window, contaminated ones included, so
      the quantiles are those of the mixture: the detector flags about alpha of ALL windows, and when the RFI occupancy
      rho of a stream exceeds alpha at least (rho - alpha) / rho of its RFI goes unflagged from the second chunk on.
      The a-priori set is the operator's statement of the null and the adaptation is "fine-tuning"
      (PAPER.md:259), so with a bound lam >= 0 an update may move a threshold at most lam * |a-priori value| in the
      loosening direction -- s_low >= s_low0 - lam |s_low0|, s_high <= s_high0 + lam |s_high0|,
      gamma <= gamma0 + lam |gamma0| -- and as far as it likes in the tightening direction.

Plain numpy / fp64; shares no code with csrc/rfi_adapt.cu; only tests/ may import it.
"""
from __future__ import annotations

import numpy as np

SUB_BITS = 6                      # 64 sub-bins per octave
TAU_LO_EXP, TAU_OCTAVES = -8, 12  # [2^-8, 2^4)
R_LO_EXP, R_OCTAVES = -6, 6       # [2^-6, 2^0)
N_TAU = TAU_OCTAVES << SUB_BITS   # 768
N_R = R_OCTAVES << SUB_BITS       # 384
N_MIN = 1000


def bin_index(values, lo_exp: int, n_bins: int):
    """A2: float32 value -> bin.  (bits >> 17) is (biased exponent << 6) | top 6 mantissa bits, monotone in the value
    for positive floats; NaN is the caller's business (it must not be counted)."""
    v = np.ascontiguousarray(values, np.float32)
    bits = v.view(np.uint32).astype(np.int64)
    idx = (bits >> (23 - SUB_BITS)) - ((127 + lo_exp) << SUB_BITS)
    idx = np.where(v <= 0, 0, idx)            # negative values and zero: first bin (sign bit would make bits huge)
    return np.clip(idx, 0, n_bins - 1)


def bin_edges(lo_exp: int, n_bins: int):
    """[n_bins + 1] edges: bin i = [2^e (1 + m/64), 2^e (1 + (m+1)/64)), e = lo_exp + i // 64, m = i % 64."""
    i = np.arange(n_bins + 1)
    e = lo_exp + (i >> SUB_BITS)
    m = i & ((1 << SUB_BITS) - 1)
    return np.ldexp(1.0 + m / float(1 << SUB_BITS), e)


def histogram(tau, r_max):
    """A1: counts of the finite windows of one class: (int64 [N_TAU], int64 [N_R])."""
    tau = np.asarray(tau, np.float32).ravel()
    r_max = np.asarray(r_max, np.float32).ravel()
    ok = np.isfinite(tau) & np.isfinite(r_max)
    ht = np.bincount(bin_index(tau[ok], TAU_LO_EXP, N_TAU), minlength=N_TAU)
    hr = np.bincount(bin_index(r_max[ok], R_LO_EXP, N_R), minlength=N_R)
    return ht.astype(np.int64), hr.astype(np.int64)


def quantile(hist, edges, q: float) -> float:
    """A4."""
    h = np.asarray(hist, np.float64)
    n = h.sum()
    target = q * n
    cum = 0.0
    for i in range(h.size):
        if h[i] > 0 and cum + h[i] >= target:
            return float(edges[i] + (edges[i + 1] - edges[i]) * ((target - cum) / h[i]))
        cum += h[i]
    return float(edges[-1])


def beta_of(alpha: float) -> float:
    return 1.0 - np.sqrt(1.0 - alpha)


def bound(new, prior, lam):
    """A8: (s_low, s_high, gamma) limited to lam * |a-priori value| of loosening; lam None or negative: no bound."""
    if lam is None or lam < 0:
        return tuple(new)
    s_low0, s_high0, gamma0 = (float(x) for x in prior)
    return (max(new[0], s_low0 - lam * abs(s_low0)), min(new[1], s_high0 + lam * abs(s_high0)),
            min(new[2], gamma0 + lam * abs(gamma0)))


def update(acc_tau, acc_r, chunk_tau, chunk_r, alpha: float, forget: float, previous, prior=None, max_loosen=None):
    """A3, A5, A6 (and A8 when max_loosen >= 0, against the a-priori set `prior`) for one class.  acc_*: float64 running
    histograms (or None); chunk_*: this chunk's counts; previous: (s_low, s_high, gamma).
    Returns (acc_tau, acc_r, (s_low, s_high, gamma))."""
    acc_tau = np.asarray(chunk_tau, np.float64) + (forget * acc_tau if acc_tau is not None else 0.0)
    acc_r = np.asarray(chunk_r, np.float64) + (forget * acc_r if acc_r is not None else 0.0)
    if acc_tau.sum() < N_MIN:
        return acc_tau, acc_r, tuple(previous)
    b = beta_of(alpha)
    et, er = bin_edges(TAU_LO_EXP, N_TAU), bin_edges(R_LO_EXP, N_R)
    new = (quantile(acc_tau, et, b / 2), quantile(acc_tau, et, 1 - b / 2), quantile(acc_r, er, 1 - b))
    return acc_tau, acc_r, bound(new, prior, max_loosen)
