"""Pins of the on-line threshold adaptation oracle (oracle/adapt_oracle.py; readings A1-A6)."""
import math

import numpy as np
import pytest

from oracle import adapt_oracle as ao


def test_bin_of_a_value_contains_the_value():
    """A2 by ordinary float arithmetic (frexp), not by the bit trick: edges[i] <= v < edges[i+1]."""
    rng = np.random.default_rng(0)
    for lo_exp, n in ((ao.TAU_LO_EXP, ao.N_TAU), (ao.R_LO_EXP, ao.N_R)):
        e = ao.bin_edges(lo_exp, n)
        assert e[0] == 2.0 ** lo_exp and e[-1] == 2.0 ** (lo_exp + n // 64) and (np.diff(e) > 0).all()
        assert ((e[1:] - e[:-1]) / e[:-1]).max() <= 1 / 64 + 1e-15              # relative bin width
        v = np.exp(rng.uniform(math.log(e[0]), math.log(e[-1]), 20000)).astype(np.float32)
        v = v[(v >= e[0]) & (v < e[-1])]
        i = ao.bin_index(v, lo_exp, n)
        assert (e[i] <= v).all() and (v < e[i + 1]).all()
        for x in v[:200]:
            m, ex = math.frexp(float(x))                                        # x = m 2^ex, m in [0.5, 1)
            assert ao.bin_index(np.float32(x), lo_exp, n) == (ex - 1 - lo_exp) * 64 + int((2 * m - 1) * 64)
        # out of range, zero and negative values
        assert ao.bin_index(np.float32([0.0, -3.0, 1e-30, e[0] * 0.999]), lo_exp, n).tolist() == [0, 0, 0, 0]
        assert ao.bin_index(np.float32([e[-1], 1e30, np.inf]), lo_exp, n).tolist() == [n - 1] * 3


def test_histogram_skips_non_finite_windows_and_counts_the_rest():
    tau = np.float32([0.5, np.nan, 1.0, np.inf, 0.25])
    r = np.float32([0.3, 0.3, np.nan, 0.3, 0.9])
    ht, hr = ao.histogram(tau, r)
    assert ht.sum() == 2 and hr.sum() == 2
    assert ht[ao.bin_index(np.float32(0.5), ao.TAU_LO_EXP, ao.N_TAU)] == 1 and hr[ao.bin_index(np.float32(0.9), ao.R_LO_EXP, ao.N_R)] == 1


def test_quantile_closed_forms():
    e = ao.bin_edges(ao.TAU_LO_EXP, ao.N_TAU)
    h = np.zeros(ao.N_TAU); h[100] = 10                                         # all mass in one bin: linear inside it
    assert ao.quantile(h, e, 0.5) == e[100] + 0.5 * (e[101] - e[100])
    assert ao.quantile(h, e, 1.0) == e[101]
    h = np.zeros(ao.N_TAU); h[10] = 1; h[20] = 3                                # q N = 1 is reached at the end of bin 10
    assert ao.quantile(h, e, 0.25) == e[11] and ao.quantile(h, e, 0.5) == e[20] + (e[21] - e[20]) / 3
    # against numpy on a large sample: within the bin width (relative 1/64) and far closer with interpolation
    rng = np.random.default_rng(1)
    v = rng.gamma(4.0, 0.1, 400000).astype(np.float32)
    ht, _ = ao.histogram(v, np.full_like(v, 0.5))
    for q in (0.0125, 0.5, 0.9875):
        assert abs(ao.quantile(ht, e, q) / np.quantile(v.astype(np.float64), q) - 1) < 2e-3


def test_beta_makes_two_independent_detectors_add_up_to_alpha():
    for a in (0.01, 0.05, 0.2):
        b = ao.beta_of(a)
        assert math.isclose(1 - (1 - b) ** 2, a, rel_tol=1e-12) and a / 2 < b < a


def test_update_holds_the_requested_false_alarm_rate_on_a_stationary_stream():
    rng = np.random.default_rng(2)
    n = 300000
    acc_t = acc_r = None
    thr = (0.0, 100.0, 1.0)
    for chunk in range(3):
        tau = rng.gamma(3.0, 0.3, n).astype(np.float32)
        r = rng.beta(2.0, 5.0, n).astype(np.float32)
        if chunk > 0:                                                           # thresholds of chunk n come from chunk n-1 (A6)
            flagged = (tau < thr[0]) | (tau > thr[1]) | (r > thr[2])
            assert abs(flagged.mean() - 0.05) < 0.003
        acc_t, acc_r, thr = ao.update(acc_t, acc_r, *ao.histogram(tau, r), alpha=0.05, forget=0.5, previous=thr)
    assert math.isclose(acc_t.sum(), n * 1.75)                                  # 1 + 0.5 + 0.25 chunks (A3)


def test_update_keeps_thresholds_below_n_min_and_forgets():
    tau = np.float32(np.linspace(0.1, 1.0, 500)); r = np.float32(np.linspace(0.1, 0.9, 500))
    a, b, thr = ao.update(None, None, *ao.histogram(tau, r), alpha=0.05, forget=0.0, previous=(1.0, 2.0, 3.0))
    assert thr == (1.0, 2.0, 3.0) and a.sum() == 500
    tau2 = np.float32(np.linspace(2.0, 3.0, 5000)); r2 = np.float32(np.linspace(0.1, 0.9, 5000))
    a, b, thr = ao.update(a, b, *ao.histogram(tau2, r2), alpha=0.05, forget=0.0, previous=thr)
    assert a.sum() == 5000 and 2.0 <= thr[0] < thr[1] <= 3.0                    # forget = 0: the old chunk is gone


def test_loosening_bound_closed_forms():
    """A8: at most lam * |a-priori value| looser, any amount tighter, sign-safe, off by default."""
    prior = (0.06, 0.52, 0.46)
    assert ao.bound((0.01, 2.0, 0.99), prior, 0.25) == (0.06 - 0.25 * 0.06, 0.52 + 0.25 * 0.52, 0.46 + 0.25 * 0.46)
    assert ao.bound((0.10, 0.40, 0.30), prior, 0.25) == (0.10, 0.40, 0.30)          # tighter than a priori: untouched
    assert ao.bound((0.01, 2.0, 0.99), prior, 0.0) == prior                         # lam = 0: never looser than a priori
    assert ao.bound((0.01, 2.0, 0.99), prior, None) == (0.01, 2.0, 0.99) == ao.bound((0.01, 2.0, 0.99), prior, -1.0)
    assert ao.bound((-3.0, 2.0, 0.9), (-1.0, 1.0, 0.5), 0.5) == (-1.5, 1.5, 0.75)   # a negative s_low loosens downwards


def _sim42_statistics(seed):
    """A section-4.2 block (five broadband footprints, two narrowband, INR 100) through the fp64
    oracle at the paper's 10 x 2 window: tau, max(r), window-level truth."""
    from oracle import rfi_oracle as orc, sim42_oracle as so
    cfg = so.Sim42Config(n_time=400, n_chan=64, n_real=4, n_sources=20, inr=100.0, seed=seed)
    ref = so.generate(cfg)
    res = orc.process(ref["vis"].reshape(cfg.n_time, cfg.n_real * cfg.n_chan, 4), 10, cfg.n_time, [[1.0, 0.0, 1e30, 1.0]], F=2)
    return res.tau[0], np.fmax(res.r_re, res.r_im), ref["truth"].reshape(-1, cfg.n_real * cfg.n_chan)


def _rates(tau, rmax, thr, truth):
    flagged = ~((tau > thr[0]) & (tau < thr[1])) | (rmax > thr[2])                  # Eq.(5), Eq.(10), OR-ed
    return (flagged & ~truth).sum() / (~truth).sum(), (~flagged & truth).sum() / truth.sum(), flagged.mean()


def test_missed_detections_when_the_rfi_occupancy_exceeds_alpha():
    """The price of A1 (every finite window is histogrammed) on the paper's own scenario, and what A8 buys back.
    Occupancy rho > alpha: the unbounded rule flags about alpha-to-a-few-alpha of all windows, so it misses at least
    (rho - flagged fraction) / rho of the RFI; with the loosening bound the thresholds stay at the a-priori ones'
    side and the missed-detection rate stays near the a-priori one."""
    from paper_2412_14775_b200 import synth
    prior = tuple(synth.default_thresholds(20)[0][1:])
    alpha = 0.05
    tau_a, r_a, truth_a = _sim42_statistics(1)
    tau_b, r_b, truth_b = _sim42_statistics(2)
    rho = truth_b.mean()
    assert truth_a.mean() > 4 * alpha and rho > 4 * alpha                           # far above alpha (about 0.55)
    ht, hr = ao.histogram(tau_a, r_a)
    free = ao.update(None, None, ht, hr, alpha, 0.0, prior)[2]
    held = ao.update(None, None, ht, hr, alpha, 0.0, prior, prior=prior, max_loosen=0.25)[2]
    assert free[0] < prior[0] and free[1] > 2 * prior[1] and free[2] > 1.5 * prior[2]   # the mixture's quantiles: far looser
    assert held == ao.bound(free, prior, 0.25) == (0.75 * prior[0], 1.25 * prior[1], 1.25 * prior[2])
    _, md_prior, _ = _rates(tau_b, r_b, prior, truth_b)
    _, md_free, frac_free = _rates(tau_b, r_b, free, truth_b)
    _, md_held, _ = _rates(tau_b, r_b, held, truth_b)
    assert md_free >= (rho - frac_free) / rho - 1e-12                               # the bound of A8's note, exactly
    assert md_free > 0.5 and md_prior < 0.05 and md_held < md_prior + 0.05
