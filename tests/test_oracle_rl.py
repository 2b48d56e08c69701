"""Pins of the RL-environment evaluator oracle (oracle_rl_evaluate in oracle/rfi_oracle_tables.cpp; PAPER.md:149-172,
readings T10-T15): cost and conversion counts by hand from the tables, features against a closed form and a numpy
restatement, errors of single groups against numpy float16 arithmetic, overflow / underflow, the reward formula."""
import math

import numpy as np
import pytest

from oracle import rfi_oracle as orc

F = orc.RL_FIELDS
THR = (1.0, 0.05, 2.5, 0.8)


def windows(n, W, scale=1.0, seed=0):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((n, W, 4, 2)) * scale).astype(np.float32)


def test_cost_model_counted_by_hand_from_tables_1_and_2():
    W = 20
    # Table 1: 3W + W + W + W + 1 + 1 + (1 + 2) = 6W + 5; Table 2: 10 per-sample rows W each + 1 + 1 + 1 + 4 + 1 = 10W + 8, twice
    assert orc.rl_cost(0, W) == (6 * W + 5 + 2 * (10 * W + 8), 0.0)
    c, v = orc.rl_cost(0x3FFF, W)
    assert math.isclose(c, 0.6 * (26 * W + 21)) and v == 2 * W + 2 * (3 * W + 3 * W)     # only the single-precision inputs convert
    # the learned assignment (Tables 3-4): Table 1 groups 5, 7 and Table 2 groups 4-7 in half
    c, v = orc.rl_cost(0x3C50, W)
    t1 = 6 * W + 0.6 * 1 + 1 + 0.6 * 3
    t2 = 3 * W + W + 3 * W + 0.6 * (3 * W + 3 + 4 + 1)
    assert math.isclose(c, t1 + 2 * t2)
    # conversions by hand: Table 1 s2 (g4, single) -> g7 (half) and s12 (g6, single) -> g7: 2; Table 2 qhat,uhat,vhat
    # (g3, single) -> sums (g4, half): 3W per part; everything downstream stays in half
    assert v == 2 + 2 * 3 * W
    # one group in half in the middle of a chain: Table 1 group 2 only -> y converts in (W) and z converts out (W)
    assert orc.rl_cost(1 << 1, W)[1] == 2 * W
    assert orc.rl_cost(1 << 4, W)[1] == 1 and orc.rl_cost(1 << 13, W)[1] == 2      # g5 -> g7; Table 2 g6 -> g7, twice


def test_features_closed_form_and_numpy():
    W = 20
    x = np.zeros((1, W, 4, 2), np.float32)
    x[0, :, 0, 0] = 1.0; x[0, :, 3, 0] = 1.0                # xx = yy = 1: I = 2, Q = U = V = 0
    out = orc.rl_evaluate(x, 0, THR)
    f = out[0, F["features"]]
    assert math.isclose(f[0], math.log(4 * W) / W) and math.isclose(f[1], math.log(16 * W) / W)
    assert f[2] == -np.inf and f[5] == -np.inf              # log 0: empty Stokes parameters
    w = windows(3, W, 5.0, seed=1)
    out = orc.rl_evaluate(w, 0x1234, THR)
    for n in range(3):
        v = w[n].astype(np.float64).view(np.complex128).reshape(W, 4)
        I = (w[n, :, 0] + w[n, :, 3]).astype(np.float64).view(np.complex128).ravel()          # single-precision Stokes (T5)
        Q = (w[n, :, 0] - w[n, :, 3]).astype(np.float64).view(np.complex128).ravel()
        U = (w[n, :, 1] + w[n, :, 2]).astype(np.float64).view(np.complex128).ravel()
        V = 1j * (w[n, :, 1] - w[n, :, 2]).astype(np.float64).view(np.complex128).ravel()
        want = []
        for part in (np.real, np.imag):
            want += [np.log((part(I) ** 2).sum()) / W, np.log((part(I) ** 4).sum()) / W, np.log((part(Q) ** 2).sum()) / W,
                     np.log((part(U) ** 2).sum()) / W, np.log((part(V) ** 2).sum()) / W]
        assert np.allclose(out[n, F["features"]], want, rtol=1e-13)
        assert out[n, F["bits"]].tolist() == [(0x1234 >> b) & 1 for b in range(14)]


def test_mask_zero_errors_are_single_precision_rounding_and_flags_match():
    W = 20
    w = windows(200, W, 3.0, seed=2)
    out = orc.rl_evaluate(w, 0, THR, rho=3.0)
    e = out[:, F["errors"]]
    assert np.isfinite(e).all() and (e >= 0).all()
    # y ~ 36, s2 ~ 700: absolute errors of a few ulp of single precision; flags are 0/1 values
    assert e[:, 0].max() < 36 * 20 * 2 ** -23 and e[:, 3].max() < 3000 * 2 ** -20
    assert e[:, 4].max() < 2 ** -22                         # tau prefactor (Wd+1)/(W-1) ~ 1.1
    assert (out[:, F["overflow"]] == 0).all() and (out[:, F["underflow"]] == 0).all()
    near = (np.abs(e[:, 6]) > 0)                            # tau error exists but does not move a flag except at a threshold
    assert (out[:, F["matches"]] == 3).mean() > 0.98
    c, v = orc.rl_cost(0, W)
    ok = out[:, F["matches"]] == 3
    assert np.allclose(out[ok, F["reward"]], 9.0 - c)


def test_single_group_errors_against_numpy_float16():
    W = 16
    w = windows(5, W, 2.0, seed=3)
    # Table 1 group 2 in half: z_i = half(sqrt(half(y_i))), y single
    out = orc.rl_evaluate(w, 1 << 1, THR)
    for n in range(5):
        xr = w[n, :, 0, 0] + w[n, :, 3, 0]; xi = w[n, :, 0, 1] + w[n, :, 3, 1]
        y = (xr * xr).astype(np.float32) + (xi * xi).astype(np.float32)
        z_h = np.sqrt(y.astype(np.float16).astype(np.float32)).astype(np.float16).astype(np.float64)
        z_d = np.sqrt(xr.astype(np.float64) ** 2 + xi.astype(np.float64) ** 2)
        assert math.isclose(out[n, 25], np.abs(z_h - z_d).mean(), rel_tol=1e-12)
        assert out[n, 24] < 1e-5                            # group 1 stays single
    # Table 2 group 1 in half: a, b, c = half(half(q)^2)
    out = orc.rl_evaluate(w, 1 << 7, THR)
    for n in range(5):
        for part in (0, 1):
            q = w[n, :, 0, part] - w[n, :, 3, part]; u = w[n, :, 1, part] + w[n, :, 2, part]
            v = -(w[n, :, 1, 1] - w[n, :, 2, 1]) if part == 0 else (w[n, :, 1, 0] - w[n, :, 2, 0])
            abc = np.stack([q, u, v], 1)
            h = abc.astype(np.float16).astype(np.float32)
            a_h = (h * h).astype(np.float16).astype(np.float64)
            a_d = abc.astype(np.float64) ** 2
            assert math.isclose(out[n, 31 + 7 * part], np.abs(a_h - a_d).mean(), rel_tol=1e-12)


def test_overflow_and_underflow_events_and_penalty():
    W = 10
    big = np.zeros((1, W, 4, 2), np.float32); big[0, :, 0, 0] = 300.0        # I = 300: y = 90000 > 65504 in half
    out = orc.rl_evaluate(big, 1 << 0, THR, rho=3.0)
    assert out[0, F["overflow"]] >= W and out[0, 24] == np.inf
    c, v = orc.rl_cost(1, W)
    assert math.isclose(out[0, F["reward"]], 3.0 * out[0, F["matches"]] - c - 0.3 * v - 20.0)
    ok = orc.rl_evaluate(big, 0, THR)
    assert ok[0, F["overflow"]] == 0 and ok[0, F["underflow"]] == 0
    small = windows(1, W, 1e-4, seed=4)                                          # y ~ 1e-8: below the smallest normal half
    out = orc.rl_evaluate(small, 1 << 0, THR)
    assert out[0, F["underflow"]] >= W and out[0, F["overflow"]] == 0
    # |x| = 255 still fits: 255^2 = 65025 < 65504
    fit = np.zeros((1, W, 4, 2), np.float32); fit[0, :, 0, 0] = 255.0
    assert orc.rl_evaluate(fit, 1 << 0, THR)[0, F["overflow"]] == 0


def test_mixed_flags_equal_the_tables_oracle_and_fp64_flags_equal_the_fp64_oracle():
    W = 20
    w = windows(300, W, 1.0, seed=5)
    thr = (1.0, 0.3, 1.6, 0.45)
    for mask in (0, 0x3C50, 0x3FFF, 0x0155):
        out = orc.rl_evaluate(w, mask, thr)
        fl = out[:, F["flags"]].astype(int)
        # chunk view: each window is one cell's only window
        vis = np.ascontiguousarray(w.transpose(1, 0, 2, 3))                  # [W, n, 4, 2]
        ref = orc.tables_process(vis, W, W, thr, mask)
        assert (((fl & 7) != 0) == ref.flags[0, 0].astype(bool)).all()
        d = orc.process(vis, W, W, np.array([thr], np.float64))
        agree = (((fl >> 3) != 0) == d.flags[0, 0].astype(bool)).mean()
        assert agree > 0.995                                                # the literal tables in double vs Eq.(4),(9): eps guards only
    m = orc.rl_evaluate(w, 0x3FFF, thr)[:, F["matches"]]
    assert m.min() >= 0 and m.max() == 3 and m.mean() < 3.0                  # all-half does lose some flags
