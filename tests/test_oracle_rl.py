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


# ---------------------------------------------------------------------------------------------------------------------
# An independent restatement of the WHOLE 52-value record: numpy scalar types per group, vectorised
# over the window (the C++ oracle and the CUDA kernel loop sample by sample), every group's outputs kept, the cost and the
# conversion count read off DATA tables written out from Tables 1-2, events from an
# exact-in-double comparison.  It shares no text with oracle_rl_evaluate or csrc/rfi_rl.cu.
# ---------------------------------------------------------------------------------------------------------------------
# operation counts per group as printed (reading T10): Table 1 rows 3W, W, W, W, 1, 1, 1 + 2; Table 2 rows (W, W, W), W,
# (W, W, W), (W, W, W), (1, 1, 1), 4, 1
_T1_OPS = lambda W: [3 * W, W, W, W, 1, 1, 3]                                   # noqa: E731
_T2_OPS = lambda W: [3 * W, W, 3 * W, 3 * W, 3, 4, 1]                           # noqa: E731
# data-flow edges (producer group, consumer group, elements carried); producer 0 = the single-precision input stream
_T1_EDGES = lambda W: [(0, 1, 2 * W),      # xr_i, xi_i -> y_i                  # noqa: E731
                       (1, 2, W),          # y_i -> z_i = sqrt(y_i)
                       (1, 4, W),          # y_i -> s2
                       (2, 3, W),          # z_i -> s1
                       (3, 6, 1),          # s1 -> s12
                       (4, 7, 1),          # s2 -> the ratio
                       (5, 7, 1),          # the prefactor (W d + 1)/(W - 1) -> tau
                       (6, 7, 1)]          # s12 -> the ratio
_T2_EDGES = lambda W: [(0, 1, 3 * W),      # q_i, u_i, v_i -> squares           # noqa: E731
                       (1, 2, 3 * W),      # a_i, b_i, c_i -> p_i
                       (0, 3, 3 * W),      # q_i, u_i, v_i -> the quotients
                       (2, 3, W),          # p_i -> the quotients
                       (3, 4, 3 * W),      # qhat, uhat, vhat -> sums
                       (4, 5, 3),          # sums -> squares
                       (5, 6, 3),          # squares -> r
                       (6, 7, 1)]          # r -> comparison


def _np_cost(mask, W):
    half1 = [False] + [bool(mask >> b & 1) for b in range(0, 7)]               # index = group number, 0 = input (single)
    half2 = [False] + [bool(mask >> b & 1) for b in range(7, 14)]
    ops = sum(n * (0.6 if half1[g + 1] else 1.0) for g, n in enumerate(_T1_OPS(W)))
    ops += 2 * sum(n * (0.6 if half2[g + 1] else 1.0) for g, n in enumerate(_T2_OPS(W)))
    conv = sum(n for a, b, n in _T1_EDGES(W) if half1[a] != half1[b]) + 2 * sum(n for a, b, n in _T2_EDGES(W) if half2[a] != half2[b])
    return ops, float(conv)


class _Grp:
    """Arithmetic of one group in numpy's own float16 / float32, with the event rule of reading T13 applied to every
    operand conversion and every result (arrays: one event per element)."""

    def __init__(self, half, events):
        self.t = np.float16 if half else np.float32
        self.tiny = 2.0 ** -14 if half else 2.0 ** -126
        self.eps = self.t(2.0 ** -10 if half else 2.0 ** -23)
        self.ev = events                                                       # [overflows, underflows]

    def into(self, x):
        x = np.asarray(x)
        with np.errstate(all="ignore"):
            r = x.astype(self.t)
        if r.dtype != x.dtype and r.dtype == np.float16:                        # a narrowing conversion can round
            xd, rd = x.astype(np.float64), r.astype(np.float64)
            changed = (xd != rd) & ~(np.isnan(xd) & np.isnan(rd))
            over = changed & np.isfinite(xd) & ~np.isfinite(rd)
            under = changed & ~over & (xd != 0) & (np.abs(rd) < self.tiny)
            self.ev[0] += int(over.sum()); self.ev[1] += int(under.sum())
        return r

    def __call__(self, f, *operands):
        a = [self.into(x) for x in operands]
        with np.errstate(all="ignore"):
            r = f(*a)
            exact = f(*[v.astype(np.float64) for v in a])
        assert r.dtype == self.t
        over = np.isfinite(exact) & ~np.isfinite(r)
        under = ~over & (exact != 0) & (np.abs(r.astype(np.float64)) < self.tiny)
        self.ev[0] += int(np.sum(over)); self.ev[1] += int(np.sum(under))
        return r

    def running_sum(self, values):
        s = self.t(0)
        for v in values:
            s = self(np.add, s, v)
        return s


def _mae(mixed, exact):
    m, e = np.atleast_1d(np.asarray(mixed, np.float64)), np.atleast_1d(np.asarray(exact, np.float64))
    return math.inf if not (np.isfinite(m).all() and np.isfinite(e).all()) else float(math.fsum(np.abs(m - e)) / m.size)


def _np_rl_record(win, mask, thr, rho):
    """win float32 [W, 4, 2]; returns the 52 values of include/rfi.h's record."""
    W = win.shape[0]
    d, s_low, s_high, gamma = (np.float32(x) for x in thr)
    xx, xy, yx, yy = (win[:, p, :] for p in range(4))                           # [W, 2] = (re, im), float32
    I, Q, U = xx + yy, xx - yy, xy + yx                                          # Eq.(2) in single precision (T5)
    dxy = xy - yx
    V = np.stack([-dxy[:, 1], dxy[:, 0]], 1)                                    # j (a + j b) = -b + j a
    rec = np.zeros(52)
    for part in range(2):                                                       # T15
        cols = [I[:, part].astype(np.float64) ** 2, I[:, part].astype(np.float64) ** 4] + [X[:, part].astype(np.float64) ** 2 for X in (Q, U, V)]
        rec[5 * part:5 * part + 5] = [math.log(math.fsum(c)) / W if math.fsum(c) > 0 else -math.inf for c in cols]
    rec[10:24] = [(mask >> b) & 1 for b in range(14)]
    ev = [0, 0]
    Wf = np.float32(W)
    # ---- Table 1 ----
    g = [None] + [_Grp(bool(mask >> b & 1), ev) for b in range(7)]
    xr, xi = I[:, 0], I[:, 1]
    y = g[1](np.add, g[1](np.multiply, xr, xr), g[1](np.multiply, xi, xi))
    z = g[2](np.sqrt, y)
    s1 = g[3].running_sum(z)
    s2 = g[4].running_sum(y)
    pre = g[5](np.divide, g[5](np.add, g[5](np.multiply, Wf, d), np.float32(1)), g[5](np.subtract, Wf, np.float32(1)))
    s12 = g[6](np.multiply, s1, s1)
    ratio = g[7](np.divide, g[7](np.multiply, Wf, s2), g[7](np.add, s12, g[7].eps))
    tau = g[7](np.multiply, pre, g[7](np.subtract, ratio, np.float32(1)))
    sk_ok = bool(tau >= g[7].into(s_low)) and bool(tau <= g[7].into(s_high))
    yd = xr.astype(np.float64) ** 2 + xi.astype(np.float64) ** 2
    zd = np.sqrt(yd)
    s1d = s2d = 0.0
    for i in range(W):
        s1d += zd[i]; s2d += yd[i]
    pred = (W * float(d) + 1.0) / (W - 1.0)
    s12d = s1d * s1d
    with np.errstate(all="ignore"):
        taud = pred * (np.float64(W) * s2d / (s12d + 2.0 ** -52) - 1.0)
    sk_ok_d = bool(taud >= float(s_low)) and bool(taud <= float(s_high))
    rec[24:31] = [_mae(y, yd), _mae(z, zd), _mae(s1, s1d), _mae(s2, s2d), _mae(pre, pred), _mae(s12, s12d), _mae(tau, taud)]
    mixed, truth = (0 if sk_ok else 1), (0 if sk_ok_d else 1)
    # ---- Table 2, real parts then imaginary parts ----
    for part in range(2):
        g = [None] + [_Grp(bool(mask >> b & 1), ev) for b in range(7, 14)]
        quv = [X[:, part] for X in (Q, U, V)]
        sq = [g[1](np.multiply, x, x) for x in quv]
        p = g[2](np.add, g[2](np.sqrt, g[2](np.add, g[2](np.add, sq[0], sq[1]), sq[2])), g[2].eps)
        hat = [g[3](np.divide, x, p) for x in quv]
        # the three running sums advance together, sample by sample (Table 2 lists them as one group of rows)
        sums = [g[4].t(0)] * 3
        for i in range(W):
            sums = [g[4](np.add, sums[k], hat[k][i]) for k in range(3)]
        sqs = [g[5](np.multiply, s, s) for s in sums]
        r = g[6](np.divide, g[6](np.sqrt, g[6](np.add, g[6](np.add, sqs[0], sqs[1]), sqs[2])), Wf)
        ok = bool(g[7].into(r) <= g[7].into(gamma))
        sqd = [x.astype(np.float64) ** 2 for x in quv]
        pd = np.sqrt(sqd[0] + sqd[1] + sqd[2]) + 2.0 ** -52
        with np.errstate(all="ignore"):
            hatd = [x.astype(np.float64) / pd for x in quv]
        sumd = [0.0, 0.0, 0.0]
        for i in range(W):
            sumd = [sumd[k] + hatd[k][i] for k in range(3)]
        sqsd = [s * s for s in sumd]
        rd = math.sqrt(sqsd[0] + sqsd[1] + sqsd[2]) / W if all(map(math.isfinite, sqsd)) else math.nan
        ok_d = bool(rd <= float(gamma))
        il = lambda cols: np.stack(cols, 1).ravel()                             # noqa: E731  (sample-major, as the means do not care)
        rec[31 + 7 * part:38 + 7 * part] = [_mae(il(sq), il(sqd)), _mae(p, pd), _mae(il(hat), il(hatd)), _mae(sums, sumd),
                                            _mae(sqs, sqsd), _mae(r, rd), _mae(0.0 if ok else 1.0, 0.0 if ok_d else 1.0)]
        mixed |= (0 if ok else 2 << part); truth |= (0 if ok_d else 2 << part)
    cost, conv = _np_cost(mask, W)
    match = sum(1 for b in range(3) if (mixed >> b & 1) == (truth >> b & 1))
    rec[45:52] = [cost, conv, ev[0], ev[1], match, rho * match - cost - 0.3 * conv - (20.0 if ev[0] + ev[1] else 0.0), mixed + 8 * truth]
    return rec


def test_cost_and_conversion_tables_equal_the_oracle_for_every_mask():
    for W in (3, 20):
        for mask in range(1 << 14):
            c, v = orc.rl_cost(mask, W)
            cn, vn = _np_cost(mask, W)
            assert v == vn and math.isclose(c, cn, rel_tol=1e-13), (hex(mask), W)


@pytest.mark.parametrize("W", [3, 20])
@pytest.mark.parametrize("scale", [1e-4, 1.0, 300.0])
def test_whole_record_against_the_independent_numpy_restatement(W, scale):
    """All 52 values, 36 masks (none, all, the learned one, every second bit both ways, 31 random) x 3 windows each:
    integers exact, errors and reward to 1e-12 (relative, on top of an absolute 1e-300), features to 1e-12."""
    rng = np.random.default_rng(1000 + W)
    masks = [0, 0x3FFF, 0x3C50, 0x2AAA, 0x1555] + [int(m) for m in rng.integers(0, 1 << 14, 31)]
    win = windows(3, W, scale=scale, seed=W)
    seen_events = 0
    for mask in masks:
        got = orc.rl_evaluate(win, mask, THR, rho=3.0)
        for n in range(win.shape[0]):
            want = _np_rl_record(win[n], mask, THR, 3.0)
            for k in list(range(10, 24)) + [45, 46, 47, 48, 49, 51]:
                assert got[n, k] == want[k] or (k == 45 and math.isclose(got[n, k], want[k], rel_tol=1e-13)), (hex(mask), n, k, got[n, k], want[k])
            for k in list(range(0, 10)) + list(range(24, 45)) + [50]:
                a, b = got[n, k], want[k]
                assert (a == b) or (math.isfinite(a) and math.isfinite(b) and abs(a - b) <= 1e-12 * max(abs(a), abs(b)) + 1e-300), (hex(mask), n, k, a, b)
            seen_events += want[47] + want[48]
    if scale != 1.0:
        assert seen_events > 0                              # the half-precision groups do overflow at 300 / underflow at 1e-4
