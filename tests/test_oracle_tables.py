"""Pins for the paper-literal mixed-precision oracle (oracle/rfi_oracle_tables.cpp): Tables 1-2 of the paper,
each group in single or half precision."""
import numpy as np
import pytest

from oracle import rfi_oracle as orc

BIG = 1e30
ALL_HALF_SK, ALL_HALF_DS = 0x7F, 0x3F80


def test_round_to_half_matches_ieee_binary16():
    """to_half against numpy.float16 (IEEE binary16, round to nearest even): normals, ties, subnormals, overflow."""
    rng = np.random.default_rng(1)
    xs = np.concatenate([rng.normal(size=2000) * 10.0 ** rng.integers(-9, 6, 2000),
                         [0.0, -0.0, 65504.0, 65519.9, 65520.0, 1e6, 6e-8, 2.98e-8, 2.99e-8, 1 + 2 ** -11, 1 + 3 * 2 ** -11]])
    for x in xs.astype(np.float32):
        with np.errstate(over="ignore"):
            got, ref = orc.to_half(float(x)), float(np.float32(np.float16(x)))
        assert got == ref or (np.isnan(got) and np.isnan(ref)), x


def test_single_precision_tables_are_eq4_and_eq9():
    """mask = 0 on |I| = 1,2,3,4: s1 = 10, s2 = 30, s12 = 100, tau = (5/3)(120/(100+eps) - 1) = 1/3 to single precision;
    against the fp64 definition on random unit-scale data the literal tables agree to a few single-precision ulps
    (the eps guards move tau by ~1e-9).  Catches: brackets of Table 1 row 7 (reading T1), group order."""
    tau, f = orc.tables_sk([1, 2, 3, 4], [0, 0, 0, 0], 1.0, -BIG, BIG, 0)
    assert tau == pytest.approx(1 / 3, rel=3e-7) and f == 0
    rng = np.random.default_rng(2)
    for W in (5, 16, 20):
        v = (rng.normal(size=(W, 4)) + 1j * rng.normal(size=(W, 4))).astype(np.complex64)
        t64, r_re64, r_im64 = orc.window_stats(v.astype(np.complex128), 0.7)
        I, Q, U = v[:, 0] + v[:, 3], v[:, 0] - v[:, 3], v[:, 1] + v[:, 2]
        V = 1j * (v[:, 1] - v[:, 2])
        tau, _ = orc.tables_sk(I.real, I.imag, 0.7, -BIG, BIG, 0)
        r_re, _ = orc.tables_ds(Q.real, U.real, V.real, BIG, 0)
        r_im, _ = orc.tables_ds(Q.imag, U.imag, V.imag, BIG, 0)
        assert tau == pytest.approx(t64, rel=2e-5, abs=2e-6)
        assert r_re == pytest.approx(r_re64, rel=1e-5) and r_im == pytest.approx(r_im64, rel=1e-5)


def _np_tables(xr, xi, q, u, v, d, mask):
    """Independent restatement with numpy scalar types: every operation is a numpy float16 / float32 operation
    (numpy rounds each half operation correctly).  Returns (tau, r)."""
    T = [np.float16 if (mask >> b) & 1 else np.float32 for b in range(14)]
    eps = {np.float16: np.float16(2.0 ** -10), np.float32: np.float32(2.0 ** -23)}
    W = len(xr)
    with np.errstate(all="ignore"):
        t1, t2, t3, t4, t5, t6, t7 = T[:7]
        s1, s2 = t3(0), t4(0)
        for i in range(W):
            y = t1(t1(xr[i]) * t1(xr[i])) + t1(t1(xi[i]) * t1(xi[i]))
            z = np.sqrt(t2(y))
            s1 = s1 + t3(z)
            s2 = s2 + t4(y)
        tau = (t5(W) * t5(d) + t5(1)) / (t5(W) - t5(1))
        s12 = t6(s1) * t6(s1)
        ratio = (t7(W) * t7(s2)) / (t7(s12) + eps[t7])
        tau = t7(tau) * (ratio - t7(1))
        d1, d2, d3, d4, d5, d6, d7 = T[7:]
        qs, us, vs = d4(0), d4(0), d4(0)
        for i in range(W):
            a, b, c = d1(q[i]) * d1(q[i]), d1(u[i]) * d1(u[i]), d1(v[i]) * d1(v[i])
            p = np.sqrt((d2(a) + d2(b)) + d2(c)) + eps[d2]
            qs = qs + d4(d3(q[i]) / d3(p))
            us = us + d4(d3(u[i]) / d3(p))
            vs = vs + d4(d3(v[i]) / d3(p))
        q2, u2, v2 = d5(qs) * d5(qs), d5(us) * d5(us), d5(vs) * d5(vs)
        r = np.sqrt((d6(q2) + d6(u2)) + d6(v2)) / d6(W)
    return float(tau), float(r)


@pytest.mark.parametrize("mask", [0, ALL_HALF_SK | ALL_HALF_DS, 0x0050 | 0x3C00] + [1 << b for b in range(14)] + [0x2AAA, 0x1555])
def test_every_mask_against_the_numpy_restatement(mask):
    """Bit-for-bit: all-single, all-half, the paper's learned assignment (Tables 3-4: SK groups 5,7 half; DS groups
    4-7 half), every single-bit mask (pins the bit order) and two alternating masks."""
    rng = np.random.default_rng(mask + 3)
    for W in (4, 20):
        xr, xi, q, u, v = (rng.normal(size=W).astype(np.float32) * 3 for _ in range(5))
        tau, _ = orc.tables_sk(xr, xi, 0.8, -BIG, BIG, mask)
        r, _ = orc.tables_ds(q, u, v, BIG, mask)
        tau_np, r_np = _np_tables(xr, xi, q, u, v, np.float32(0.8), mask)
        assert tau == tau_np and r == r_np, (mask, tau, tau_np, r, r_np)


def test_half_overflow_flags_the_window():
    """y = x^2 overflows binary16 above |x| = 255.9 (the paper's overflow penalty case): s2 = inf,
    tau is not finite and the negated comparison flags."""
    xr = np.array([300, 1, 1, 1], np.float32)
    tau, f = orc.tables_sk(xr, np.zeros(4, np.float32), 1.0, 0.0, 100.0, 0x01)
    assert not np.isfinite(tau) and f == 1
    tau32, f32 = orc.tables_sk(xr, np.zeros(4, np.float32), 1.0, 0.0, 100.0, 0x00)
    assert np.isfinite(tau32) and f32 == 0


def test_decisions_and_chunk_outputs():
    """Strict comparisons in the group-7 format; chunk-level flags = SK OR DS_re OR DS_im, averages exclude flagged windows."""
    assert orc.tables_ds([1, 1, -1, 1], [0] * 4, [0] * 4, 0.5, 0)[1] == 0            # r = 0.5 - O(eps): not > gamma
    assert orc.tables_ds([1, 1, 1, 1], [0] * 4, [0] * 4, 0.9, 0)[1] == 1
    rng = np.random.default_rng(9)
    M, n_int, T, C = 8, 16, 64, 5
    vis = rng.normal(size=(T, C, 4, 2)).astype(np.float32)
    vis[16:24, 2] += np.array([[6, 0], [0, 6], [0, -6], [6, 0]], np.float32)         # polarised window on cell 2
    thr = (1.0, 0.02, 1.6, 0.75)
    res = orc.tables_process(vis, M, n_int, thr, 0)
    assert res.flags[0][2, 2] == 1
    for o in range(T // n_int):
        for c in range(C):
            keep = [w for w in range(o * 2, o * 2 + 2) if not res.flags[0][w, c]]
            assert res.weight[0, o, c] == M * len(keep)
            if keep:
                rows = np.concatenate([np.arange(w * M, (w + 1) * M) for w in keep])
                ref = vis[rows, c].astype(np.float64).mean(0)
                np.testing.assert_allclose(res.avg[0, o, c].view(np.float64).reshape(4, 2), ref, rtol=1e-12, atol=1e-15)
    # with everything in single precision the flags agree with the fp64 oracle on this data
    ref64 = orc.process(vis, M, n_int, [thr])
    assert (res.flags[0] != ref64.flags[0]).mean() < 0.02
