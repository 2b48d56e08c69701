"""Pins for the fp64 oracle (oracle/rfi_oracle.cpp): what the paper and the mathematics fix.

No paper-printed worked example exists (PAPER.md prints no numeric value of tau or r), so the
oracle is pinned to closed forms, textbook identities, invariants and a brute-force restatement
in a different style (numpy complex arithmetic).  Each test names the mistake it would catch.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import rfi_oracle as orc

INF = float("inf")
NO_FLAG = [1.0, -INF, INF, INF]          # d=1, detectors disabled


def cvis(xx, xy, yx, yy):
    """[..., 4] complex128 sample(s) in the boundary's pol order (XX, XY, YX, YY)."""
    return np.stack(np.broadcast_arrays(xx, xy, yx, yy), axis=-1).astype(np.complex128)


def coherency(g, amp=1.0):
    """Rank-1 coherency  amp * g g^H  of a Jones vector g=(gx,gy) -> (xx,xy,yx,yy)."""
    gx, gy = complex(g[0]), complex(g[1])
    return amp * np.array([gx * np.conj(gx), gx * np.conj(gy), gy * np.conj(gx), gy * np.conj(gy)])


def as_chunk(windows):
    """[n_win, M, 4] complex -> one-cell chunk [n_time, 1, 4]."""
    w = np.asarray(windows, dtype=np.complex128)
    return w.reshape(-1, 1, 4)


# ----------------------------------------------------------------------------------------------
# Stokes formation, Eq.(2), reading G1
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("g,expect", [
    ((1, 0), (1, 1, 0, 0)),                               # pure X feed: Q = +I
    ((0, 1), (1, -1, 0, 0)),                              # pure Y feed: Q = -I
    ((1 / math.sqrt(2), 1 / math.sqrt(2)), (1, 0, 1, 0)),   # +45 deg linear: U = +I
    ((1 / math.sqrt(2), -1 / math.sqrt(2)), (1, 0, -1, 0)),  # -45 deg linear: U = -I
    ((1 / math.sqrt(2), 1j / math.sqrt(2)), (1, 0, 0, 1)),   # circular: V = j(xy-yx) = +I
    ((1 / math.sqrt(2), -1j / math.sqrt(2)), (1, 0, 0, -1)),
])
def test_stokes_textbook_fully_polarised(g, expect):
    """Catches: swapped xy/yx, transposed pol order, wrong sign in Q or U, V without the j."""
    v = coherency(g, 3.0)
    s = orc.stokes(v.view(np.float64))
    got = s[0::2] + 1j * s[1::2]
    np.testing.assert_allclose(got, 3.0 * np.array(expect, dtype=complex), atol=1e-15)


def test_stokes_rank1_identity_random():
    """For V_i = A e^{j phi} g g^H the triple (Q,U,V)/(A e^{j phi}) is real with Q^2+U^2+V^2 = I^2.
    Only V = j(xy-yx) satisfies it (V = xy-yx would be imaginary)."""
    rng = np.random.default_rng(1)
    for _ in range(50):
        g = rng.normal(size=2) + 1j * rng.normal(size=2)
        a = rng.uniform(0.1, 10) * np.exp(1j * rng.uniform(0, 2 * np.pi))
        v = a * coherency(g)
        s = orc.stokes(np.ascontiguousarray(v).view(np.float64))
        I, Q, U, V = (s[0::2] + 1j * s[1::2]) / a
        assert abs(I.imag) < 1e-12 and abs(Q.imag) < 1e-12 and abs(U.imag) < 1e-12 and abs(V.imag) < 1e-12
        assert Q.real ** 2 + U.real ** 2 + V.real ** 2 == pytest.approx(I.real ** 2, rel=1e-12)
        assert I.real == pytest.approx(np.linalg.norm(g) ** 2, rel=1e-12)


# ----------------------------------------------------------------------------------------------
# Spectral kurtosis, Eq.(3)-(4)
# ----------------------------------------------------------------------------------------------
def test_sk_hand_worked_window():
    """|I| = 1,2,3,4: S1=10, S2=30, W*S2/S1^2-1 = 0.2; d=1: tau = (5/3)*0.2 = 1/3; d=0.5: (3/3)*0.2.
    Catches: S1/S2 swapped, missing square, (W d+1)/(W-1) mistyped, Table-1-row-7 form (reading G3)."""
    win = cvis(np.array([1, 2, 3, 4.0]), 0, 0, 0)
    assert orc.window_stats(win, 1.0)[0] == pytest.approx(1.0 / 3.0, rel=1e-14)
    assert orc.window_stats(win, 0.5)[0] == pytest.approx(0.2, rel=1e-14)
    # the literal Table 1 row 7 reading would give (5/3)*1.2 - 1 = 1.0: make sure we are not that
    assert abs(orc.window_stats(win, 1.0)[0] - 1.0) > 0.5


def test_sk_uses_amplitude_of_complex_I():
    """|I_i| is the modulus of the complex I = xx + yy (3+4j -> 5), not the real part or the power."""
    win = cvis(np.array([3 + 4j, 5.0, 0 + 5j, -5.0]), 0, 0, 0)   # all |I| = 5
    assert orc.window_stats(win, 1.0)[0] == pytest.approx(0.0, abs=1e-15)
    win2 = cvis(np.array([1.0, 0, 0, 0]), 0, 0, np.array([0, 2j, 0, 0]))  # I = 1, 2j, 0, 0
    # S1 = 3, S2 = 5: x = 4*5/9 - 1 = 11/9, c = 5/3
    assert orc.window_stats(win2, 1.0)[0] == pytest.approx(5.0 / 3.0 * 11.0 / 9.0, rel=1e-14)


@pytest.mark.parametrize("M", [2, 5, 16, 20, 64])
def test_sk_constant_amplitude_tone_is_zero(M):
    """P1: noiseless CW tone with any phase drift has tau = 0 (north_star 'known SK for a CW tone')."""
    rng = np.random.default_rng(M)
    phase = np.exp(1j * np.cumsum(rng.uniform(-0.3, 0.3, M)))
    g = np.array([0.6, 0.8j])
    win = 2.0 * phase[:, None] * coherency(g)[None, :]
    tau, r_re, r_im = orc.window_stats(win, 1.0)
    assert abs(tau) < 1e-13


def test_sk_M2_closed_form_and_directional_two_vectors():
    """P2: M=2: tau = (2d+1)((a-b)/(a+b))^2 ; two unit vectors at angle theta: r = |cos(theta/2)|."""
    for a, b, d in [(1.0, 3.0, 1.0), (0.2, 0.7, 0.5), (5.0, 5.0, 0.8)]:
        win = cvis(np.array([a, b]), 0, 0, 0)
        assert orc.window_stats(win, d)[0] == pytest.approx((2 * d + 1) * ((a - b) / (a + b)) ** 2, rel=1e-13, abs=1e-15)
    for theta in [0.0, 0.3, 1.0, math.pi / 2, 2.5, math.pi]:
        # real-part triple (Q,U,V): sample 1 along +Q, sample 2 at angle theta in the Q-U plane
        q2, u2 = 2.0 * math.cos(theta), 2.0 * math.sin(theta)
        # Q = xx - yy, U = xy + yx with xx=-yy=Q/2 and xy=yx=U/2
        win = cvis(np.array([0.5, q2 / 2]), np.array([0.0, u2 / 2]), np.array([0.0, u2 / 2]), np.array([-0.5, -q2 / 2]))
        r_re = orc.window_stats(win, 1.0)[1]
        assert r_re == pytest.approx(abs(math.cos(theta / 2)), abs=1e-14)


@pytest.mark.parametrize("M,d", [(8, 1.0), (16, 0.5), (64, 1.0)])
def test_sk_single_spike_reaches_upper_bound(M, d):
    """P3: one sample >> the rest: W*S2/S1^2 - 1 -> W-1, tau -> W d + 1 (its maximum)."""
    amp = np.full(M, 1e-9)
    amp[M // 3] = 1.0
    tau = orc.window_stats(cvis(amp, 0, 0, 0), d)[0]
    assert tau == pytest.approx(M * d + 1, rel=1e-6)
    assert tau <= M * d + 1


def test_sk_exponential_amplitudes_unbiased_and_variance():
    """P4: |I| i.i.d. exponential, d=1: E[tau]=1, Var = 4M^2/((M-1)(M+2)(M+3)) (generalised SK,
    Nita & Gary 2010, cited PAPER.md:66).  Gamma(1/2) amplitudes with d=1/2: E[tau]=1 (pins where d enters)."""
    rng = np.random.default_rng(11)
    M, N = 16, 200_000
    amp = rng.exponential(2.5, size=(M, N))
    vis = np.zeros((M, N, 4), np.complex128)
    vis[..., 0] = amp * 0.25
    vis[..., 3] = amp * 0.75                       # I = xx + yy = amp
    res = orc.process(vis, M, M, [NO_FLAG])
    tau = res.tau[0, 0]
    var = 4.0 * M * M / ((M - 1) * (M + 2) * (M + 3))
    assert abs(tau.mean() - 1.0) < 4 * math.sqrt(var / N)
    assert tau.var() == pytest.approx(var, rel=0.05)
    # Gamma(shape 1/2): amp = g^2
    amp = rng.normal(size=(M, N)) ** 2
    vis[..., 0] = amp
    vis[..., 3] = 0
    tau = orc.process(vis, M, M, [[0.5, -INF, INF, INF]]).tau[0, 0]
    d = 0.5
    var = 2 * d * (d + 1) * M * M / ((M - 1) * (M * d + 2) * (M * d + 3))
    assert abs(tau.mean() - 1.0) < 4 * math.sqrt(var / N)
    assert tau.var() == pytest.approx(var, rel=0.06)


@pytest.mark.parametrize("M,tol", [(16, 1.5e-3), (64, 5e-4)])
def test_sk_circular_gaussian_noise_mean(M, tol):
    """P5: circular-Gaussian visibilities: |I| is Rayleigh.  Second-order delta method:
       E[W S2/S1^2] = (4/pi) (1 - (4 - 12/pi ... ) ) -- written out:  mu2/mu1^2 [1 - 2 Cov(z^2,z)/(mu2 mu1 W) + 3 Var(z)/(mu1^2 W)]
       with Rayleigh moments mu1 = s sqrt(pi/2), mu2 = 2 s^2, E z^3 = 3 s^3 sqrt(pi/2):
       = (4/pi) (1 + (3 (4/pi - 1) - 1)/W).
       With d_R = pi/(4-pi) the mean of tau is ~1 ('mean SK ~ 1 on circular-Gaussian noise')."""
    rng = np.random.default_rng(5 + M)
    N = 100_000
    z = (rng.normal(size=(M, N, 4)) + 1j * rng.normal(size=(M, N, 4))) / math.sqrt(2)
    d_r = math.pi / (4 - math.pi)
    res = orc.process(z, M, M, [[1.0, -INF, INF, INF], [d_r, -INF, INF, INF]])
    c1 = (M * 1.0 + 1) / (M - 1)
    x = res.tau[0, 0] / c1
    expect = (4 / math.pi) * (1 + (3 * (4 / math.pi - 1) - 1) / M) - 1
    assert abs(x.mean() - expect) < 4 * x.std() / math.sqrt(N) + tol
    # large-W limit 4/pi - 1 within 3 % of ... and mean tau with d_R within 3 % of 1
    assert res.tau[1, 0].mean() == pytest.approx(1.0, abs=0.03)
    # identity G10: tau_d / tau_1 = (W d + 1)/(W + 1)
    np.testing.assert_allclose(res.tau[1, 0], res.tau[0, 0] * (M * d_r + 1) / (M + 1), rtol=1e-12)


def test_sk_bounds_and_zero_window():
    """P11: -(Wd+1)/(W-1) <= tau <= Wd+1 ; all-zero window: tau = -(Wd+1)/(W-1), r = 0 (reading G4)."""
    rng = np.random.default_rng(3)
    M = 8
    for _ in range(200):
        scale = 10 ** rng.uniform(-3, 3)
        win = (rng.normal(size=(M, 4)) + 1j * rng.normal(size=(M, 4))) * scale * (rng.random((M, 1)) < 0.7)
        tau, r_re, r_im = orc.window_stats(win, 0.7)
        assert -(M * 0.7 + 1) / (M - 1) - 1e-12 <= tau <= M * 0.7 + 1 + 1e-12
        assert 0 <= r_re <= 1 + 1e-15 and 0 <= r_im <= 1 + 1e-15
    tau, r_re, r_im = orc.window_stats(np.zeros((M, 4), complex), 0.7)
    assert tau == -(M * 0.7 + 1) / (M - 1) and r_re == 0 and r_im == 0


# ----------------------------------------------------------------------------------------------
# Directional statistics, Eq.(6)-(10)
# ----------------------------------------------------------------------------------------------
def test_ds_fully_polarised_constant_signal_alignment_is_one():
    """P6: V_i = A e^{j phi} g g^H, phi fixed and not a multiple of pi/2: r_re = r_im = 1."""
    rng = np.random.default_rng(7)
    for _ in range(20):
        M = int(rng.integers(2, 40))
        g = rng.normal(size=2) + 1j * rng.normal(size=2)
        a = rng.uniform(0.1, 10) * np.exp(1j * rng.uniform(0.2, 1.3))
        amp = rng.uniform(0.5, 2.0, size=M)          # amplitude may vary: only direction matters
        win = amp[:, None] * a * coherency(g)[None, :]
        tau, r_re, r_im = orc.window_stats(win, 1.0)
        assert r_re == pytest.approx(1.0, abs=1e-13) and r_im == pytest.approx(1.0, abs=1e-13)


@pytest.mark.parametrize("M,k", [(16, 4), (16, 8), (20, 3), (10, 0), (64, 21)])
def test_ds_sign_flips(M, k):
    """P7: k of M samples sign-flipped: r = |M - 2k| / M, exactly representable cases included."""
    g = np.array([1.0, 0.0])                        # Stokes direction exactly (1,0,0)
    sign = np.ones(M)
    sign[:k] = -1
    win = sign[:, None] * (1 + 1j) * coherency(g)[None, :]
    tau, r_re, r_im = orc.window_stats(win, 1.0)
    assert r_re == abs(M - 2 * k) / M and r_im == abs(M - 2 * k) / M


def test_ds_varying_phase():
    """P7 (general): r_re = |sum sign(cos phi_i)|/M, r_im = |sum sign(sin phi_i)|/M."""
    rng = np.random.default_rng(9)
    M = 24
    phi = rng.uniform(0, 2 * np.pi, M)
    g = rng.normal(size=2) + 1j * rng.normal(size=2)
    win = np.exp(1j * phi)[:, None] * coherency(g)[None, :]
    tau, r_re, r_im = orc.window_stats(win, 1.0)
    assert r_re == pytest.approx(abs(np.sign(np.cos(phi)).sum()) / M, abs=1e-13)
    assert r_im == pytest.approx(abs(np.sign(np.sin(phi)).sum()) / M, abs=1e-13)


def test_ds_isotropic_null_second_moment():
    """P8: i.i.d. circular Gaussian pols: the (Q,U,V) real triple is isotropic, so E[r^2] = 1/M exactly
    and Var[M r^2] = 2(M-1)/(3M) (resultant of M independent uniform unit vectors in 3-D)."""
    rng = np.random.default_rng(13)
    M, N = 16, 100_000
    z = (rng.normal(size=(M, N, 4)) + 1j * rng.normal(size=(M, N, 4)))
    res = orc.process(z, M, M, [NO_FLAG])
    for r in (res.r_re[0], res.r_im[0]):
        m = (r ** 2 * M)
        assert abs(m.mean() - 1.0) < 4 * math.sqrt(2 * (M - 1) / (3 * M) / N)
        assert m.var() == pytest.approx(2 * (M - 1) / (3 * M), rel=0.05)


def test_ds_sign_of_j_cannot_matter_and_hermitian_has_zero_imag_part():
    """G1: V enters only through v^2 and (sum v)^2, so the sign of j cannot matter: swapping xy and yx
    flips the sign of (xy - yx) and must leave r unchanged.  P10: Hermitian samples (autos) have an
    identically zero imaginary triple, r_im = 0.  Purely real samples have imaginary triple
    (0, 0, xy - yx), so r_im = |sum sign(xy_i - yx_i)| / M (SURVEY.md P10 says 0; that only holds for xy = yx)."""
    rng = np.random.default_rng(17)
    M = 12
    win = rng.normal(size=(M, 4)) + 1j * rng.normal(size=(M, 4))
    swapped = win[:, [0, 2, 1, 3]]
    a = orc.window_stats(win, 1.0)
    b = orc.window_stats(swapped, 1.0)
    assert a[0] == b[0] and a[1] == pytest.approx(b[1], rel=1e-14) and a[2] == pytest.approx(b[2], rel=1e-14)
    herm = win.copy()
    herm[:, 0] = herm[:, 0].real
    herm[:, 3] = herm[:, 3].real
    herm[:, 2] = np.conj(herm[:, 1])
    assert orc.window_stats(herm, 1.0)[2] == 0.0
    real = win.real.astype(complex)
    assert orc.window_stats(real, 1.0)[2] == abs(np.sign(real[:, 1].real - real[:, 2].real).sum()) / M
    real[:, 2] = real[:, 1]
    assert orc.window_stats(real, 1.0)[2] == 0.0


def test_scale_invariance():
    """P9: multiplying a cell by c > 0 leaves tau, r and flags unchanged and scales avg by c."""
    rng = np.random.default_rng(19)
    T, C, M = 64, 5, 8
    vis = rng.normal(size=(T, C, 4)) + 1j * rng.normal(size=(T, C, 4))
    thr = [[1.0, 0.1, 0.9, 0.45]]
    a = orc.process(vis, M, 32, thr)
    for c in (2.0 ** -10, 1024.0):                   # powers of two: exact in floating point
        b = orc.process(vis * c, M, 32, thr)
        np.testing.assert_array_equal(a.flags, b.flags)
        np.testing.assert_allclose(a.tau, b.tau, rtol=1e-13)
        np.testing.assert_allclose(a.r_re, b.r_re, rtol=1e-13)
        np.testing.assert_allclose(a.avg * c, b.avg, rtol=1e-13)
    assert 0 < a.flags.mean() < 1


# ----------------------------------------------------------------------------------------------
# Decision rules Eq.(5),(10), OR-combination, readings G5, G6
# ----------------------------------------------------------------------------------------------
def test_decision_is_strict_and_ored():
    assert orc.decide(0.5, 0.1, 0.1, 0.5, 2.0, 0.3) == 0        # tau == s_low: not flagged
    assert orc.decide(2.0, 0.1, 0.1, 0.5, 2.0, 0.3) == 0        # tau == s_high: not flagged
    assert orc.decide(0.49, 0.1, 0.1, 0.5, 2.0, 0.3) == 1       # below s_low
    assert orc.decide(2.01, 0.1, 0.1, 0.5, 2.0, 0.3) == 1       # above s_high
    assert orc.decide(1.0, 0.3, 0.3, 0.5, 2.0, 0.3) == 0        # r == gamma: not flagged
    assert orc.decide(1.0, 0.31, 0.0, 0.5, 2.0, 0.3) == 1       # real part alone
    assert orc.decide(1.0, 0.0, 0.31, 0.5, 2.0, 0.3) == 1       # imaginary part alone
    assert orc.decide(float("nan"), 0.0, 0.0, -INF, INF, INF) == 1   # G6: NaN flags
    assert orc.decide(1.0, float("nan"), 0.0, -INF, INF, INF) == 1
    assert orc.decide(1e30, 1.0, 1.0, -INF, INF, INF) == 0      # disabled detectors never flag finite stats


def test_ties_on_exactly_representable_statistics():
    """G5 through the whole path: r = |16-2*4|/16 = 0.5 with gamma = 0.5 is unflagged; tau = 0 with s_low = 0 too."""
    M = 16
    sign = np.ones(M)
    sign[:4] = -1
    win = sign[:, None] * (1 + 1j) * coherency((1.0, 0.0))[None, :]
    vis = as_chunk([win])
    assert orc.process(vis, M, M, [[1.0, -INF, INF, 0.5]]).flags.item() == 0
    assert orc.process(vis, M, M, [[1.0, -INF, INF, np.nextafter(0.5, 0)]]).flags.item() == 1
    # |I| = 2 exactly for every sample: S1 = 32, S2 = 64, 16*64/1024 - 1 = 0 exactly
    vis = as_chunk([sign[:, None] * 2.0 * coherency((1.0, 0.0))[None, :]])
    assert orc.process(vis, M, M, [[1.0, -INF, INF, INF]]).tau.item() == 0.0
    assert orc.process(vis, M, M, [[1.0, 0.0, INF, INF]]).flags.item() == 0     # tau == 0 == s_low
    assert orc.process(vis, M, M, [[1.0, 1e-300, INF, INF]]).flags.item() == 1
    assert orc.process(vis, M, M, [[1.0, -INF, 0.0, INF]]).flags.item() == 0    # tau == 0 == s_high
    assert orc.process(vis, M, M, [[1.0, -INF, -1e-300, INF]]).flags.item() == 1


def test_nan_window_is_flagged_and_excluded():
    """G6: one NaN sample flags exactly its window; averages stay finite."""
    rng = np.random.default_rng(23)
    T, M = 64, 8
    vis = rng.normal(size=(T, 2, 4)) + 1j * rng.normal(size=(T, 2, 4))
    vis[19, 1, 2] = np.nan
    res = orc.process(vis, M, 32, [NO_FLAG])
    assert res.flags.sum() == 1 and res.flags[0, 19 // M, 1] == 1
    assert np.isfinite(res.avg).all()
    assert res.weight[0, 0, 1] == 32 - M and res.weight[0, 1, 1] == 32 and (res.weight[0, :, 0] == 32).all()


# ----------------------------------------------------------------------------------------------
# Exclusion + averaging, brute force, K sets
# ----------------------------------------------------------------------------------------------
def numpy_restatement(vis, M, n_int, thr):
    """A second implementation in a different style (vectorised complex numpy).  Independent of the
    C++ oracle: used only to cross-check it on small inputs (P12)."""
    vis = np.asarray(vis, np.complex128)
    T, C, _ = vis.shape
    W = T // M
    v = vis.reshape(W, M, C, 4)
    xx, xy, yx, yy = v[..., 0], v[..., 1], v[..., 2], v[..., 3]
    I, Q, U, V = xx + yy, xx - yy, xy + yx, 1j * (xy - yx)
    S1, S2 = np.abs(I).sum(1), (np.abs(I) ** 2).sum(1)
    out = []
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(S1 == 0, 0.0, M * S2 / S1 ** 2)
        rs = []
        for part in (np.real, np.imag):
            t = np.stack([part(Q), part(U), part(V)], -1)
            n = np.linalg.norm(t, axis=-1, keepdims=True)
            unit = np.where(n == 0, 0.0, t / n)
            rs.append(np.linalg.norm(unit.sum(1), axis=-1) / M)
    for d, lo, hi, g in thr:
        tau = (M * d + 1) / (M - 1) * (ratio - 1)
        flag = ~((tau >= lo) & (tau <= hi)) | ~(rs[0] <= g) | ~(rs[1] <= g)
        keep = (~flag).reshape(T // n_int, n_int // M, 1, C, 1)
        vv = v.reshape(T // n_int, n_int // M, M, C, 4)
        wsum = np.where(keep, np.nan_to_num(vv), 0).sum((1, 2))
        wt = (keep[:, :, 0, :, 0].sum(1) * M)
        avg = np.where(wt[..., None] > 0, wsum / np.maximum(wt, 1)[..., None], 0)
        out.append((tau, flag, avg, wt))
    return rs, out


def test_brute_force_random_small_chunks():
    """P12: every output of the C++ oracle against the numpy restatement on random inputs with bursts."""
    rng = np.random.default_rng(29)
    for trial in range(6):
        M = [2, 4, 5, 8, 10, 16][trial]
        n_int = M * int(rng.integers(1, 5))
        T = n_int * int(rng.integers(1, 4))
        C = int(rng.integers(1, 9))
        vis = rng.normal(size=(T, C, 4)) + 1j * rng.normal(size=(T, C, 4))
        # polarised bursts
        for _ in range(3):
            t0, c0 = int(rng.integers(0, T)), int(rng.integers(0, C))
            g = rng.normal(size=2) + 1j * rng.normal(size=2)
            vis[t0:t0 + int(rng.integers(1, M + 2)), c0] += 5 * coherency(g / np.linalg.norm(g))
        vis[:, 0, :] *= 0 if trial == 0 else 1        # an all-zero cell
        thr = [[1.0, 0.05, 1.2, 0.6], [0.5, 0.1, 0.8, 0.5], [0.8, -INF, INF, INF]]
        res = orc.process(vis, M, n_int, thr)
        rs, out = numpy_restatement(vis, M, n_int, thr)
        np.testing.assert_allclose(res.r_re, rs[0], rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(res.r_im, rs[1], rtol=1e-12, atol=1e-14)
        for k, (tau, flag, avg, wt) in enumerate(out):
            np.testing.assert_allclose(res.tau[k], tau, rtol=1e-11, atol=1e-13)
            np.testing.assert_array_equal(res.flags[k], flag.astype(np.uint8))
            np.testing.assert_array_equal(res.weight[k], wt)
            np.testing.assert_allclose(res.avg[k], avg, rtol=1e-12, atol=1e-14)
        assert 0 < res.flags[:2].mean() < 1


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_all_flag_patterns(n):
    """P12: all 2^n flagged/unflagged patterns of n windows in one output: weight = M * #unflagged,
    avg = plain mean of the unflagged samples, all-flagged output is 0 with weight 0 (reading G9)."""
    rng = np.random.default_rng(31 + n)
    M = 6
    g = np.array([0.6, 0.8j])
    for pattern in itertools.product([0, 1], repeat=n):
        wins = []
        for f in pattern:
            noise = 0.05 * (rng.normal(size=(M, 4)) + 1j * rng.normal(size=(M, 4)))
            if f:      # strong constant polarised signal: r ~ 1 -> flagged by gamma = 0.9
                wins.append(noise + 10 * (1 + 0.5j) * coherency(g))
            else:      # random polarisation per sample: r small
                wins.append(noise + rng.normal(size=(M, 4)) + 1j * rng.normal(size=(M, 4)))
        vis = as_chunk(wins)
        res = orc.process(vis, M, M * n, [[1.0, -INF, INF, 0.9]])
        np.testing.assert_array_equal(res.flags[0, :, 0], np.array(pattern, np.uint8))
        keep = [w for w, f in zip(wins, pattern) if not f]
        assert res.weight.item() == M * len(keep)
        expect = np.concatenate(keep).mean(0) if keep else np.zeros(4)
        np.testing.assert_allclose(res.avg[0, 0, 0], expect, rtol=1e-13, atol=1e-15)


def test_flag_monotonicity_and_k_sets_equal_single_runs():
    """P13: widening thresholds never adds flags; a K-set run equals K single-set runs bit for bit."""
    rng = np.random.default_rng(37)
    T, C, M = 160, 7, 10
    vis = rng.normal(size=(T, C, 4)) + 1j * rng.normal(size=(T, C, 4))
    sets = [[1.0, 0.10, 0.60, 0.40], [1.0, 0.05, 0.60, 0.40], [1.0, 0.05, 0.90, 0.40], [1.0, 0.05, 0.90, 0.55],
            [0.6, 0.05, 0.70, 0.55]]
    res = orc.process(vis, M, 40, sets)
    for k in range(3):
        assert (res.flags[k + 1] <= res.flags[k]).all()
    assert res.flags[0].sum() > res.flags[3].sum() > 0
    for k, s in enumerate(sets):
        one = orc.process(vis, M, 40, [s])
        np.testing.assert_array_equal(one.flags[0], res.flags[k])
        np.testing.assert_array_equal(one.avg[0], res.avg[k])
        np.testing.assert_array_equal(one.weight[0], res.weight[k])
        np.testing.assert_array_equal(one.tau[0], res.tau[k])


def test_burst_excised_average_is_cleaner():
    """The point of the method: a polarised burst is flagged, and the excised average is
    closer to the burst-free average than the plain average is."""
    rng = np.random.default_rng(41)
    T, M = 1024, 16
    clean = (rng.normal(size=(T, 1, 4)) + 1j * rng.normal(size=(T, 1, 4))) / math.sqrt(2)
    dirty = clean.copy()
    g = np.array([0.8, 0.6j])
    dirty[496:528, 0] += 6.0 * (1 + 1j) / math.sqrt(2) * coherency(g)      # two whole windows
    res = orc.process(dirty, M, T, [[1.0, -INF, INF, 0.62]])
    assert res.flags[0, 496 // M, 0] == 1 and res.flags[0, 527 // M, 0] == 1
    err_plain = np.abs(dirty.mean(0) - clean.mean(0)).max()
    err_excised = np.abs(res.avg[0, 0] - clean.mean(0)).max()
    assert err_excised < 0.5 * err_plain


# ----------------------------------------------------------------------------------------------
# storage widening and flag packing
# ----------------------------------------------------------------------------------------------
def test_storage_types_are_widened_exactly():
    """float16 / float32 inputs give bit-identical results to the same values passed as float64
    (all 63488 finite binary16 bit patterns go through the hand-written decoder)."""
    bits = np.arange(65536, dtype=np.uint16)
    h = bits.view(np.float16)
    h = h[np.isfinite(h)]
    n = (h.size // (8 * 8)) * 8 * 8
    v16 = h[:n].reshape(8, -1, 4, 2)
    thr = [[1.0, 0.2, 1.5, 0.7]]
    a = orc.process(v16, 4, 8, thr)
    b = orc.process(v16.astype(np.float64), 4, 8, thr)
    c = orc.process(v16.astype(np.float32), 4, 8, thr)
    for x, y in ((a, b), (c, b)):
        np.testing.assert_array_equal(x.tau, y.tau)
        np.testing.assert_array_equal(x.r_re, y.r_re)
        np.testing.assert_array_equal(x.flags, y.flags)
        np.testing.assert_array_equal(x.avg, y.avg)


@pytest.mark.parametrize("B,C", [(3, 16), (2, 64), (5, 40), (1, 1), (4, 33)])
def test_pack_flags_layout(B, C):
    """flags[row][b][c/32] bit c%32 (include/rfi.h) against numpy packbits (little bit order)."""
    rng = np.random.default_rng(B * 100 + C)
    f = (rng.random((3, 4, B * C)) < 0.3).astype(np.uint8)
    got = orc.pack_flags(f, B, C)
    wpb = (C + 31) // 32
    padded = np.zeros((3, 4, B, wpb * 32), np.uint8)
    padded[..., :C] = f.reshape(3, 4, B, C)
    expect = np.packbits(padded, axis=-1, bitorder="little").view(np.uint32).reshape(3, 4, B, wpb)
    np.testing.assert_array_equal(got, expect)


def test_invalid_arguments_rejected():
    vis = np.zeros((16, 1, 4, 2), np.float32)
    with pytest.raises(ValueError):
        orc.process(vis, 1, 16, [NO_FLAG])       # M >= 2 (Eq.(4) divides by W-1)
    with pytest.raises(ValueError):
        orc.process(vis, 3, 16, [NO_FLAG])       # n_int % M
    with pytest.raises(ValueError):
        orc.process(vis, 4, 12, [NO_FLAG])       # n_time % n_int


# ----------------------------------------------------------------------------------------------
# T x F window footprints, W = T x F (10 x 2 and 5 x 4 at PAPER.md:182,233,241)
# ----------------------------------------------------------------------------------------------
def test_tf_hand_worked_2x2():
    """2 time x 2 channel footprint with |I| = 1,2 (channel 0) and 3,4 (channel 1): the same four amplitudes as
    the hand-worked W=4 window -> x = 0.2, tau(d=1) = 1/3; all Q > 0 -> r_re = 1.  Catches: W taken as T."""
    vis = np.zeros((2, 2, 4), np.complex128)
    vis[:, 0, 0] = [1, 2]
    vis[:, 1, 0] = [3, 4]
    res = orc.process(vis, 2, 2, [NO_FLAG], F=2)
    assert res.tau[0, 0, 0] == pytest.approx(1 / 3, rel=1e-14) and res.tau[0, 0, 1] == res.tau[0, 0, 0]
    assert res.r_re[0, 0] == pytest.approx(1.0, rel=1e-14) and res.r_im[0, 1] == 0.0


@pytest.mark.parametrize("T,F", [(10, 2), (5, 4), (1, 8), (16, 1), (3, 3)])
def test_tf_window_equals_time_window_of_the_rearranged_samples(T, F):
    """The statistics are sums over the W = T*F samples of the footprint, so they must equal those of a
    per-channel window of length W holding the same samples (the F = 1 path is pinned by the closed forms above).
    Catches: a channel left out, per-channel instead of joint statistics, W = T in Eq.(4)/(9)."""
    rng = np.random.default_rng(T * 10 + F)
    n_win = 3
    vis = rng.normal(size=(n_win * T, 2 * F, 4)) + 1j * rng.normal(size=(n_win * T, 2 * F, 4))
    vis[T:2 * T, :F] += 4 * coherency(np.array([0.6, 0.8j]))          # a polarised window in group 0
    thr = [[0.7, 0.1, 1.1, 0.55]]
    res = orc.process(vis, T, T, thr, F=F)
    for grp in range(2):
        flat = vis[:, grp * F:(grp + 1) * F].reshape(n_win * T * F, 1, 4)   # window w -> rows w*T*F ... (t-major, f inner)
        ref = orc.process(flat, T * F, T * F, thr)
        for f in range(F):
            c = grp * F + f
            np.testing.assert_allclose(res.tau[0][:, c], ref.tau[0][:, 0], rtol=1e-13, atol=1e-15)
            np.testing.assert_allclose(res.r_re[:, c], ref.r_re[:, 0], rtol=1e-13, atol=1e-15)
            np.testing.assert_allclose(res.r_im[:, c], ref.r_im[:, 0], rtol=1e-13, atol=1e-15)
            np.testing.assert_array_equal(res.flags[0][:, c], ref.flags[0][:, 0])
    assert res.flags[0][1, :F].all() and not res.flags[0][1, F:].all()


def test_tf_exclusion_is_per_footprint_and_average_per_channel():
    """A burst in ONE channel flags the whole T x F footprint: both channels lose that window's
    samples, and each channel's average is the plain mean of its own remaining samples (no frequency averaging)."""
    rng = np.random.default_rng(77)
    T, F, n_win = 5, 2, 4
    vis = 0.1 * (rng.normal(size=(n_win * T, F, 4)) + 1j * rng.normal(size=(n_win * T, F, 4)))
    vis[2 * T:3 * T, 1] += 10 * coherency(np.array([0.6, 0.8j]))
    # half of the footprint at amplitude ~10, half at ~0.1: x = W S2/S1^2 - 1 ~ 1, tau ~ 11/9; noise windows ~0.3
    res = orc.process(vis, T, n_win * T, [[1.0, -INF, 1.0, INF]], F=F)
    assert res.tau[0][2, 0] == pytest.approx(11 / 9, rel=0.15) and res.tau[0][[0, 1, 3], 0].max() < 0.9
    assert res.flags[0][:, 0].tolist() == [0, 0, 1, 0] and res.flags[0][:, 1].tolist() == [0, 0, 1, 0]
    keep = np.r_[0:2 * T, 3 * T:4 * T]
    assert res.weight[0, 0].tolist() == [3 * T, 3 * T]
    for c in range(F):
        np.testing.assert_allclose(res.avg[0, 0, c], vis[keep, c].mean(0), rtol=1e-12, atol=1e-15)


def test_tf_f1_is_the_per_channel_path_and_bad_shapes_are_rejected():
    rng = np.random.default_rng(5)
    vis = rng.normal(size=(32, 6, 4)) + 1j * rng.normal(size=(32, 6, 4))
    a = orc.process(vis, 8, 16, [[1.0, 0.1, 0.9, 0.5]])
    b = orc.process(vis, 8, 16, [[1.0, 0.1, 0.9, 0.5]], F=1)
    for key in ("tau", "r_re", "r_im", "flags", "avg", "weight"):
        np.testing.assert_array_equal(getattr(a, key), getattr(b, key))
    with pytest.raises(ValueError):
        orc.process(vis, 8, 16, [NO_FLAG], F=4)           # 6 cells are not whole groups of 4
    with pytest.raises(ValueError):
        orc.process(vis, 1, 16, [NO_FLAG], F=1)           # W = 1: Eq.(4) divides by W - 1
