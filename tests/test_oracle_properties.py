"""Property tests of the fp64 oracle (hypothesis): invariants that hold for every input."""
import numpy as np
from hypothesis import given, settings, strategies as st

from oracle import rfi_oracle as orc

INF = float("inf")


@st.composite
def chunks(draw):
    M = draw(st.sampled_from([2, 3, 4, 5, 8, 10, 16]))
    F = draw(st.sampled_from([1, 1, 2, 4]))
    wpo = draw(st.integers(1, 4))
    n_out = draw(st.integers(1, 2))
    groups = draw(st.integers(1, 3))
    seed = draw(st.integers(0, 2 ** 31 - 1))
    rng = np.random.default_rng(seed)
    T, C = M * wpo * n_out, groups * F
    vis = rng.normal(size=(T, C, 4)) + 1j * rng.normal(size=(T, C, 4))
    if draw(st.booleans()):                       # a strong polarised burst somewhere
        t0, c0 = int(rng.integers(0, T)), int(rng.integers(0, C))
        g = rng.normal(size=2) + 1j * rng.normal(size=2)
        coh = np.array([g[0] * g[0].conj(), g[0] * g[1].conj(), g[1] * g[0].conj(), g[1] * g[1].conj()])
        vis[t0:t0 + int(rng.integers(1, M + 1)), c0] += draw(st.floats(0.5, 50.0)) * coh
    d = draw(st.floats(0.5, 1.0))
    return vis, M, F, M * wpo, d


@settings(max_examples=60, deadline=None)
@given(chunks(), st.floats(1e-6, 1e6))
def test_bounds_scale_invariance_and_weights(chunk, scale):
    vis, M, F, n_int, d = chunk
    W = M * F
    c = (W * d + 1) / (W - 1)
    thr = [[d, 0.1 * c, 0.6 * c, 0.55]]
    a = orc.process(vis, M, n_int, thr, F=F)
    # P11: bounds
    assert (a.tau >= -c - 1e-12).all() and (a.tau <= W * d + 1 + 1e-9).all()
    assert (a.r_re >= 0).all() and (a.r_re <= 1 + 1e-12).all() and (a.r_im >= 0).all() and (a.r_im <= 1 + 1e-12).all()
    # P9: a positive rescaling changes no statistic or flag (away from rounding of a threshold) and scales the averages
    b = orc.process(vis * scale, M, n_int, thr, F=F)
    np.testing.assert_allclose(b.tau, a.tau, rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(b.r_re, a.r_re, rtol=1e-9, atol=1e-12)
    near = (np.abs(a.tau[0] - 0.1 * c) < 1e-9) | (np.abs(a.tau[0] - 0.6 * c) < 1e-9) | (np.abs(a.r_re - 0.55) < 1e-9) | (np.abs(a.r_im - 0.55) < 1e-9)
    assert (a.flags[0] == b.flags[0])[~near].all()
    if not near.any():
        np.testing.assert_allclose(b.avg, a.avg * scale, rtol=1e-9)
    # weight = samples of the unflagged windows of the output; the F channels of a footprint share the flag
    wpo = n_int // M
    kept = (1 - a.flags[0].astype(np.int64)).reshape(-1, wpo, a.flags.shape[2]).sum(1) * M
    assert (a.weight[0] == kept).all()
    fl = a.flags[0].reshape(a.flags.shape[1], -1, F)
    assert (fl == fl[..., :1]).all()


@settings(max_examples=40, deadline=None)
@given(chunks())
def test_monotonicity_in_the_thresholds(chunk):
    vis, M, F, n_int, d = chunk
    W = M * F
    c = (W * d + 1) / (W - 1)
    tight = [d, 0.15 * c, 0.5 * c, 0.45]
    loose = [d, 0.10 * c, 0.7 * c, 0.60]
    off = [d, -INF, INF, INF]
    res = orc.process(vis, M, n_int, [tight, loose, off], F=F)
    assert (res.flags[1] <= res.flags[0]).all()          # P13: loosening any threshold never adds a flag
    assert res.flags[2].sum() == 0
    single = orc.process(vis, M, n_int, [loose], F=F)
    assert (single.flags[0] == res.flags[1]).all() and (single.avg[0] == res.avg[1]).all()
