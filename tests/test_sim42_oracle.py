"""Pins of the section-4.2 simulator oracle (oracle/sim42_oracle.py) against what the paper and the mathematics fix
(PAPER.md:219-237).  Each pin is chosen so that a plausible mistake in the recipe fails it."""
import math

import numpy as np
import pytest

from oracle import sim42_oracle as so


def cfg(**kw):
    base = dict(n_time=40, n_chan=16, n_real=2, n_sources=5, n_broadband=2, n_narrowband=1, n_narrowdur=1, inr=10.0, seed=7,
                window_T=10, window_F=2)
    base.update(kw)
    return so.Sim42Config(**base)


# ---- the counter-based generator: published known-answer vectors, then what the construction fixes -------
def _philox_kat():
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "philox_kat.txt")
    rows = [[int(w, 16) for w in line.split()] for line in open(path) if line.strip() and not line.startswith("#")]
    assert len(rows) == 3 and all(len(r) == 10 for r in rows)
    return rows


def test_philox_reproduces_the_published_known_answer_vectors():
    """The restatement IS Philox-4x32-10: counter, key -> output of tests/golden/philox_kat.txt (SC'11 / Random123)."""
    for row in _philox_kat():
        c, key, want = row[:4], row[4:6], row[6:]
        got = so.philox4x32(*[np.uint64(x) for x in c], seed=key[0] | (key[1] << 32))
        assert [int(x) for x in got] == want, [hex(int(x)) for x in got]


def test_philox_is_a_bijection_of_the_counter_and_depends_on_every_input():
    """Philox is a keyed permutation of the 128-bit counter: distinct counters -> distinct outputs; one changed bit
    of counter or key changes about half of the 128 output bits (avalanche)."""
    j = np.arange(4096)
    out = np.stack(so.philox4x32(j, 0, 0, 3, seed=11), 1)
    assert len({tuple(row) for row in out.tolist()}) == 4096
    base = np.stack(so.philox4x32(np.uint64(5), 6, 7, 8, seed=9)).astype(np.uint64)
    for args, seed in (((4, 6, 7, 8), 9), ((5, 7, 7, 8), 9), ((5, 6, 6, 8), 9), ((5, 6, 7, 9), 9), ((5, 6, 7, 8), 8),
                       ((5, 6, 7, 8), 9 + (1 << 32))):
        other = np.stack(so.philox4x32(*[np.uint64(a) for a in args], seed=seed)).astype(np.uint64)
        flipped = sum(bin(int(a) ^ int(b)).count("1") for a, b in zip(base.flatten(), other.flatten()))
        assert 34 <= flipped <= 94                             # 128 bits, p = 1/2: mean 64, sigma 5.7 (> 5 sigma band)


def test_philox_words_are_uniform_and_uncorrelated():
    n = 1 << 16
    x = np.stack(so.philox4x32(np.arange(n), 0, 1, 0, seed=123), 1).astype(np.float64) / 2.0 ** 32     # [n, 4]
    for q in range(4):
        hist, _ = np.histogram(x[:, q], bins=64, range=(0, 1))
        chi2 = ((hist - n / 64) ** 2 / (n / 64)).sum()
        assert chi2 < 63 + 6 * math.sqrt(2 * 63)                # chi^2_63: mean 63, sigma 11.2
        assert abs(x[:, q].mean() - 0.5) < 5 / math.sqrt(12 * n)
    c = np.corrcoef(x.T)
    assert np.abs(c - np.eye(4)).max() < 5 / math.sqrt(n)
    assert abs(np.corrcoef(x[:-1, 0], x[1:, 0])[0, 1]) < 5 / math.sqrt(n)    # consecutive counters


def test_normal_pairs_are_standard_normal_and_exactly_representable_inputs():
    n = 1 << 17
    x = so.philox4x32(np.arange(n), 0, 1, 1, seed=5)
    z0, z1 = so.normal_pair(x[0], x[1])
    z = np.concatenate([z0, z1])
    assert abs(z.mean()) < 5 / math.sqrt(2 * n) and abs(z.var() - 1) < 5 * math.sqrt(2 / (2 * n))
    assert abs((z ** 4).mean() - 3) < 0.1                       # Gaussian kurtosis
    assert abs(np.corrcoef(z0, z1)[0, 1]) < 5 / math.sqrt(n)
    # the transform's inputs are exact in float32 (so an fp32 implementation sees the same u and angle)
    ua = (2.0 * (x[0] >> np.uint32(9)).astype(np.float64) + 1.0) * 2.0 ** -24
    assert (ua.astype(np.float32).astype(np.float64) == ua).all() and ua.min() > 0 and ua.max() < 1


# ---- noise -----------------------------------------------------------------------------
def test_noise_power_per_term():
    """receiver noise e_p e_q^H has unit power per correlation (E|e|^2 = 1 for both voltages), sky noise unit power:
    total power per correlation = a^2 + 1; the four receiver terms are a rank-1 outer product."""
    c = cfg(n_time=256, n_chan=64, n_sources=0, n_broadband=0, n_narrowband=0, n_narrowdur=0, inr=0.0)
    p = so.draw_params(c, 0)
    assert 0.0 < p["a"] < 100.0
    n = so.noise(c, p, 0)
    npts = c.n_time * c.n_chan
    pw = (np.abs(n) ** 2).mean((0, 1))
    # var of |a e1 e2* + s|^2: dominated by the product term, E|e1|^4 E|e2|^4 = 4 -> relative sigma ~ sqrt(3/npts)
    assert np.allclose(pw, p["a"] ** 2 + 1, rtol=6 * math.sqrt(3.0 / npts) + 0.02)
    p1 = dict(p, a=1.0); p0 = dict(p, a=0.0)
    rx = so.noise(c, p1, 0) - so.noise(c, p0, 0)               # the receiver term alone
    det = rx[..., 0] * rx[..., 3] - rx[..., 1] * rx[..., 2]    # xx yy - xy yx = 0 for an outer product
    assert np.abs(det).max() < 1e-12 * (np.abs(rx) ** 2).max()
    sky = so.noise(c, p0, 0)
    assert np.allclose((np.abs(sky) ** 2).mean((0, 1)), 1.0, rtol=6 / math.sqrt(npts))
    assert np.abs(np.corrcoef(sky.reshape(-1, 4).T) - np.eye(4)).max() < 6 / math.sqrt(npts)
    assert abs((sky ** 2).mean()) < 6 / math.sqrt(npts)        # circular: E[z^2] = 0


def test_receiver_scale_is_constant_over_the_block_and_uniform_over_realisations():
    c = cfg(n_real=400)
    a = np.array([so.draw_params(c, r)["a"] for r in range(400)])
    assert 0 < a.min() and a.max() < 100 and abs(a.mean() - 50) < 5 * 100 / math.sqrt(12 * 400)


# ---- sources ---------------------------------------------------------------------------
def test_source_phase_hand_case():
    """one source, u = 300 m, l = 0.1, v = w = 0: coherence = S exp(j 2 pi f 30 / c) at f = 120 MHz + k 200 kHz / n_chan"""
    c = cfg(n_chan=8)
    p = {"S": np.array([2.5]), "kappa": np.array([300.0 * 0.1 / so.C_LIGHT])}
    s = so.source_signal(c, p)
    f = 120.0e6 + np.arange(8) * 25.0e3
    assert so.frequencies(c)[0] == 120.0e6 and so.frequencies(c)[-1] < 120.2e6
    expect = 2.5 * np.exp(2j * np.pi * f * 30.0 / 299792458.0)
    assert np.allclose(s, expect, rtol=0, atol=1e-9)
    # w term: (n - 1) with n = sqrt(1 - l^2 - m^2)
    c2 = cfg()
    pr = so.draw_params(c2, 1)
    u, v, w = pr["uvw"]
    n = np.sqrt(1 - pr["l"] ** 2 - pr["m"] ** 2)
    assert np.allclose(pr["kappa"], (u * pr["l"] + v * pr["m"] + w * (n - 1)) / 299792458.0)
    assert (np.abs(pr["l"]) <= 0.5).all() and (np.abs(pr["m"]) <= 0.5).all() and (pr["S"] >= 1).all() and (pr["S"] <= 10).all()


def test_uvw_scale_and_source_distributions():
    c = cfg(n_real=600, n_sources=50)
    uvw = np.array([so.draw_params(c, r)["uvw"] for r in range(600)])
    assert np.allclose(uvw.std(0), 300.0, rtol=5 / math.sqrt(2 * 600)) and np.abs(uvw.mean(0)).max() < 5 * 300 / math.sqrt(600)
    p = so.draw_params(cfg(n_sources=4000), 0)
    assert abs(p["S"].mean() - 5.5) < 5 * 9 / math.sqrt(12 * 4000) and abs(p["l"].mean()) < 5 / math.sqrt(12 * 4000)


def test_sources_enter_xx_and_yy_only_and_are_constant_in_time():
    c = cfg(inr=0.0, n_broadband=0, n_narrowband=0, n_narrowdur=0)
    g = so.generate(c)
    c0 = cfg(inr=0.0, n_broadband=0, n_narrowband=0, n_narrowdur=0, n_sources=0)
    g0 = so.generate(c0)
    d = g["vis"] - g0["vis"]                                   # sources only (noise draws do not depend on n_sources)
    assert np.abs(d[..., 1]).max() == 0 and np.abs(d[..., 2]).max() == 0
    assert np.allclose(d[..., 0], d[..., 3]) and np.allclose(d[0], d[-1])
    src = so.source_signal(c, so.draw_params(c, 1))
    assert np.allclose(d[5, 1, :, 0] + d[5, 1, :, 3], src)     # Stokes I = xx + yy carries the full coherence


# ---- RFI ---------------------------------------------------------------------------
def test_rfi_polarisation_vectors():
    c = cfg(n_real=60)
    ps, tries = [], []
    for r in range(60):
        for comp in so.draw_params(c, r)["components"]:
            J = comp["J"]
            assert abs((np.abs(J) ** 2).sum() - 1.0) < 1e-12   # J / ||J||
            ps.append(so.polarised_fraction(J)); tries.append(comp["tries"])
    ps = np.array(ps)
    assert ps.max() <= 0.9 + 1e-12 and ps.min() >= 0           # the 90 % cut
    assert 1.05 < np.mean(tries) < 1.9                         # P(p > 0.9) = 1 - 0.9^3 = 0.271 for a 2x2 complex Gaussian matrix
    # textbook coherencies: identity -> unpolarised, rank one -> fully polarised
    assert so.polarised_fraction([1, 0, 0, 1]) == 0.0
    assert abs(so.polarised_fraction([1, 0, 1j, 0]) - 1.0) < 1e-12
    cu = cfg(polarized=False)
    J = so.draw_params(cu, 0)["components"][0]["J"]
    assert np.allclose(J, np.array([1, 0, 0, 1]) / math.sqrt(2))
    I, Q, U, V = J[0] + J[3], J[0] - J[3], J[1] + J[2], 1j * (J[1] - J[2])
    assert abs(I) > 1 and Q == 0 and U == 0 and V == 0          # Eq.(2): completely unpolarised


def test_polarised_fraction_distribution_closed_form():
    """p of J J^H for a 2x2 complex Gaussian J has density 3 p^2 on [0,1] (eigenvalues of a complex Wishart(2,2))."""
    rng = np.random.default_rng(1)
    J = (rng.standard_normal((20000, 4)) + 1j * rng.standard_normal((20000, 4))) / math.sqrt(2)
    p = np.array([so.polarised_fraction(j) for j in J[:4000]])
    for q in (0.3, 0.6, 0.9):
        assert abs((p <= q).mean() - q ** 3) < 5 * math.sqrt(q ** 3 * (1 - q ** 3) / 4000)


def test_footprints_and_field():
    c = cfg(n_time=80, n_chan=32, n_real=30)
    for r in range(30):
        p = so.draw_params(c, r)
        field, support = so.rfi_signal(c, p)
        kinds = [k["kind"] for k in p["components"]]
        assert kinds == [0, 0, 1, 2]
        for comp in p["components"]:
            assert 0 <= comp["t0"] < comp["t1"] <= c.n_time and 0 <= comp["c0"] < comp["c1"] <= c.n_chan
        nb, nd = p["components"][2], p["components"][3]
        assert (nb["t0"], nb["t1"], nb["c1"] - nb["c0"]) == (0, c.n_time, 1) and 2 <= nb["period"] <= 120
        assert (nd["c0"], nd["c1"], nd["t1"] - nd["t0"]) == (0, c.n_chan, 1) and 2 <= nd["period"] <= 1024
        # the field vanishes exactly outside the support, and a lone broadband footprint has unit amplitude
        assert (np.abs(field[~support]) == 0).all()
        one = dict(p, components=[p["components"][0]])
        f1, s1 = so.rfi_signal(c, one)
        assert np.allclose((np.abs(f1[s1]) ** 2).sum(-1), 1.0)
        # the narrowband exponential: unit modulus, phase step 2 pi / P per sample
        f2, s2 = so.rfi_signal(c, dict(p, components=[nb]))
        col = f2[:, nb["c0"], :] @ nb["J"].conj()              # <field, J> = exp(j 2 pi t / P)
        assert np.allclose(np.abs(col), 1.0) and np.allclose(col[1:] / col[:-1], np.exp(2j * np.pi / nb["period"]))
        f3, _ = so.rfi_signal(c, dict(p, components=[nd]))
        row = f3[nd["t0"], :, :] @ nd["J"].conj()
        assert np.allclose(row[1:] / row[:-1], np.exp(2j * np.pi / nd["period"]))


def test_footprint_edges_cover_the_whole_block_uniformly():
    c = cfg(n_time=10, n_chan=4, n_real=3000, n_broadband=1, n_narrowband=0, n_narrowdur=0, n_sources=0)
    t0 = np.array([so.draw_params(c, r)["components"][0]["t0"] for r in range(1500)])
    t1 = np.array([so.draw_params(c, r)["components"][0]["t1"] for r in range(1500)])
    assert t0.min() == 0 and t1.max() == 10 and (t1 > t0).all()
    assert abs((t1 - t0).mean() - (11 ** 2 - 1) / (3.0 * 11) - 1 / 11) < 0.3    # E|e0 - e1| over {0..10}^2 plus the widened ties


def test_measured_inr_equals_set_inr_and_truth_is_the_support():
    for inr in (0.5, 100.0):
        c = cfg(inr=inr, n_real=3)
        g = so.generate(c)
        assert np.allclose(g["inr_measured"], inr, rtol=1e-12)
        for r in range(3):
            p = g["params"][r]
            field, support = so.rfi_signal(c, p)
            # data - celestial = g * field: recompute the celestial part with the RFI switched off
            cel = so.generate(cfg(inr=0.0, n_real=3))["vis"][:, r]
            assert np.allclose(g["vis"][:, r] - cel, g["gain"][r] * field, atol=1e-9 * g["gain"][r])
            wt = support.reshape(4, 10, 8, 2).any(axis=(1, 3))
            assert (g["truth"][:, r] == np.repeat(wt, 2, axis=1)).all()
    g0 = so.generate(cfg(inr=0.0))
    assert not g0["truth"].any() and (g0["gain"] == 0).all()


def test_determinism_and_independence_of_realisations():
    a, b = so.generate(cfg()), so.generate(cfg())
    assert (a["vis"] == b["vis"]).all()
    assert not np.allclose(a["vis"][:, 0], a["vis"][:, 1])
    c = so.generate(cfg(seed=8))
    assert not np.allclose(a["vis"], c["vis"])
    # realisation r of a larger batch equals realisation r of a smaller one (counters carry r, not the batch size)
    d = so.generate(cfg(n_real=1))
    assert (d["vis"][:, 0] == a["vis"][:, 0]).all()
