"""GPU parity of the section-4.2 simulator (rfi_sim42_generate) against oracle/sim42_oracle.py,
element by element on the same seed, and the Fig. 2 / Fig. 3 shaped scenario through the K-set kernel.

Both sides draw the identical Philox integers; the parameter table and the source coherence are fp64 on both sides
(tolerance 1e-12 relative: libm vs CUDA math), the noise runs its Gaussian transform in fp32 on the device and in
fp64 in the oracle: |d| <= 1e-5 * max(|x|, rms(x)) per real component (same form as the averages' tolerance)."""
import math

import numpy as np
import pytest
import torch

import paper_2412_14775_b200 as rfi
from oracle import sim42_oracle as so
from paper_2412_14775_b200 import synth

pytestmark = pytest.mark.gpu


def _both(**kw):
    cfg = so.Sim42Config(**kw)
    ref = so.generate(cfg)
    vis, truth, tab, src = rfi.sim42_generate(cfg.n_real, cfg.inr, seed=cfg.seed, n_time=cfg.n_time, n_chan=cfg.n_chan,
                                              n_sources=cfg.n_sources, n_broadband=cfg.n_broadband,
                                              n_narrowband=cfg.n_narrowband, n_narrowdur=cfg.n_narrowdur,
                                              polarized=cfg.polarized, window_T=cfg.window_T, window_F=cfg.window_F,
                                              diagnostics=True)
    torch.cuda.synchronize()
    return cfg, ref, vis, truth, tab, src


def _check_table(cfg, ref, tab):
    for r in range(cfg.n_real):
        p, t = ref["params"][r], tab[r]
        assert math.isclose(t.a, p["a"], rel_tol=1e-14)
        assert np.allclose([t.u, t.v, t.w], p["uvw"], rtol=1e-12)
        assert t.n_comp == len(p["components"])
        for i, c in enumerate(p["components"]):
            g = t.comp[i]
            assert (g.kind, g.t0, g.t1, g.c0, g.c1, g.tries) == (c["kind"], c["t0"], c["t1"], c["c0"], c["c1"], c["tries"])
            assert math.isclose(g.period, c["period"], rel_tol=1e-14, abs_tol=0)
            J = np.array(list(g.J)).view(np.complex128)
            assert np.allclose(J, c["J"], rtol=0, atol=1e-12)
        if cfg.inr > 0:                                            # with inr = 0 the RFI kernels are not launched
            assert math.isclose(t.p_rfi, ref["p_rfi"][r], rel_tol=1e-9, abs_tol=1e-12)
        assert math.isclose(t.p_cel, ref["p_cel"][r], rel_tol=2e-6)          # fp32 samples, fp64 sum
        assert math.isclose(t.gain, ref["gain"][r], rel_tol=2e-6, abs_tol=0)


@pytest.mark.parametrize("kw", [
    dict(n_time=40, n_chan=16, n_real=3, n_sources=5, n_broadband=2, inr=10.0, seed=7),
    dict(n_time=64, n_chan=300, n_real=2, n_sources=200, inr=100.0, seed=2, window_T=16, window_F=4),      # ragged channel tile
    dict(n_time=50, n_chan=40, n_real=5, n_sources=3, n_broadband=5, inr=0.3, seed=11, window_T=5, window_F=4),
    dict(n_time=40, n_chan=64, n_real=2, n_sources=10, inr=0.0, seed=3),                                    # no RFI
    dict(n_time=40, n_chan=64, n_real=2, n_sources=10, inr=50.0, seed=3, polarized=False),                  # Fig. 3(b)
    dict(n_time=30, n_chan=32, n_real=2, n_sources=0, n_broadband=0, n_narrowband=3, n_narrowdur=2, inr=5.0, seed=4, window_T=10),
], ids=["small", "ragged_200src", "five_footprints", "inr0", "unpolarised", "narrow_only"])
def test_generator_matches_the_oracle(kw):
    cfg, ref, vis, truth, tab, src = _both(**kw)
    _check_table(cfg, ref, tab)
    # source coherence (fp64 both sides)
    for r in range(cfg.n_real):
        s_ref = so.source_signal(cfg, ref["params"][r])
        s_gpu = src[r].cpu().numpy().view(np.complex128).reshape(-1)
        assert np.allclose(s_gpu, s_ref, rtol=0, atol=1e-9 * max(1.0, np.abs(s_ref).max()))
    # the field
    got = vis.cpu().numpy().astype(np.float64).reshape(cfg.n_time, cfg.n_real, cfg.n_chan, 4, 2)
    want = ref["vis"].view(np.float64).reshape(cfg.n_time, cfg.n_real, cfg.n_chan, 4, 2)
    for r in range(cfg.n_real):
        rms = math.sqrt(float((want[:, r] ** 2).mean()))
        d = np.abs(got[:, r] - want[:, r])
        bound = 1e-5 * np.maximum(np.abs(want[:, r]), rms)
        assert (d <= bound).all(), f"realisation {r}: worst |d|/bound = {(d / bound).max():.3g}"
    # the window-level ground truth: bit-exact
    t_gpu = rfi.unpack_flags(truth, cfg.n_chan).cpu().numpy()
    assert (t_gpu == ref["truth"]).all()
    # measured INR = set INR on the generated data itself, from the device field
    if cfg.inr > 0:
        cel = so.generate(so.Sim42Config(**dict(kw, inr=0.0)))["vis"]
        for r in range(cfg.n_real):
            rf = got[:, r].reshape(cfg.n_time, cfg.n_chan, 4, 2) - cel[:, r].view(np.float64).reshape(cfg.n_time, cfg.n_chan, 4, 2)
            assert math.isclose((rf ** 2).sum() / (cel[:, r].real ** 2 + cel[:, r].imag ** 2).sum(), cfg.inr, rel_tol=2e-3)


def test_generator_is_deterministic_and_realisations_are_coordinates():
    a = rfi.sim42_generate(4, 10.0, seed=9, n_time=40, n_chan=64, n_sources=8)
    b = rfi.sim42_generate(4, 10.0, seed=9, n_time=40, n_chan=64, n_sources=8)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    c = rfi.sim42_generate(2, 10.0, seed=9, n_time=40, n_chan=64, n_sources=8)
    assert torch.equal(c[0], a[0][:, :2]) and torch.equal(c[1], a[1][:, :2])        # realisation r does not depend on the batch
    d = rfi.sim42_generate(4, 10.0, seed=10, n_time=40, n_chan=64, n_sources=8)
    assert not torch.equal(d[0], a[0])


def test_generator_rejects_bad_configurations():
    for kw in (dict(n_broadband=20), dict(inr=-1.0), dict(n_sources=5000), dict(window_T=7)):
        with pytest.raises(rfi.RfiError):
            rfi.sim42_generate(2, kw.pop("inr", 1.0), n_time=40, n_chan=16, **kw)


def _null_thresholds(tau, rmax, fa):
    """thresholds holding a per-detector false-alarm rate `fa` on RFI-free data ("providing a desired
    false alarm probability" -- here from the empirical null quantiles of the statistics planes)"""
    s_low = float(torch.quantile(tau, fa / 2)); s_high = float(torch.quantile(tau, 1 - fa / 2))
    gamma = float(torch.quantile(rmax, 1 - fa))
    return s_low, s_high, gamma


def _planes(plan, vis):
    avg, weight, stats = plan.alloc_outputs(stats=True)
    plan.process_chunk(vis, avg, weight, stats)
    torch.cuda.synchronize()
    s = stats.reshape(3, plan.n_win, plan.n_baselines, plan.n_chan)[:, :, :, ::plan.window_F]     # one value per footprint
    return s[0].flatten(), torch.maximum(s[1], s[2]).flatten()


def test_fig2_shaped_scenario_detector_ordering():
    """PAPER.md:233 (Fig. 2): 2000 x 512 block, 10 x 2 windows, INR 100, thresholds tuned to a false-alarm rate of about
    0.01: the paper reports SK 0.01/0.89, DS 0.01/0.06, BOTH 0.01/0.05.  Its fine-tuned thresholds are not printed, so
    the numbers are context; what must hold is the ordering MD(DS) << MD(SK) and MD(BOTH) <= MD(DS), with the false
    alarms of every detector near the design value."""
    INF = float("inf")
    R, T, C = 28, 2000, 512                                       # 28 = 8*7/2 realisations (one per "baseline")
    plan = rfi.RfiPlan(8, R, C, T, 10, n_int=T)
    plan.set_window_freq(2)
    clean, _ = rfi.sim42_generate(R, 0.0, seed=101, n_time=T, n_chan=C)
    plan.set_thresholds([[1.0, -INF, INF, INF]])
    tau, rmax = _planes(plan, clean)
    idx = torch.randperm(tau.numel(), device=tau.device)[:2_000_000]
    s_low, s_high, gamma = _null_thresholds(tau[idx], rmax[idx], 0.01)
    del clean
    vis, truth = rfi.sim42_generate(R, 100.0, seed=202, n_time=T, n_chan=C)
    plan.set_thresholds([[1.0, s_low, s_high, INF], [1.0, -INF, INF, gamma], [1.0, s_low, s_high, gamma]])   # SK, DS, BOTH
    avg, weight, _ = plan.alloc_outputs()
    plan.process_chunk(vis, avg, weight)
    counts = plan.confusion_counts(truth).cpu().double()
    fa = (counts[:, 0] / counts[:, 1]).tolist(); md = (counts[:, 2] / counts[:, 3]).tolist()
    print(f"sim42 INR=100, 10x2, FA target 0.01:  SK {fa[0]:.3f}/{md[0]:.3f}  DS {fa[1]:.3f}/{md[1]:.3f}  BOTH {fa[2]:.3f}/{md[2]:.3f}"
          f"   (paper Fig. 2: 0.01/0.89, 0.01/0.06, 0.01/0.05)")
    plan.destroy()
    assert all(f < 0.05 for f in fa)
    assert md[1] < 0.5 * md[0]                                    # polarisation beats energy on polarised RFI
    assert md[2] <= md[1] + 1e-12                                 # OR-combination can only remove missed detections
    assert md[2] < 0.5


def test_device_philox_known_answer_through_the_parameter_table():
    """The device generator's first draw of realisation 0 with seed 0 is Philox-4x32-10 of the all-zero counter and key:
    word 0 of the published vector (tests/golden/philox_kat.txt, 6627e8d5) fixes the receiver-noise scale
    a = 100 (x + 1/2) 2^-32 exactly (one rounding, IEEE on both sides).  With seed = key (ffffffff, ffffffff) and the
    pi vector no counter of the draw table matches, so those two stay CPU-side pins of the oracle, which the element by
    element parity above ties to the device."""
    _, _, tab, _ = rfi.sim42_generate(1, 1.0, seed=0, n_time=10, n_chan=8, n_sources=1, diagnostics=True)
    torch.cuda.synchronize()
    assert tab[0].a == 100.0 * ((0x6627E8D5 + 0.5) * 2.0 ** -32)
    # words 0..3 of that vector drive (u, v) through the next call's pair as well: against the oracle's own draw
    p = so.draw_params(so.Sim42Config(n_time=10, n_chan=8, n_real=1, n_sources=1, inr=1.0, seed=0), 0)
    assert p["a"] == tab[0].a
