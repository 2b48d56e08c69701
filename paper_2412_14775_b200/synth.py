"""Seeded synthetic correlator output for tests and bench.py.

This module serves BOTH the CUDA path and the CPU oracle with the same inputs and holds none of
the method's arithmetic (no Stokes parameters, no statistics, no thresholds applied): it only
draws noise and injects RFI.  The recipes stand in for the paper's LOFAR-LBA data and its
section-4.2 simulator, whose datasets are not available; they follow
BASELINE.json `configs` and SURVEY.md section 8(d) and are restated in DESIGN.md ("Input recipe").

Layout produced (include/rfi.h): vis[t][b][c][pol][re,im], time slowest, pol order XX,XY,YX,YY.
Everything is torch so the same code runs seeded on the CPU (small parity cases, shared with the
oracle) and on the GPU (full-size bench inputs).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace
from typing import Optional

import torch

RHO = 0.05          # XY/YX correlation of the 2x2 coherency with unit diagonal (BASELINE.json configs[0])
N_ACC_AUTO = 4      # spectra accumulated per auto-correlation dump (SURVEY.md 8(d) noise model)


@dataclass(frozen=True)
class Workload:
    name: str
    n_stations: int
    autos: bool                 # baselines = N(N+1)/2 if autos else N(N-1)/2
    n_chan: int
    n_time: int
    window_M: int
    n_int: int
    fp16: bool = False
    window_F: int = 1           # window extent in frequency (channels): footprint T x F, W = window_M * window_F
    channel_gain: bool = False  # per-channel gain U[0.8,1.2]
    # RFI recipe
    burst_cell_frac: float = 0.0    # fraction of cells carrying random low-duty-cycle polarised bursts
    burst_window_prob: float = 0.25
    tone_chan_frac: float = 0.0     # fraction of channels carrying a CW tone on all baselines
    mixed_cell_frac: float = 0.0    # config 4: each affected cell gets one of burst / tone / spikes
    fixed_burst: bool = False       # config 1: one 40-sample burst on 2 channels x 3 baselines

    @property
    def n_baselines(self) -> int:
        n = self.n_stations
        return n * (n + 1) // 2 if self.autos else n * (n - 1) // 2

    @property
    def n_cells(self) -> int:
        return self.n_baselines * self.n_chan

    @property
    def n_win(self) -> int:
        return self.n_time // self.window_M

    @property
    def n_out(self) -> int:
        return self.n_time // self.n_int

    @property
    def bytes_per_sample(self) -> int:
        return 16 if self.fp16 else 32

    @property
    def input_bytes(self) -> int:
        return self.n_time * self.n_cells * self.bytes_per_sample

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


# BASELINE.json configs[0..4].  "large" keeps B, C, M, n_int of configs[3] with chunk = one integration
# (73.6 GB): the stated 4 integrations per chunk (294.5 GB) exceed HBM.
WORKLOADS = {
    "tiny": Workload("tiny", 4, False, 16, 1024, 64, 64, fixed_burst=True),
    "lofar": Workload("lofar", 48, True, 64, 7680, 16, 768, channel_gain=True, burst_cell_frac=0.02),
    "lofar_fp16": Workload("lofar_fp16", 48, True, 64, 7680, 16, 768, fp16=True, channel_gain=True,
                           burst_cell_frac=0.02, tone_chan_frac=0.01),
    "large": Workload("large", 76, True, 256, 3072, 32, 3072, channel_gain=True, mixed_cell_frac=0.03),
    "sweep": Workload("sweep", 48, True, 64, 7680, 16, 768, channel_gain=True, burst_cell_frac=0.02),
    # the paper's own footprints, W = 20 as 10 x 2 and 5 x 4, on the LOFAR-subband shape;
    # 760 samples per integration so that T = 10 and T = 5 divide it (not BASELINE.json configs: SURVEY 8(f) NEXT-1)
    "lofar_tf10x2": Workload("lofar_tf10x2", 48, True, 64, 7600, 10, 760, window_F=2, channel_gain=True, burst_cell_frac=0.02),
    "lofar_tf5x4": Workload("lofar_tf5x4", 48, True, 64, 7600, 5, 760, window_F=4, channel_gain=True, burst_cell_frac=0.02),
}
BASELINE_CONFIG_INDEX = {"tiny": 0, "lofar": 1, "lofar_fp16": 2, "large": 3, "sweep": 4}


def auto_baseline_mask(w: Workload, device="cpu") -> torch.Tensor:
    """bool[n_baselines]: True where the baseline is an auto-correlation.  Baseline order is
    (p,q), p<=q, p-major (opaque to the kernel, which treats every stream alike)."""
    m = []
    for p in range(w.n_stations):
        for q in range(p if w.autos else p + 1, w.n_stations):
            m.append(p == q)
    return torch.tensor(m, dtype=torch.bool, device=device)


def _mix_matrix(device) -> torch.Tensor:
    """Real Cholesky factor L of Sigma (x) Sigma, Sigma = [[1,rho],[rho,1]]: vec(V) = L z has the
    covariance of vec(e_p e_q^H) for station voltages e ~ CN(0, Sigma)."""
    s = torch.tensor([[1.0, RHO], [RHO, 1.0]], dtype=torch.float64)
    return torch.linalg.cholesky(torch.kron(s, s)).to(torch.float32).to(device)


def _unit_jones(gen, shape, device):
    """Random unit Jones vectors g in C^2 -> rank-1 coherency g g^H as [..., 4] complex (xx,xy,yx,yy)."""
    g = torch.randn(*shape, 2, 2, generator=gen, device=device)
    g = torch.view_as_complex(g.contiguous())
    g = g / g.abs().pow(2).sum(-1, keepdim=True).sqrt()
    gx, gy = g[..., 0], g[..., 1]
    return torch.stack([gx * gx.conj(), gx * gy.conj(), gy * gx.conj(), gy * gy.conj()], -1)


def _loguniform(gen, shape, lo, hi, device):
    u = torch.rand(*shape, generator=gen, device=device)
    return torch.exp(math.log(lo) + u * (math.log(hi) - math.log(lo)))


def make_chunk(w: Workload, seed: int = 1234, device="cpu", slab_rows: int = 256,
               out: Optional[torch.Tensor] = None):
    """Draw one chunk.

    Returns (vis, truth):
      vis   real tensor [n_time, n_baselines, n_chan, 4, 2], float32 (or float16 if w.fp16)
      truth bool [n_win, n_cells]: windows that contain injected RFI samples (ground truth for the
            false-alarm / missed-detection rates of PAPER.md:235).
    """
    device = torch.device(device)
    # independent streams: the noise realisation does not depend on which RFI recipe is switched on
    gen = torch.Generator(device=device)          # RFI plan
    gen.manual_seed(seed * 3 + 1)
    gen_noise = torch.Generator(device=device)
    gen_noise.manual_seed(seed * 3)
    gen_gain = torch.Generator(device=device)
    gen_gain.manual_seed(seed * 3 + 2)
    T, B, C, M = w.n_time, w.n_baselines, w.n_chan, w.window_M
    ncell = B * C
    L = _mix_matrix(device)
    autos = auto_baseline_mask(w, device)
    dtype = torch.float16 if w.fp16 else torch.float32
    vis = out if out is not None else torch.empty(T, B, C, 4, 2, dtype=dtype, device=device)
    assert vis.shape == (T, B, C, 4, 2) and vis.dtype == dtype
    gain = (0.8 + 0.4 * torch.rand(C, generator=gen_gain, device=device)) if w.channel_gain else None
    sig = torch.tensor([1.0, RHO, RHO, 1.0], device=device)

    # ---- RFI plan (additive, complex, per affected cell) ----
    truth = torch.zeros(w.n_win, ncell, dtype=torch.bool, device=device)
    adds = []   # list of (cell_index[n], add[T, n, 4] complex64)

    def burst_add(cells, amp_lo=0.3, amp_hi=30.0):
        n = cells.numel()
        has = torch.rand(w.n_win, n, generator=gen, device=device) < w.burst_window_prob
        u = 0.01 + 0.19 * torch.rand(w.n_win, n, generator=gen, device=device)
        length = torch.clamp(torch.round(u * M), min=1)
        off = torch.floor(torch.rand(w.n_win, n, generator=gen, device=device) * (M - length + 1))
        amp = _loguniform(gen, (w.n_win, n), amp_lo, amp_hi, device)
        phase = 2 * math.pi * torch.rand(w.n_win, n, generator=gen, device=device)
        coh = _unit_jones(gen, (w.n_win, n), device) * torch.polar(amp, phase)[..., None]
        tin = torch.arange(M, device=device).view(1, M, 1)
        active = has[:, None, :] & (tin >= off[:, None, :]) & (tin < (off + length)[:, None, :])   # [W,M,n]
        add = (active[..., None] * coh[:, None, :, :]).reshape(T, n, 4)
        truth[:, cells] |= has
        return add

    def tone_add(cells):
        n = cells.numel()
        amp = _loguniform(gen, (n,), 0.3, 30.0, device)
        phi0 = 2 * math.pi * torch.rand(n, generator=gen, device=device)
        omega = -0.3 + 0.6 * torch.rand(n, generator=gen, device=device)
        t = torch.arange(T, device=device, dtype=torch.float32)[:, None]
        ph = phi0[None, :] + omega[None, :] * t
        coh = _unit_jones(gen, (n,), device)
        truth[:, cells] = True
        return torch.polar(amp[None, :].expand(T, n).contiguous(), ph)[..., None] * coh[None]

    def spike_add(cells):
        n = cells.numel()
        has = torch.rand(w.n_win, n, generator=gen, device=device) < w.burst_window_prob
        off = torch.floor(torch.rand(w.n_win, n, generator=gen, device=device) * M)
        tin = torch.arange(M, device=device).view(1, M, 1)
        active = has[:, None, :] & (tin == off[:, None, :])
        ph = 2 * math.pi * torch.rand(w.n_win, n, 4, generator=gen, device=device)   # unpolarised: independent phases
        val = torch.polar(torch.full_like(ph, 100.0), ph)
        truth[:, cells] |= has
        return (active[..., None] * val[:, None]).reshape(T, n, 4)

    if w.fixed_burst:
        # one fully polarised rectangular burst of 40 samples at 10x noise power on 2 channels x 3 baselines;
        # start differs per baseline: inside one window / straddling a boundary / ending at a boundary
        coh = _unit_jones(gen, (1,), device)[0] * torch.polar(torch.tensor(math.sqrt(10.0)), torch.tensor(0.7)).to(device)
        starts = [M * 5 + 10, M * 8 + 40, M * 12 + (M - 40 if M >= 40 else 0)]
        chans = [3 % C, 7 % C]
        cells, cols = [], []
        for bi, st in enumerate(starts[:min(3, B)]):
            for c in chans:
                col = torch.zeros(T, 4, dtype=torch.complex64, device=device)
                st_ = min(st, max(T - 40, 0))
                col[st_:st_ + 40] = coh
                cells.append(bi * C + c)
                cols.append(col)
                truth[st_ // M:(min(st_ + 40, T) - 1) // M + 1, bi * C + c] = True
        adds.append((torch.tensor(cells, device=device), torch.stack(cols, 1)))
    if w.burst_cell_frac > 0:
        n_aff = max(1, int(round(w.burst_cell_frac * ncell)))
        cells = torch.randperm(ncell, generator=gen, device=device)[:n_aff].sort().values
        adds.append((cells, burst_add(cells)))
    if w.tone_chan_frac > 0:
        n_ch = max(1, math.ceil(w.tone_chan_frac * C))
        ch = torch.randperm(C, generator=gen, device=device)[:n_ch]
        cells = (torch.arange(B, device=device)[:, None] * C + ch[None, :]).reshape(-1).sort().values
        adds.append((cells, tone_add(cells)))
    if w.mixed_cell_frac > 0:
        n_aff = max(3, int(round(w.mixed_cell_frac * ncell)))
        cells = torch.randperm(ncell, generator=gen, device=device)[:n_aff]
        third = n_aff // 3
        for part, fn in ((cells[:third], burst_add), (cells[third:2 * third], tone_add), (cells[2 * third:], spike_add)):
            part = part.sort().values
            adds.append((part, fn(part)))

    # ---- noise, slab by slab over time (bounds temporaries at full size) ----
    vflat = vis.view(T, ncell, 4, 2)
    for t0 in range(0, T, slab_rows):
        t1 = min(T, t0 + slab_rows)
        z = torch.randn(t1 - t0, B, C, 4, 2, generator=gen_noise, device=device) * math.sqrt(0.5)
        x = torch.einsum("qp,tbcpr->tbcqr", L, z).contiguous()                       # cross-baseline noise, unit variance per pol
        if autos.any():
            xa = torch.view_as_complex(x[:, autos].contiguous())        # [t, n_auto, C, 4]
            h = torch.stack([xa[..., 0].real * math.sqrt(2.0) + 0j,
                             (xa[..., 1] + xa[..., 2].conj()) / math.sqrt(2.0),
                             (xa[..., 2] + xa[..., 1].conj()) / math.sqrt(2.0),
                             xa[..., 3].real * math.sqrt(2.0) + 0j], -1)
            h[..., 2] = h[..., 1].conj()
            va = sig + h / math.sqrt(N_ACC_AUTO)                        # Hermitian: Sigma + n_acc^-1/2 H
            x[:, autos] = torch.view_as_real(va)
        x = x.view(t1 - t0, ncell, 4, 2)
        for cells, add in adds:
            x[:, cells] += torch.view_as_real(add[t0:t1].to(torch.complex64))
        if gain is not None:
            x = (x.view(t1 - t0, B, C, 8) * gain[None, None, :, None]).view(t1 - t0, ncell, 4, 2)
        vflat[t0:t1] = x.to(dtype)
    return vis, truth


# Null quantiles of the two statistics under this noise model, used only to place thresholds
# (survey-derived Monte Carlo; the paper prints no threshold values).
# x = W*S2/S1^2 - 1;  rows: W -> (x 0.1%, 1%, 5%, 95%, 99%, 99.9%), (max(r_re,r_im) 95%, 99%, 99.9%)
_NULL_Q = {
    16: ((0.063, 0.094, 0.128, 0.431, 0.538, 0.684), (0.435, 0.504, 0.584)),
    32: ((0.100, 0.137, 0.165, 0.385, 0.454, 0.545), (0.310, 0.362, 0.422)),
    64: ((0.140, 0.172, 0.195, 0.350, 0.398, 0.455), (0.219, 0.258, 0.302)),
}


# The same for the auto-correlations of this noise model (Hermitian, Sigma + H/sqrt(n_acc)): |I| is nearly constant,
# so x sits far below the cross-correlation values; r_im = 0 exactly.  Written by tests/golden/make_null_quantiles.py
# (a committed script that calls only oracle/ and this module; tests/test_synth.py re-derives an entry); only used to
# place the class-1 thresholds -- parity never depends on them.
_NULL_Q_AUTO = {
    16: ((0.024, 0.0386, 0.0546, 0.207, 0.2571, 0.3342), (0.418, 0.496, 0.575)),
    20: ((0.031, 0.0447, 0.0602, 0.198, 0.2430, 0.3030), (0.377, 0.449, 0.522)),
    32: ((0.046, 0.0578, 0.0724, 0.183, 0.2158, 0.2601), (0.307, 0.365, 0.432)),
    64: ((0.064, 0.0750, 0.0867, 0.165, 0.1870, 0.2147), (0.230, 0.273, 0.323)),
}


def auto_thresholds(M: int, d: float = 1.0):
    """One (d, s_low, s_high, gamma) set near the 1 % / 99 % null quantiles of the auto-correlations (class 1)."""
    xq, rq = _NULL_Q_AUTO[M] if M in _NULL_Q_AUTO else _NULL_Q_AUTO[min(_NULL_Q_AUTO, key=lambda k: abs(k - M))]
    c = (M * d + 1) / (M - 1)
    return [d, c * xq[1], c * xq[4], rq[1]]


def _quantiles(M: int):
    if M in _NULL_Q:
        return _NULL_Q[M]
    # large-W normal approximation around the Rayleigh limit 4/pi - 1, and the chi^2_3 Rayleigh-test
    # approximation P(r > g) ~ P(chi2_3 > 3 W g^2) for the directional statistic
    mu, sd = 4 / math.pi - 1 - 0.23 / M, 0.40 / math.sqrt(M)
    xq = tuple(max(mu + z * sd, 0.01) for z in (-3.1, -2.33, -1.64, 1.64, 2.33, 3.1))
    rq = tuple(min(math.sqrt(c / (3 * M)), 0.999) for c in (9.35, 12.84, 17.73))
    return xq, rq


def default_thresholds(M: int, d: float = 1.0):  # M = window size W (T*F for footprints)
    """One (d, s_low, s_high, gamma) set near the 1 % / 99 % null quantiles."""
    xq, rq = _quantiles(M)
    c = (M * d + 1) / (M - 1)
    return [[d, c * xq[1], c * xq[4], rq[1]]]


def sweep_thresholds(M: int, K: int = 64, seed: int = 99):
    """K threshold sets for the batched sweep: d ~ U[0.5,1]; s_low, s_high, gamma uniform
    between the 0.1 %..5 % / 95 %..99.9 % null quantiles (the paper states no ranges, reading G11)."""
    g = torch.Generator().manual_seed(seed)
    xq, rq = _quantiles(M)
    u = torch.rand(K, 4, generator=g, dtype=torch.float64)
    d = 0.5 + 0.5 * u[:, 0]
    c = (M * d + 1) / (M - 1)
    s_low = c * (xq[0] + (xq[2] - xq[0]) * u[:, 1])
    s_high = c * (xq[3] + (xq[5] - xq[3]) * u[:, 2])
    gamma = rq[0] + (rq[2] - rq[0]) * u[:, 3]
    return torch.stack([d, s_low, s_high, gamma], 1).tolist()


def rl_windows(n: int, T: int = 10, F: int = 2, seed: int = 0, rfi_prob: float = 0.4, device="cpu") -> torch.Tensor:
    """Windows as the paper's RL training simulator draws them: float32 [n, W = T*F, 4, 2].
    Complex circular Gaussian noise (standard normal real and imaginary parts) times a scale factor U[0.01, 1000]; with
    probability 0.4 an RFI signal: a uniformly drawn rectangular footprint inside the T x F window filled with ones
    times a complex scale factor of modulus U[0.01, 1000], multiplied by a 2 x 2 complex circular Gaussian matrix whose
    four entries scale the four correlations (reading: the matrix entries are the per-correlation gains that "create
    correlation between the polarizations of the RFI signal").  Sample order inside a window: time-major (t, f)."""
    g = torch.Generator(device=device).manual_seed(seed)
    W = T * F
    x = torch.randn(n, W, 4, 2, generator=g, device=device)
    scale = 0.01 + (1000.0 - 0.01) * torch.rand(n, 1, 1, 1, generator=g, device=device)
    x = x * scale
    has = torch.rand(n, generator=g, device=device) < rfi_prob
    t0 = torch.floor(torch.rand(n, generator=g, device=device) * T); t1 = torch.floor(torch.rand(n, generator=g, device=device) * T)
    f0 = torch.floor(torch.rand(n, generator=g, device=device) * F); f1 = torch.floor(torch.rand(n, generator=g, device=device) * F)
    tt = torch.arange(T, device=device).view(1, T, 1); ff = torch.arange(F, device=device).view(1, 1, F)
    foot = ((tt >= torch.minimum(t0, t1).view(n, 1, 1)) & (tt <= torch.maximum(t0, t1).view(n, 1, 1))
            & (ff >= torch.minimum(f0, f1).view(n, 1, 1)) & (ff <= torch.maximum(f0, f1).view(n, 1, 1)) & has.view(n, 1, 1))
    amp = torch.polar(0.01 + (1000.0 - 0.01) * torch.rand(n, generator=g, device=device),
                      2 * math.pi * torch.rand(n, generator=g, device=device))
    mix = torch.view_as_complex((torch.randn(n, 4, 2, generator=g, device=device) * math.sqrt(0.5)).contiguous())   # 2 x 2, unit variance
    rfi = foot.reshape(n, W, 1).to(torch.complex64) * (amp.view(n, 1, 1) * mix.view(n, 1, 4))
    return (x + torch.view_as_real(rfi)).to(torch.float32).contiguous()
