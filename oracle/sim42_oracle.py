"""Oracle of the section-4.2 simulator: TEST INFRASTRUCTURE, not the product.

Plain numpy, fp64, one statement per sentence of the recipe, no blocking or fusion.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / verification legs may import this module; nothing under paper_2412_14775_b200/ does, and
this module imports nothing from it.  The CUDA generator (csrc/rfi_sim42.cu) shares no code with it: both restate the
same published counter-based generator (Philox-4x32, 10 rounds; Salmon et al., SC'11) and the same draw table below,
so that the random numbers the recipe draws are identical integers on both sides and the generated fields can be
compared element by element (floating point: the CUDA side evaluates the Gaussian transform in fp32, this side in
fp64; tolerance in tests/).

What the paper fixes and the readings taken where it is silent or garbled (DESIGN.md section 2,
S1-S9) -- per realisation (one simulated baseline, a block of n_time x n_chan time-frequency samples, 4 correlations):

  noise      e_p, e_q ~ CN(0, I_2) per sample (station voltages);  receiver noise = e_p e_q^H (conjugate product);
             sky noise ~ CN(0,1) per correlation;  total = a * receiver + sky,  a = 100 U(0,1), one per realisation
             (PAPER.md:223).
  sources    n_src = 200; (u,v,w) = 300 N(0,1) each, one baseline per realisation; (l,m) ~ U(-0.5,0.5),
             n = sqrt(1-l^2-m^2); flux S ~ U(1,10); coherence S exp(j 2 pi f (ul + vm + w(n-1))/c),
             f_k = 120 MHz + k * 200 kHz / n_chan.  Reading S3: sources are unpolarised, xx = yy = S/2 * phase
             (Eq.(2) has I = xx + yy without a half), xy = yx = 0; constant in time.
  RFI        n_bb broadband footprints [t0,t1) x [c0,c1) (two sorted uniform edges per axis), filled with ones;
             n_nb narrowband: one channel, all times, exp(j 2 pi t / P), P = max(120 U(0,1), 2) samples;
             n_nd narrow-duration: one time sample, all channels, exp(j 2 pi c / P), P = max(1024 U(0,1), 2) samples
             (the units of the two periods are garbled: read as samples along the axis the signal
             extends over).  Each component is scaled by J/||J||, J = 4 draws from CN(0,1) read both as the four
             correlations (xx,xy,yx,yy) and as the 2x2 matrix whose coherency J J^H defines the polarised fraction
             p = sqrt(Q^2+U^2+V^2)/I; draws with p > 0.9 are eliminated (redrawn, at most 16 times).
             polarized = False (Fig. 3(b)): J = (1,0,0,1)/sqrt(2), Q = U = V = 0.
  mixing     celestial = noise + sources;  data = celestial + g * rfi,  g^2 = INR * P_cel / P_rfi with P = total power
             (sum of |.|^2 over the block and the 4 correlations).
  truth      a time-frequency point carries RFI where any component is non-zero; a T x F window (footprint) carries
             RFI if any of its points does (PAPER.md:235 definitions of false alarm / missed detection).

Draw table (stream 0 of realisation r; call j = Philox(counter = (j, 0, 0, r), key = seed) -> 4 words x0..x3):
  U(x) = (x + 0.5) 2^-32;  normal pair from (xa, xb): R = sqrt(-2 ln ua), ua = (2 (xa >> 9) + 1) 2^-24,
  phi = 2 pi (xb >> 8) 2^-24, (R cos phi, R sin phi).
  call 0: a = 100 U(x0)          call 1: (u, v) = 300 * pair(x0,x1), w = 300 * first of pair(x2,x3)
  call 2+s: l = U(x0)-0.5, m = U(x1)-0.5, S = 1 + 9 U(x2)                                   (s < n_src)
  component i (broadband first, then narrowband, then narrow-duration), base = 2 + n_src + i * 33:
    call base: broadband  e = floor(U(x0..x3) * (n+1)) on the time (x0,x1) and channel (x2,x3) axes, sorted, widened to
               one sample if equal;  narrowband  channel = floor(U(x0) n_chan), P = max(120 U(x1), 2);
               narrow-duration  time = floor(U(x0) n_time), P = max(1024 U(x1), 2)
    calls base+1+2k, base+2+2k (k = 0..15): try k of J: (J0, J1) and (J2, J3) = pairs / sqrt(2)
Noise (stream 1): sample (t, c) call q = 0..3, counter = ((t n_chan + c) 4 + q, 0, 1, r):
  q = 0: e_p = (pair(x0,x1), pair(x2,x3)) / sqrt(2) as (x-pol, y-pol);  q = 1: e_q likewise;
  q = 2: sky xx, xy;  q = 3: sky yx, yy   (each pair / sqrt(2): unit variance per complex value)
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

C_LIGHT = 299792458.0
MAX_TRIES = 16
CALLS_PER_COMPONENT = 1 + 2 * MAX_TRIES


@dataclass
class Sim42Config:
    n_time: int = 2000
    n_chan: int = 512
    n_real: int = 1
    n_sources: int = 200
    n_broadband: int = 5
    n_narrowband: int = 1
    n_narrowdur: int = 1
    polarized: bool = True
    inr: float = 100.0
    seed: int = 1
    window_T: int = 10
    window_F: int = 2


# ---------------------------------------------------------------------------------------------------------
# Philox-4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3", SC'11), restated.
# ---------------------------------------------------------------------------------------------------------
_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32(c0, c1, c2, c3, seed: int):
    """10 rounds on arrays of 32-bit counter words (any broadcastable shapes); returns 4 uint32 arrays."""
    c0, c1, c2, c3 = (np.asarray(x, np.uint64) & _MASK for x in np.broadcast_arrays(c0, c1, c2, c3))
    k0, k1 = seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0                                   # 32 x 32 -> 64 bit products
        p1 = _M1 * c2
        n0 = (p1 >> np.uint64(32)) ^ c1 ^ np.uint64(k0)
        n1 = p1 & _MASK
        n2 = (p0 >> np.uint64(32)) ^ c3 ^ np.uint64(k1)
        n3 = p0 & _MASK
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0, k1 = (k0 + _W0) & 0xFFFFFFFF, (k1 + _W1) & 0xFFFFFFFF
    return tuple(x.astype(np.uint32) for x in (c0, c1, c2, c3))


def uniform01(x):
    return (np.asarray(x, np.float64) + 0.5) * 2.0 ** -32


def normal_pair(xa, xb):
    ua = (2.0 * (np.asarray(xa, np.uint32) >> np.uint32(9)).astype(np.float64) + 1.0) * 2.0 ** -24
    phi = 2.0 * np.pi * (np.asarray(xb, np.uint32) >> np.uint32(8)).astype(np.float64) * 2.0 ** -24
    r = np.sqrt(-2.0 * np.log(ua))
    return r * np.cos(phi), r * np.sin(phi)


def _call(j, stream, r, seed):
    return philox4x32(np.uint64(j), np.uint64(0), np.uint64(stream), np.uint64(r), seed)


def polarised_fraction(J):
    """p of the coherency C = J J^H of the 2x2 matrix J = [[J0,J1],[J2,J3]]: I = C00 + C11, Q = C00 - C11,
    U = 2 Re C01, V = -2 Im C01 (real Stokes of a Hermitian coherency); p = sqrt(Q^2+U^2+V^2)/I in [0,1]."""
    Jm = np.asarray(J, np.complex128).reshape(2, 2)
    C = Jm @ Jm.conj().T
    I = (C[0, 0] + C[1, 1]).real
    Q = (C[0, 0] - C[1, 1]).real
    U, V = 2.0 * C[0, 1].real, -2.0 * C[0, 1].imag
    return float(np.sqrt(Q * Q + U * U + V * V) / I)


def draw_params(cfg: Sim42Config, r: int) -> dict:
    """The per-realisation parameter table (module docstring, stream 0)."""
    x = _call(0, 0, r, cfg.seed)
    a = 100.0 * uniform01(x[0])
    x = _call(1, 0, r, cfg.seed)
    z0, z1 = normal_pair(x[0], x[1])
    z2, _ = normal_pair(x[2], x[3])
    u, v, w = 300.0 * z0, 300.0 * z1, 300.0 * z2
    js = np.arange(cfg.n_sources)
    xs = philox4x32(2 + js, 0, 0, r, cfg.seed)
    l, m = uniform01(xs[0]) - 0.5, uniform01(xs[1]) - 0.5
    S = 1.0 + 9.0 * uniform01(xs[2])
    n = np.sqrt(1.0 - l * l - m * m)
    kappa = (u * l + v * m + w * (n - 1.0)) / C_LIGHT            # seconds: phase = 2 pi f kappa
    comps = []
    n_comp = cfg.n_broadband + cfg.n_narrowband + cfg.n_narrowdur
    for i in range(n_comp):
        base = 2 + cfg.n_sources + i * CALLS_PER_COMPONENT
        x = _call(base, 0, r, cfg.seed)
        uu = [float(uniform01(x[q])) for q in range(4)]
        if i < cfg.n_broadband:
            e = sorted((int(np.floor(uu[0] * (cfg.n_time + 1))), int(np.floor(uu[1] * (cfg.n_time + 1)))))
            f = sorted((int(np.floor(uu[2] * (cfg.n_chan + 1))), int(np.floor(uu[3] * (cfg.n_chan + 1)))))
            if e[0] == e[1]:
                e = [e[0] - 1, e[0]] if e[0] == cfg.n_time else [e[0], e[0] + 1]
            if f[0] == f[1]:
                f = [f[0] - 1, f[0]] if f[0] == cfg.n_chan else [f[0], f[0] + 1]
            comp = {"kind": 0, "t0": e[0], "t1": e[1], "c0": f[0], "c1": f[1], "period": 0.0}
        elif i < cfg.n_broadband + cfg.n_narrowband:
            ch = min(int(np.floor(uu[0] * cfg.n_chan)), cfg.n_chan - 1)
            comp = {"kind": 1, "t0": 0, "t1": cfg.n_time, "c0": ch, "c1": ch + 1, "period": max(120.0 * uu[1], 2.0)}
        else:
            tt = min(int(np.floor(uu[0] * cfg.n_time)), cfg.n_time - 1)
            comp = {"kind": 2, "t0": tt, "t1": tt + 1, "c0": 0, "c1": cfg.n_chan, "period": max(1024.0 * uu[1], 2.0)}
        if cfg.polarized:
            J = None
            for k in range(MAX_TRIES):
                xa = _call(base + 1 + 2 * k, 0, r, cfg.seed)
                xb = _call(base + 2 + 2 * k, 0, r, cfg.seed)
                g = [normal_pair(xa[0], xa[1]), normal_pair(xa[2], xa[3]), normal_pair(xb[0], xb[1]), normal_pair(xb[2], xb[3])]
                J = np.array([complex(float(re), float(im)) for re, im in g]) / np.sqrt(2.0)
                if polarised_fraction(J) <= 0.9:             # eliminate draws that are more than 90 % polarised
                    break
            comp["tries"] = k + 1
        else:
            J = np.array([1.0, 0.0, 0.0, 1.0], np.complex128)
            comp["tries"] = 0
        comp["J"] = J / np.sqrt((np.abs(J) ** 2).sum())          # J / ||J||
        comps.append(comp)
    return {"a": float(a), "uvw": (float(u), float(v), float(w)), "l": l, "m": m, "S": S, "kappa": kappa, "components": comps}


def frequencies(cfg: Sim42Config):
    return 120.0e6 + np.arange(cfg.n_chan) * (200.0e3 / cfg.n_chan)


def source_signal(cfg: Sim42Config, p: dict):
    """[n_chan] complex: sum_s S_s exp(j 2 pi f kappa_s); enters xx and yy with weight 1/2."""
    f = frequencies(cfg)
    return (p["S"][None, :] * np.exp(2j * np.pi * f[:, None] * p["kappa"][None, :])).sum(1)


def noise(cfg: Sim42Config, p: dict, r: int):
    """[n_time, n_chan, 4] complex: a * e_p e_q^H + sky."""
    T, C = cfg.n_time, cfg.n_chan
    idx = (np.arange(T, dtype=np.uint64)[:, None] * np.uint64(C) + np.arange(C, dtype=np.uint64)[None, :]) * np.uint64(4)
    out = []
    for q in range(4):
        j = idx + np.uint64(q)
        x = philox4x32(j & _MASK, j >> np.uint64(32), 1, r, cfg.seed)
        a_re, a_im = normal_pair(x[0], x[1])
        b_re, b_im = normal_pair(x[2], x[3])
        out.append(((a_re + 1j * a_im) / np.sqrt(2.0), (b_re + 1j * b_im) / np.sqrt(2.0)))
    (epx, epy), (eqx, eqy), (sxx, sxy), (syx, syy) = out
    rx = np.stack([epx * eqx.conj(), epx * eqy.conj(), epy * eqx.conj(), epy * eqy.conj()], -1)   # e_p e_q^H
    sky = np.stack([sxx, sxy, syx, syy], -1)
    return p["a"] * rx + sky


def rfi_signal(cfg: Sim42Config, p: dict):
    """([n_time, n_chan, 4] complex unscaled RFI field, [n_time, n_chan] bool support)."""
    T, C = cfg.n_time, cfg.n_chan
    field = np.zeros((T, C, 4), np.complex128)
    support = np.zeros((T, C), bool)
    t = np.arange(T, dtype=np.float64)[:, None]
    c = np.arange(C, dtype=np.float64)[None, :]
    for comp in p["components"]:
        sl = (slice(comp["t0"], comp["t1"]), slice(comp["c0"], comp["c1"]))
        if comp["kind"] == 0:
            amp = np.ones((T, C), np.complex128)
        elif comp["kind"] == 1:
            amp = np.exp(2j * np.pi * t / comp["period"]) * np.ones((1, C))
        else:
            amp = np.exp(2j * np.pi * c / comp["period"]) * np.ones((T, 1))
        field[sl] += amp[sl][..., None] * comp["J"][None, None, :]
        support[sl] = True
    return field, support


def window_truth(cfg: Sim42Config, support):
    """[n_win, n_chan] bool: every channel of a T x F footprint that holds an RFI point."""
    T, C, wt, wf = cfg.n_time, cfg.n_chan, cfg.window_T, cfg.window_F
    s = support.reshape(T // wt, wt, C // wf, wf).any(axis=(1, 3))
    return np.repeat(s, wf, axis=1)


def generate(cfg: Sim42Config):
    """Returns dict: vis [n_time, n_real, n_chan, 4] complex128 (layout of include/rfi.h with b = realisation),
    truth [n_win, n_real, n_chan] bool, inr_measured [n_real], params (list of tables), p_cel, p_rfi, gain."""
    T, C, R = cfg.n_time, cfg.n_chan, cfg.n_real
    vis = np.zeros((T, R, C, 4), np.complex128)
    truth = np.zeros((T // cfg.window_T, R, C), bool)
    inr_m, params, pc, pr, gains = np.zeros(R), [], np.zeros(R), np.zeros(R), np.zeros(R)
    for r in range(R):
        p = draw_params(cfg, r)
        cel = noise(cfg, p, r)
        src = source_signal(cfg, p)
        cel[:, :, 0] += 0.5 * src[None, :]
        cel[:, :, 3] += 0.5 * src[None, :]
        field, support = rfi_signal(cfg, p)
        p_cel = float((np.abs(cel) ** 2).sum())
        p_rfi = float((np.abs(field) ** 2).sum())
        g = np.sqrt(cfg.inr * p_cel / p_rfi) if (cfg.inr > 0 and p_rfi > 0) else 0.0
        data = cel + g * field
        vis[:, r] = data
        truth[:, r] = window_truth(cfg, support) if g > 0 else False
        inr_m[r] = float((np.abs(g * field) ** 2).sum()) / p_cel
        params.append(p); pc[r], pr[r], gains[r] = p_cel, p_rfi, g
    return {"vis": vis, "truth": truth, "inr_measured": inr_m, "params": params, "p_cel": pc, "p_rfi": pr, "gain": gains}
