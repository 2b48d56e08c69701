"""rfi_sim42_generate_static: the section-4.2 generator with its work arrays in a fixed array inside
librfi.so, for callers that cannot allocate device memory -- a plug-in inside a correlator process that gave the whole
GPU to its own pool at start-up and passes only input and output buffers, or a tuning loop that generates blocks next
to live flagging streams, which a cudaMalloc / cudaFree (both serialise with every stream of the device) would stall.

What is checked: its output against the existing entry point (rfi_sim42_generate with internally allocated work
buffers) on the same configuration and seed, for several calls in a row of different shapes -- the array is shared by
all calls and still holds the previous call's table and source rows, so a later, smaller call would show any state
that leaks from one call into the next.  Tolerances are those of tests/test_gpu_sim42.py: the truth mask bit for bit;
the field within 1e-5 * max(|x|, rms) per real component (both entry points accumulate the two power totals of the
mixing gain with floating-point atomics, so the gain may differ in its last bits from run to run); bit for bit where
inr = 0, where no total enters the field.  The size cap is checked without a GPU.

This file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here hides nothing after it.
It passes alone in a fresh process and after the rest of the suite."""
import ctypes
import math

import numpy as np
import pytest
import torch

import paper_2412_14775_b200 as rfi
from paper_2412_14775_b200 import binding


def _existing(kw):
    vis, truth = rfi.sim42_generate(kw["n_real"], kw["inr"], seed=kw["seed"], n_time=kw["n_time"], n_chan=kw["n_chan"],
                                    n_sources=kw["n_sources"], n_broadband=kw.get("n_broadband", 5),
                                    polarized=kw.get("polarized", True), window_T=kw["window_T"], window_F=kw["window_F"])
    torch.cuda.synchronize()
    return vis, truth


def _static(kw, fill):
    """Caller-owned outputs, pre-filled with a pattern so that anything the call leaves unwritten shows."""
    vis = torch.full((kw["n_time"], kw["n_real"], kw["n_chan"], 4, 2), float(fill), dtype=torch.float32, device="cuda")
    truth = torch.full((kw["n_time"] // kw["window_T"], kw["n_real"], (kw["n_chan"] + 31) // 32), -1, dtype=torch.int32,
                       device="cuda")
    rfi.sim42_generate_static(vis, truth, kw["inr"], seed=kw["seed"], n_sources=kw["n_sources"],
                              n_broadband=kw.get("n_broadband", 5), polarized=kw.get("polarized", True),
                              window_T=kw["window_T"], window_F=kw["window_F"])
    torch.cuda.synchronize()
    return vis, truth


def _assert_same(kw, got, want):
    (g_vis, g_truth), (w_vis, w_truth) = got, want
    assert torch.equal(g_truth, w_truth), "truth mask differs"
    if kw["inr"] == 0.0:
        assert torch.equal(g_vis, w_vis), "inr = 0: the field must be identical bit for bit"
        return
    g = g_vis.cpu().numpy().astype(np.float64)
    w = w_vis.cpu().numpy().astype(np.float64)
    for r in range(kw["n_real"]):
        rms = math.sqrt(float((w[:, r] ** 2).mean()))
        d = np.abs(g[:, r] - w[:, r])
        bound = 1e-5 * np.maximum(np.abs(w[:, r]), rms)
        assert (d <= bound).all(), f"realisation {r}: worst |d| / bound = {(d / bound).max():.3g}"


CALLS = [
    dict(n_time=60, n_chan=96, n_real=6, n_sources=40, inr=10.0, seed=21, window_T=10, window_F=2),
    dict(n_time=40, n_chan=40, n_real=3, n_sources=7, inr=0.5, seed=22, window_T=5, window_F=4, n_broadband=2),   # smaller: stale rows stay behind it
    dict(n_time=30, n_chan=64, n_real=2, n_sources=10, inr=0.0, seed=23, window_T=10, window_F=2),               # bit for bit
    dict(n_time=64, n_chan=300, n_real=4, n_sources=200, inr=100.0, seed=24, window_T=16, window_F=4),           # ragged channel tile
]


@pytest.mark.gpu
def test_static_entry_point_equals_the_allocating_one_call_after_call():
    want = [_existing(kw) for kw in CALLS]
    # the calls in a row, then the first configuration once more on top of what the others left in the array
    for i, kw in enumerate(CALLS + CALLS[:1]):
        got = _static(kw, fill=1.0e30 if i % 2 else -7.0)
        _assert_same(kw, got, want[i % len(CALLS)])


@pytest.mark.gpu
def test_static_entry_point_back_to_back_on_one_stream_without_a_sync_between():
    """Two calls enqueued one after the other on the same stream are ordered, so the second may reuse the array as soon
    as the first one's kernels are done with it: both outputs must still be right."""
    a, b = CALLS[0], CALLS[1]
    want_a, want_b = _existing(a), _existing(b)
    outs = []
    for kw in (a, b):
        vis = torch.empty(kw["n_time"], kw["n_real"], kw["n_chan"], 4, 2, dtype=torch.float32, device="cuda")
        truth = torch.empty(kw["n_time"] // kw["window_T"], kw["n_real"], (kw["n_chan"] + 31) // 32, dtype=torch.int32, device="cuda")
        rfi.sim42_generate_static(vis, truth, kw["inr"], seed=kw["seed"], n_sources=kw["n_sources"],
                                  n_broadband=kw.get("n_broadband", 5), window_T=kw["window_T"], window_F=kw["window_F"])
        outs.append((vis, truth))
    torch.cuda.synchronize()
    _assert_same(a, outs[0], want_a)
    _assert_same(b, outs[1], want_b)


@pytest.mark.gpu
def test_static_entry_point_at_its_size_limit():
    """512 realisations x 512 channels fills the array exactly; a short block keeps the run small."""
    kw = dict(n_time=10, n_chan=512, n_real=binding.SIM42_STATIC_MAX_REAL, n_sources=3, inr=4.0, seed=5, window_T=10, window_F=2)
    assert kw["n_real"] * kw["n_chan"] == binding.SIM42_STATIC_MAX_CELLS
    _assert_same(kw, _static(kw, fill=0.0), _existing(kw))


@pytest.mark.parametrize("n_real,n_chan", [(binding.SIM42_STATIC_MAX_REAL + 1, 8), (512, 513), (300, 1024)])
def test_static_entry_point_refuses_what_does_not_fit(n_real, n_chan):
    """The cap is checked before anything touches the GPU, so this runs anywhere.  The pointer is never dereferenced."""
    lib = rfi.load_library()
    assert lib.rfi_sim42_static_bytes() <= 8 << 20
    cfg = binding.Sim42Config(20, n_chan, n_real, 5, 1, 0, 0, 1, 1.0, 10, 2, 3)
    rc = lib.rfi_sim42_generate_static(ctypes.byref(cfg), ctypes.c_void_p(256), None, None)
    assert rc == -1
    msg = lib.rfi_last_cuda_error().decode()
    assert "do not fit the built-in work area" in msg and str(binding.SIM42_STATIC_MAX_CELLS) in msg
