"""GPU parity of the paper-literal mixed-precision mode (rfi_plan_set_arithmetic, RFI_ARITH_TABLES) against the
step-by-step CPU restatement of Tables 1-2 (oracle/rfi_oracle_tables.cpp).  Both sides perform the same IEEE
operations in the same order, so statistics and flags are compared BIT FOR BIT; the averages (fp32 sums on the
GPU, fp64 in the oracle) to relative 1e-5 with the floor of DESIGN.md section 5."""
import math

import numpy as np
import pytest
import torch

import paper_2412_14775_b200 as rfi
from paper_2412_14775_b200 import synth
from oracle import rfi_oracle as orc

pytestmark = pytest.mark.gpu
PAPER = 0x3C50


def run_tables(w, vis, thr, mask):
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_arithmetic("tables", mask)
    plan.set_thresholds([thr])
    avg, weight, stats = plan.alloc_outputs(stats=True)
    avg.fill_(float("nan")); weight.fill_(-1); stats.fill_(float("nan"))
    plan.process_chunk(vis.cuda(), avg, weight, stats)
    torch.cuda.synchronize()
    assert plan.last_variant == "tables" and plan.launch_count == 1
    flags = rfi.unpack_flags(plan.get_flags(), w.n_chan).reshape(plan.n_win, plan.n_cells).cpu().numpy()
    s = stats.cpu().numpy().reshape(3, plan.n_win, plan.n_cells)
    out = dict(tau=s[0], r_re=s[1], r_im=s[2], flags=flags,
               avg=avg.cpu().numpy().reshape(plan.n_out, plan.n_cells, 8),
               weight=weight.cpu().numpy().reshape(plan.n_out, plan.n_cells).astype(np.int64))
    plan.destroy()
    return out


def check_tables(w, thr, mask, seed=1234, mutate=None):
    vis, _ = synth.make_chunk(w, seed=seed)
    if mutate is not None:
        mutate(vis)
    out = run_tables(w, vis, thr, mask)
    ref = orc.tables_process(vis.numpy().reshape(w.n_time, w.n_cells, 4, 2), w.window_M, w.n_int, thr, mask)
    for key, r in (("tau", ref.tau[0]), ("r_re", ref.r_re), ("r_im", ref.r_im)):
        nan = np.isnan(r)                      # NaN payloads / signs differ between x86 and the GPU: positions must agree
        np.testing.assert_array_equal(np.isnan(out[key]), nan, err_msg=f"{key} NaN positions, mask={mask:#x}")
        np.testing.assert_array_equal(out[key][~nan].view(np.uint32), r[~nan].view(np.uint32), err_msg=f"{key} mask={mask:#x}")
    np.testing.assert_array_equal(out["flags"], ref.flags[0].astype(bool))
    np.testing.assert_array_equal(out["weight"], ref.weight[0])
    a = ref.avg[0].view(np.float64).reshape(out["avg"].shape)
    rms = math.sqrt(float((a ** 2).mean()))
    fin = np.isfinite(a)
    assert (np.abs(out["avg"] - a)[fin] <= 1e-5 * np.maximum(np.abs(a[fin]), rms)).all()
    return out, ref


@pytest.mark.parametrize("mask", [0, PAPER, 0x3FFF, 0x007F, 0x3F80, 0x2AAA, 0x1555, 0x0001, 0x0400])
def test_tables_mode_is_bit_exact(mask):
    w = synth.WORKLOADS["lofar"].scaled(n_stations=5, n_time=640, n_int=320, window_M=20, burst_cell_frac=0.15)
    c = (20 * 0.9 + 1) / 19
    out, ref = check_tables(w, (0.9, 0.08 * c, 0.6 * c, 0.5), mask)
    assert 0.0 < out["flags"].mean() < 0.9


def test_tables_any_mask_bit_exact_through_the_per_sample_instantiations(monkeypatch):
    """An RL search visits arbitrary masks: 24 random ones (even windows -> rfi_tables_kernel<2, ps, -1>, the 8
    per-sample bits compile-time) bit-exact against the oracle and equal to the fully run-time-mask kernel."""
    w = synth.WORKLOADS["lofar"].scaled(n_stations=4, n_time=320, n_int=160, window_M=16, burst_cell_frac=0.15)
    c = (16 * 0.9 + 1) / 15
    thr = (0.9, 0.08 * c, 0.6 * c, 0.5)
    rng = np.random.default_rng(14)
    vis, _ = synth.make_chunk(w, seed=1234, device="cpu")
    for mask in rng.integers(1, 1 << 14, 24).tolist():
        out, ref = check_tables(w, thr, int(mask))
        monkeypatch.setenv("RFI_TABLES_PS", "0")
        rt = run_tables(w, vis, thr, int(mask))
        monkeypatch.delenv("RFI_TABLES_PS")
        for key in ("tau", "r_re", "r_im", "flags", "weight", "avg"):
            np.testing.assert_array_equal(out[key], rt[key], err_msg=f"{key}, mask {mask:#06x}")
    # the block length does not enter the arithmetic (sums are sequential in the samples): 1, 2 and 4 rows agree bit for bit
    for mask in (0, 0x3C50, 0x0A53):
        ref_out = None
        for rows in (1, 2, 4):
            monkeypatch.setenv("RFI_TABLES_ROWS", str(rows))
            o = run_tables(w, vis, thr, mask)
            monkeypatch.delenv("RFI_TABLES_ROWS")
            if ref_out is None:
                ref_out = o
            for key in ("tau", "r_re", "r_im", "flags", "weight", "avg"):
                np.testing.assert_array_equal(o[key], ref_out[key], err_msg=f"{key}, mask {mask:#06x}, rows {rows}")


@pytest.mark.parametrize("M,n_int,n_time,n_chan", [(16, 64, 256, 13), (5, 20, 40, 64), (3, 12, 48, 16)])
def test_tables_mode_ragged_shapes(M, n_int, n_time, n_chan):
    w = synth.Workload("tab", 4, False, n_chan, n_time, M, n_int, burst_cell_frac=0.2, channel_gain=True)
    check_tables(w, (1.0, 0.05, 1.4, 0.7), PAPER, seed=M)
    check_tables(w, (1.0, 0.05, 1.4, 0.7), 0x3FFF, seed=M + 1)


def test_tables_mode_overflow_nan_and_scale():
    """Amplitudes above 255.9 overflow y = x^2 in half (PAPER.md:172's penalty case): non-finite tau, flagged, on both
    sides alike; NaN input; all-zero cell (the eps guards give tau = -c, r = 0)."""
    w = synth.Workload("tab_deg", 4, True, 16, 128, 16, 64, burst_cell_frac=0.2)

    def mutate(vis):
        v = vis.view(w.n_time, w.n_cells, 4, 2)
        v[:, 3] *= 400.0
        v[:, 5] = 0.0
        v[17, 9, 2, 1] = float("nan")
        v[:, 11] *= 1e-3

    out, ref = check_tables(w, (1.0, 0.1, 1.2, 0.6), 0x3FFF, mutate=mutate)
    assert out["flags"][:, 3].all() and not np.isfinite(out["tau"][:, 3]).any()
    assert out["flags"][1, 9]
    out32, _ = check_tables(w, (1.0, 0.1, 1.2, 0.6), 0, mutate=mutate)
    assert np.isfinite(out32["tau"][:, 3]).all()
    assert np.allclose(out32["tau"][:, 5], -17 / 15) and (out32["r_re"][:, 5] == 0).all()


def test_tables_mode_rejects_unsupported_plans():
    plan = rfi.RfiPlan(4, 10, 32, 64, 16, rfi.RFI_FP16)
    plan.set_arithmetic("tables", 0)
    plan.set_thresholds([[1.0, 0.1, 1.0, 0.5]])
    avg, weight, _ = plan.alloc_outputs()
    vis = torch.zeros(64, 10, 32, 4, 2, dtype=torch.float16, device="cuda")
    with pytest.raises(rfi.RfiError) as e:
        plan.process_chunk(vis, avg, weight)
    assert e.value.code == -1
    plan.destroy()


def test_flag_agreement_of_the_learned_assignment_with_the_fast_path():
    """mixed precision changes < 1 % of the flags.  Same data through the fast fp32 kernels and
    through the tables with the learned assignment: agreement is reported and must exceed 99 %."""
    w = synth.WORKLOADS["lofar"].scaled(n_stations=8, n_time=1536, n_int=768)
    thr = synth.default_thresholds(16)[0]
    vis, _ = synth.make_chunk(w, seed=21)
    tab = run_tables(w, vis, thr, PAPER)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_thresholds([thr])
    avg, weight, _ = plan.alloc_outputs()
    plan.process_chunk(vis.cuda(), avg, weight)
    torch.cuda.synchronize()
    fast = rfi.unpack_flags(plan.get_flags(), w.n_chan).reshape(plan.n_win, plan.n_cells).cpu().numpy()
    plan.destroy()
    agree = float((fast == tab["flags"]).mean())
    assert agree > 0.99, agree


def test_tables_mode_with_baseline_classes():
    """Per-class thresholds in the tables arithmetic: every cell bit-exact against the oracle run with its class's set."""
    w = synth.Workload("tab_cls", 5, True, 32, 256, 16, 128, burst_cell_frac=0.15)
    vis, _ = synth.make_chunk(w, seed=3)
    autos = synth.auto_baseline_mask(w).numpy()
    sets = [(1.0, 0.1, 0.7, 0.5), (0.6, 0.02, 0.3, 0.52)]
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_arithmetic("tables", PAPER)
    plan.set_baseline_classes(autos.astype(int).tolist())
    plan.set_thresholds([[list(sets[0]), list(sets[1])]])
    avg, weight, stats = plan.alloc_outputs(stats=True)
    plan.process_chunk(vis.cuda(), avg, weight, stats)
    torch.cuda.synchronize()
    flags = rfi.unpack_flags(plan.get_flags(), w.n_chan).reshape(plan.n_win, plan.n_cells).cpu().numpy()
    tau = stats.cpu().numpy().reshape(3, plan.n_win, plan.n_cells)[0]
    plan.destroy()
    v = vis.numpy().reshape(w.n_time, w.n_cells, 4, 2)
    cell_auto = np.repeat(autos, w.n_chan)
    for cls in (0, 1):
        sel = np.nonzero(cell_auto == bool(cls))[0]
        ref = orc.tables_process(v[:, sel], w.window_M, w.n_int, sets[cls], PAPER)
        np.testing.assert_array_equal(tau[:, sel].view(np.uint32), ref.tau[0].view(np.uint32))
        np.testing.assert_array_equal(flags[:, sel], ref.flags[0].astype(bool))
