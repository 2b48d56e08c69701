"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the whole chunk is
generated and processed on the device; a seeded sample of cells (all time samples of each) is brought back and
compared with the fp64 oracle element by element, plus properties that hold at any size."""
import numpy as np
import pytest
import torch

import paper_2412_14775_b200 as rfi
from paper_2412_14775_b200 import synth
from tests.parity_util import compare, fp16_vs_fp32_original

pytestmark = pytest.mark.gpu


def _sample_cells(w, truth, n_clean, n_rfi, seed):
    g = torch.Generator().manual_seed(seed)
    has = truth.any(0).cpu()
    rfi_cells = torch.nonzero(has).flatten()
    clean = torch.nonzero(~has).flatten()
    pick = torch.cat([rfi_cells[torch.randperm(rfi_cells.numel(), generator=g)[:n_rfi]],
                      clean[torch.randperm(clean.numel(), generator=g)[:n_clean]]])
    return pick.sort().values


def _run_full(name, K, n_clean=768, n_rfi=256, layout="time_major", vs_fp32_original=False):
    w = synth.WORKLOADS[name]
    need = w.input_bytes * (1.15 + (1.0 if layout == "cell_major" else 0.0) + (2.0 if vs_fp32_original else 0.0)) + 6e9
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip("not enough free device memory for the full-size chunk")
    dev = torch.device("cuda")
    sub32 = None
    if vs_fp32_original:
        # the same seeded chunk BEFORE rounding to half (make_chunk rounds as its last step)
        vis32, truth = synth.make_chunk(w.scaled(fp16=False), seed=1234, device=dev)
        vis = vis32.to(torch.float16)
    else:
        vis, truth = synth.make_chunk(w, seed=1234, device=dev)
    W, F = w.window_M * w.window_F, w.window_F
    thr = synth.default_thresholds(W) if K == 1 else synth.sweep_thresholds(W, K)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if F > 1:
        plan.set_window_freq(F)
    plan.set_thresholds(thr)
    avg, weight, stats = plan.alloc_outputs(stats=True)
    if layout == "cell_major":
        plan.set_layout("cell_major")
        d_in = vis.permute(1, 2, 0, 3, 4).contiguous()          # vis[b][c][t][pol][re,im]
        del vis                                                 # one resident copy: the sample below is read through
        vis = d_in.permute(2, 0, 1, 3, 4)                       # the time-major VIEW of the cell-major buffer
    else:
        d_in = vis
    plan.process_chunk(d_in, avg, weight, stats)                # auto variant: what bench.py times
    torch.cuda.synchronize()
    assert plan.launch_count == 1
    flags = rfi.unpack_flags(plan.get_flags(), w.n_chan).reshape(K, plan.n_win, plan.n_cells)
    # properties at full size
    wt = weight.reshape(K, plan.n_out, plan.n_cells).long()
    kept = (~flags).reshape(K, plan.n_out, w.n_int // w.window_M, plan.n_cells).sum(2) * w.window_M
    assert torch.equal(wt, kept)                                 # weight = unflagged sample count
    assert torch.isfinite(avg).all()
    s = stats.reshape(3, plan.n_win, plan.n_cells)
    assert (s[1] >= 0).all() and (s[1] <= 1 + 1e-6).all() and (s[2] >= 0).all() and (s[2] <= 1 + 1e-6).all()
    # sampled cells against the oracle
    idx = _sample_cells(w, truth.reshape(plan.n_win, plan.n_cells), n_clean, n_rfi, seed=3)
    if F > 1:                                                    # whole footprints: the F channels of a window share a flag
        idx = torch.unique((idx // F)[:, None] * F + torch.arange(F)[None, :]).sort().values
    idx = idx.to(dev)
    sub = vis.reshape(w.n_time, plan.n_cells, 4, 2)[:, idx].cpu().numpy()
    if vs_fp32_original:
        sub32 = vis32.reshape(w.n_time, plan.n_cells, 4, 2)[:, idx].cpu().numpy()
        del vis32
    out = {
        "avg": avg.reshape(K, plan.n_out, plan.n_cells, 4, 2)[:, :, idx].cpu().numpy().view(np.complex64).reshape(K, plan.n_out, -1, 4),
        "weight": wt[:, :, idx].cpu().numpy(),
        "flags": flags[:, :, idx].cpu().numpy(),
        "tau": s[0][:, idx].cpu().numpy(), "r_re": s[1][:, idx].cpu().numpy(), "r_im": s[2][:, idx].cpu().numpy(),
    }
    used = plan.last_variant
    plan.destroy()
    del vis, d_in, avg, weight, stats
    torch.cuda.empty_cache()
    rep = compare(sub, w.window_M, w.n_int, thr, out, tol=2e-3 if w.fp16 else 1e-5, fp16=w.fp16, F=F)
    if sub32 is not None:
        rep.update(fp16_vs_fp32_original(sub32, w.window_M, w.n_int, thr, out))
    return rep, used


def test_lofar_fp32_full_size():
    rep, used = _run_full("lofar", 1)
    assert used == "direct" and rep["flag_mismatch_unexplained"] == 0


def test_lofar_fp16_full_size():
    """configs[2]: statistics against the oracle on the same fp16-rounded values (2e-3), and -- SURVEY 8(c)-T,
    PAPER.md:251,269 -- flag agreement >= 99.9 % against the oracle on the ORIGINAL fp32 values."""
    rep, used = _run_full("lofar_fp16", 1, vs_fp32_original=True)
    print({k: rep[k] for k in ("flag_agreement", "flag_agreement_vs_fp32_original", "quantisation_dtau_max",
                               "quantisation_dr_max", "outputs_skipped", "outputs_total")})
    assert rep["flag_agreement"] >= 0.999
    assert rep["flag_agreement_vs_fp32_original"] >= 0.999


def test_sweep_K64_full_size():
    rep, used = _run_full("sweep", 64, n_clean=192, n_rfi=64)
    assert used == "batched" and rep["K"] == 64 and rep["flag_mismatch_unexplained"] == 0


def test_large_K64_full_size():
    """configs[3] shape with the K = 64 sweep (DESIGN.md section 7 row "large K=64")."""
    rep, used = _run_full("large", 64, n_clean=96, n_rfi=96)
    assert used == "batched" and rep["K"] == 64 and rep["flag_mismatch_unexplained"] == 0


@pytest.mark.parametrize("name,K", [("lofar", 1), ("lofar_fp16", 1), ("sweep", 64)])
def test_cell_major_full_size(name, K):
    """Cell-major input vis[b][c][t][pol] at the sizes bench.py times."""
    rep, used = _run_full(name, K, n_clean=192, n_rfi=64, layout="cell_major")
    assert used == ("tma" if K == 1 else "batched")
    assert rep["flag_agreement"] >= 0.999 if synth.WORKLOADS[name].fp16 else rep["flag_mismatch_unexplained"] == 0


def test_large_array_full_size():
    """BASELINE.json configs[3] as read in DESIGN.md (C4): 2926 baselines x 256 channels, W=32, one 3072-sample
    integration per chunk (73.6 GB); bursts, tones and 100-sigma unpolarised spikes."""
    rep, used = _run_full("large", 1, n_clean=384, n_rfi=384)
    assert used == "direct" and rep["flag_mismatch_unexplained"] == 0


# ---- the shapes DESIGN.md section 7 quotes a time for that had no full-size test ----------------
def test_fp16_storage_K64_full_size():
    rep, used = _run_full("lofar_fp16", 64, n_clean=160, n_rfi=64)
    assert used == "batched" and rep["K"] == 64 and rep["flag_agreement"] >= 0.999


@pytest.mark.parametrize("K", [1, 64])
def test_tf10x2_full_size(K):
    """The paper's 10 x 2 footprint on the lofar shape, single set and the K = 64 sweep."""
    rep, used = _run_full("lofar_tf10x2", K, n_clean=160 if K > 1 else 512, n_rfi=64 if K > 1 else 128)
    assert used == ("batched" if K > 1 else "direct") and rep["flag_mismatch_unexplained"] == 0


def test_large_array_cell_major_full_size():
    rep, used = _run_full("large", 1, n_clean=256, n_rfi=256, layout="cell_major")
    assert used == "tma" and rep["flag_mismatch_unexplained"] == 0


@pytest.mark.parametrize("mode", ["tables", "adaptive", "adaptive_baseline", "classes"])
def test_other_modes_at_the_lofar_size(mode):
    """Tables arithmetic (mask 0x3C50: bit for bit against oracle_tables_process), on-line adaptation per class and per
    baseline (the flags of the chunk after the first update against the oracle with the thresholds then in force) and
    cross / auto threshold classes, on the full lofar chunk, through the verification leg bench.py runs after timing
    these modes (bench.mode_parity: thresholds read back, one launch with the statistics planes, sampled cells through
    the oracle group by group)."""
    import types
    import bench
    w = synth.WORKLOADS["lofar"]
    if torch.cuda.mem_get_info()[0] < w.input_bytes * 1.15 + 8e9:
        pytest.skip("not enough free device memory for the full-size chunk")
    dev = torch.device("cuda")
    vis, truth = synth.make_chunk(w, seed=1234, device=dev)
    thr = synth.default_thresholds(w.window_M)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    args = types.SimpleNamespace(layout="time_major", adaptive=0.05 if mode.startswith("adaptive") else 0.0,
                                 adaptive_scope="baseline" if mode == "adaptive_baseline" else "class",
                                 arith="tables" if mode == "tables" else "fast", mask=0x3C50, K=1)
    two_classes = mode == "classes"
    if two_classes:
        plan.set_baseline_classes(synth.auto_baseline_mask(w).int().tolist())
        plan.set_thresholds([[thr[0], synth.auto_thresholds(w.window_M)]])
    else:
        plan.set_thresholds(thr)
    if mode == "tables":
        plan.set_arithmetic("tables", 0x3C50)
    if args.adaptive > 0:
        plan.set_adaptive(0.05, 0.5)
        plan.set_adaptive_scope(args.adaptive_scope)
    avg, weight, _ = plan.alloc_outputs()
    plan.process_chunk(vis, avg, weight)                        # chunk 1 (with adaptation on: the first update follows it)
    torch.cuda.synchronize()
    if args.adaptive > 0:
        now = plan.get_stream_thresholds()[:, 1:] if mode == "adaptive_baseline" else np.array(plan.get_thresholds())[:, 1:]
        assert not np.allclose(now, np.array(thr[0][1:])[None, :])      # the thresholds did move
    rep = bench.mode_parity(args, w, plan, vis, truth, thr, two_classes, dev)
    plan.destroy()
    assert rep["status"] == "ok", rep
    assert rep["flag_mismatch_unexplained"] == 0 and rep["cells_sampled"] >= 500, rep
    if mode == "tables":
        assert rep["against"].startswith("tables oracle") and rep["flag_mismatch"] == 0
