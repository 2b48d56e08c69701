"""CPU tests of the boundary: librfi.so loads, exports every symbol include/rfi.h declares, validates its
arguments, and fails loudly (no CPU fallback) when no B200 is present.  No compute calls."""
import ctypes
import os
import re

import pytest
import torch

import paper_2412_14775_b200 as rfi
from paper_2412_14775_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rfi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rfi_[a-z_0-9]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    lib = rfi.load_library()
    syms = declared_symbols()
    assert len(syms) >= 8 and "rfi_process_chunk" in syms and "rfi_get_flags" in syms
    raw = ctypes.CDLL(rfi.library_path())
    for s in syms:
        assert hasattr(raw, s), f"{s} declared in include/rfi.h but not exported"
    assert sorted(binding.EXPORTS) == syms
    assert b"sm_100a" in lib.rfi_version()


def test_library_is_sm100a_sass_with_tma():
    """The .so must hold sm_100a SASS whose TMA kernel uses the tensor-map bulk copy (UTMALDG)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-sass", rfi.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert "UTMALDG" in out, "TMA variant lost its cp.async.bulk.tensor"
    assert "LDG.E.256" in out or "LDG.E.ENL2.256" in out or ".256" in out, "direct variant lost its 256-bit loads"


@pytest.mark.parametrize("args", [
    dict(n_stations=0), dict(n_baselines=7), dict(n_chan=0), dict(n_time=1000), dict(window_M=1), dict(precision=2),
])
def test_plan_create_rejects_bad_shapes(args):
    base = dict(n_stations=4, n_baselines=6, n_chan=16, n_time=1024, window_M=64, precision=0)
    base.update(args)
    with pytest.raises(rfi.RfiError) as e:
        rfi.RfiPlan(**base)
    assert e.value.code == -1


def test_baseline_counts_cross_and_with_autos():
    rfi.RfiPlan(4, 6, 16, 1024, 64).destroy()
    rfi.RfiPlan(4, 10, 16, 1024, 64).destroy()
    rfi.RfiPlan(48, 1176, 64, 7680, 16, rfi.RFI_FP16, n_int=768).destroy()


def test_integration_and_threshold_validation():
    p = rfi.RfiPlan(4, 6, 16, 1024, 64)
    for bad in (100, 32, 96, 0):
        with pytest.raises(rfi.RfiError):
            p.set_integration(bad)
    p.set_integration(128)
    with pytest.raises(rfi.RfiError):
        p.set_thresholds([[0.0, 0.1, 0.5, 0.3]])              # d must be > 0
    with pytest.raises(rfi.RfiError):
        p.set_thresholds([[1.0, float("nan"), 0.5, 0.3]])
    with pytest.raises(rfi.RfiError):
        p.set_thresholds([])
    p.set_thresholds([[1.0, -float("inf"), float("inf"), float("inf")]])
    lib = rfi.load_library()
    assert lib.rfi_avg_bytes(p._h) == 8 * 6 * 16 * 32
    assert lib.rfi_weight_bytes(p._h) == 8 * 6 * 16 * 4
    assert lib.rfi_flags_bytes(p._h) == 16 * 6 * 1 * 4
    assert lib.rfi_stats_bytes(p._h) == 3 * 16 * 96 * 4
    assert lib.rfi_vis_bytes(p._h) == 1024 * 96 * 32
    p.set_variant("direct")
    with pytest.raises(rfi.RfiError):
        p.set_variant(7)
    p.destroy()


def test_pack_flags_is_the_boundary_layout():
    """binding.pack_flags (argument marshalling for the ground-truth mask) against the oracle's layout pin."""
    import torch
    from oracle import rfi_oracle as orc
    g = torch.Generator().manual_seed(3)
    for B, C in ((3, 64), (4, 45), (2, 7)):
        m = torch.rand(5, B, C, generator=g) < 0.4
        got = rfi.pack_flags(m).numpy().view("uint32")
        ref = orc.pack_flags(m.numpy().reshape(5, B * C).astype("uint8"), B, C)
        assert (got == ref).all()
        assert torch.equal(rfi.unpack_flags(rfi.pack_flags(m), C), m)


def test_baseline_classes_validation():
    plan = rfi.RfiPlan(4, 10, 24, 40, 10)
    plan.set_thresholds([[1.0, 0.1, 1.0, 0.5]])
    plan.set_baseline_classes([0, 1] * 5)
    assert plan.K == 0                                     # thresholds must be set again
    plan.set_thresholds([[[1.0, 0.1, 1.0, 0.5], [0.5, 0.0, 2.0, 0.9]]])
    assert plan.K == 1
    with pytest.raises(ValueError):
        plan.set_thresholds([[1.0, 0.1, 1.0, 0.5]] * 3)   # not pairs
    with pytest.raises(ValueError):
        plan.set_baseline_classes([0] * 9)
    with pytest.raises(rfi.RfiError) as e:
        plan.set_baseline_classes([0] * 9 + [2])
    assert e.value.code == -1
    plan.set_baseline_classes(None)
    plan.set_thresholds([[1.0, 0.1, 1.0, 0.5]])
    plan.destroy()


def test_arithmetic_mode_validation():
    plan = rfi.RfiPlan(4, 10, 24, 40, 10)
    plan.set_arithmetic("tables", 0x3C50)
    plan.set_arithmetic("tables", 0x3FFF)
    plan.set_arithmetic("fast")
    for mode, mask in ((1, 1 << 14), (2, 0), (-1, 0), (0, 1)):
        with pytest.raises(rfi.RfiError) as e:
            plan.set_arithmetic(mode, mask)
        assert e.value.code == -1
    plan.destroy()


def test_window_freq_validation():
    plan = rfi.RfiPlan(4, 10, 24, 40, 10)
    for F in (1, 2, 4, 8):
        plan.set_window_freq(F)
    for F in (0, 3, 16, 64, -2):                   # not a power of two / does not divide 24 channels / too wide
        with pytest.raises(rfi.RfiError) as e:
            plan.set_window_freq(F)
        assert e.value.code == -1
    plan.destroy()


def test_baseline_shard_validation():
    plan = rfi.RfiPlan(48, 1176, 64, 7680, 16)
    plan.set_baseline_shard(588, 588)
    assert plan.n_baselines == 588 and plan.b_first == 588
    for first, count in ((-1, 4), (0, 0), (1000, 177), (1176, 1)):
        with pytest.raises(rfi.RfiError) as e:
            plan.set_baseline_shard(first, count)
        assert e.value.code == -1
    plan.set_baseline_shard(0, 1176)
    plan.destroy()


def test_call_order_errors():
    p = rfi.RfiPlan(4, 6, 16, 1024, 64)
    lib = rfi.load_library()
    ptr, n = ctypes.c_void_p(), ctypes.c_size_t()
    assert lib.rfi_get_flags(p._h, ctypes.byref(ptr), ctypes.byref(n)) == -4       # nothing processed
    assert lib.rfi_process_chunk(p._h, 16, 16, 16, None, None) == -4               # thresholds never set
    p.set_thresholds([[1.0, 0.1, 0.5, 0.3]])
    assert lib.rfi_process_chunk(p._h, None, 16, 16, None, None) == -1             # NULL
    assert lib.rfi_process_chunk(p._h, 8, 16, 16, None, None) == -1                # misaligned
    assert lib.rfi_plan_destroy(None) == -1
    p.destroy()


@pytest.mark.skipif(torch.cuda.is_available(), reason="needs a box WITHOUT a GPU")
def test_no_cpu_fallback_without_gpu():
    """The product path must fail loudly when there is no device: it never computes on the CPU."""
    p = rfi.RfiPlan(4, 6, 16, 1024, 64, n_int=64)
    p.set_thresholds([[1.0, 0.1, 0.5, 0.3]])
    with pytest.raises(rfi.RfiError) as e:
        p.process_chunk_host(torch.zeros(1024, 6, 16, 4, 2))
    assert e.value.code == -5
    lib = rfi.load_library()
    assert lib.rfi_process_chunk(p._h, 256, 256, 256, None, None) == -5
    p.destroy()


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_14775_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f), errors="ignore").read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "rfi_oracle" not in text and "liboracle" not in text, f
    oracle_dir = os.path.join(ROOT, "oracle")
    for f in os.listdir(oracle_dir):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(oracle_dir, f)).read()
            assert "import paper_2412_14775_b200" not in text and "from paper_2412_14775_b200" not in text
            assert "librfi" not in text and "rfi_kernels" not in text
