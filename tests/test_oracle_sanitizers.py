"""the C++ oracle under AddressSanitizer + UndefinedBehaviorSanitizer.  The two oracle sources are
built with -fsanitize=address,undefined into a temporary library and every entry point the parity tests rely on is driven
through it in a fresh interpreter (the sanitizer runtime has to be loaded first, hence LD_PRELOAD and a subprocess).
An out-of-bounds index, a use of uninitialised stack beyond a frame, a signed overflow or a misaligned access in the
checker itself would fail here instead of silently bending a parity verdict."""
import os
import shutil
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
import numpy as np
from oracle import rfi_oracle as orc
rng = np.random.default_rng(3)
# the whole path: ragged cell count, K = 3 sets, NaN / Inf / all-zero windows, fp16 and fp32 storage, T x F footprints
for dtype, M, F, cells in ((np.float32, 16, 1, 37), (np.float16, 8, 1, 5), (np.float32, 10, 2, 12), (np.float64, 5, 4, 8)):
    vis = rng.standard_normal((M * 12, cells, 4, 2)).astype(dtype)
    vis[3, 1] = np.nan; vis[M + 1, 2] = np.inf; vis[2 * M:3 * M, 0] = 0
    thr = [[1.0, 0.05, 0.6, 0.5], [0.7, 0.0, 9.0, 1.0], [0.5, 0.2, 0.3, 0.1]]
    res = orc.process(vis, M, M * 4, thr, F=F)
    assert res.flags.shape == (3, 12, cells) and res.weight.min() >= 0
    orc.pack_flags(res.flags[0], 1, cells)
    orc.process(vis, M, M * 4, thr[:1], want_stats=False, n_threads=1, F=F)
w = rng.standard_normal((20, 4, 2))
orc.stokes(w[0]); orc.window_stats(w, 1.0); orc.decide(0.3, 0.1, 0.2, 0.05, 0.6, 0.5)
# the tables oracle and the RL record: every mask bit once, a window that overflows half precision
vis = rng.standard_normal((64, 9, 4, 2)).astype(np.float32)
for mask in (0, 0x3FFF, 0x3C50, 0x2AAA, 0x1555):
    orc.tables_process(vis, 16, 32, [1.0, 0.05, 0.6, 0.5], mask)
win = rng.standard_normal((7, 20, 4, 2)).astype(np.float32)
win[2] *= 300.0; win[3] *= 1e-4; win[4, 5] = np.nan
for mask in (0, 0x3FFF, 0x3C50):
    orc.rl_evaluate(win, mask, [1.0, 0.05, 0.6, 0.5])
    orc.rl_cost(mask, 20)
maps = open("/proc/self/maps").read()
assert "liboracle_rfi_san.so" in maps and "libasan" in maps, "the instrumented library is not the one that ran"
print("sanitizer-run-ok")
"""


def test_oracle_is_clean_under_asan_and_ubsan():
    gxx = shutil.which("g++")
    asan = subprocess.run([gxx, "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip() if gxx else ""
    if not gxx or not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("g++ with libasan is not available")
    with tempfile.TemporaryDirectory() as tmp:
        lib = os.path.join(tmp, "liboracle_rfi_san.so")
        cmd = [gxx, "-O1", "-g", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-o", lib,
               os.path.join(ROOT, "oracle", "rfi_oracle.cpp"), os.path.join(ROOT, "oracle", "rfi_oracle_tables.cpp")]
        subprocess.run(cmd, check=True)
        env = dict(os.environ, LD_PRELOAD=asan, ORACLE_RFI_LIB=lib, PYTHONPATH=ROOT,
                   ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=86", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
        res = subprocess.run([sys.executable, "-c", DRIVER], capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert res.returncode == 0 and "sanitizer-run-ok" in res.stdout, res.stderr[-4000:]
    assert "AddressSanitizer" not in res.stderr and "runtime error" not in res.stderr, res.stderr[-4000:]
