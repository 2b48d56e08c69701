"""ctypes loader for the fp64 CPU oracle (oracle/rfi_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It holds
no arithmetic of the method: it builds the C++ file with g++, loads it and
marshals numpy arrays.  Nothing here imports the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rfi_oracle.cpp")
_SRC_TABLES = os.path.join(_HERE, "rfi_oracle_tables.cpp")
_LIB = os.path.join(_HERE, "liboracle_rfi.so")
_lib = None

_STORAGE = {np.dtype(np.float32): 0, np.dtype(np.float16): 1, np.dtype(np.float64): 2}


def build(force: bool = False) -> str:
    """Compile oracle/rfi_oracle.cpp -> oracle/liboracle_rfi.so (g++ -O2 -fopenmp)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_TABLES))):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
           "-ffp-contract=off", "-o", tmp, _SRC, _SRC_TABLES]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        # ORACLE_RFI_LIB: load a pre-built library instead (tests/test_oracle_sanitizers.py: the same sources built
        # with -fsanitize=address,undefined)
        lib = ctypes.CDLL(os.environ.get("ORACLE_RFI_LIB") or build())
        c_dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_rfi_stokes.argtypes = [c_dp, c_dp]
        lib.oracle_rfi_stokes.restype = None
        lib.oracle_rfi_window_stats.argtypes = [c_dp, ctypes.c_int, ctypes.c_double, c_dp, c_dp, c_dp]
        lib.oracle_rfi_window_stats.restype = ctypes.c_int
        lib.oracle_rfi_decide.argtypes = [ctypes.c_double] * 6
        lib.oracle_rfi_decide.restype = ctypes.c_int
        lib.oracle_rfi_process.argtypes = [
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_int64,
            ctypes.c_int, c_dp, c_dp, c_dp, c_dp, ctypes.c_void_p, c_dp, ctypes.c_void_p, ctypes.c_int]
        lib.oracle_rfi_process.restype = ctypes.c_int
        lib.oracle_rfi_process_tf.argtypes = [
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
            ctypes.c_int, c_dp, c_dp, c_dp, c_dp, ctypes.c_void_p, c_dp, ctypes.c_void_p, ctypes.c_int]
        lib.oracle_rfi_process_tf.restype = ctypes.c_int
        lib.oracle_rfi_pack_flags.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64,
                                              ctypes.c_int64, ctypes.c_void_p]
        lib.oracle_rfi_pack_flags.restype = ctypes.c_int
        c_fp = ctypes.POINTER(ctypes.c_float)
        cf, cu = ctypes.c_float, ctypes.c_uint32
        lib.oracle_tables_sk.argtypes = [c_fp, c_fp, ctypes.c_int, cf, cf, cf, cu, c_fp]
        lib.oracle_tables_sk.restype = ctypes.c_int
        lib.oracle_tables_ds.argtypes = [c_fp, c_fp, c_fp, ctypes.c_int, cf, cu, c_fp]
        lib.oracle_tables_ds.restype = ctypes.c_int
        lib.oracle_tables_process.argtypes = [
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_int64, cf, cf, cf, cf, cu,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, c_dp, ctypes.c_void_p, ctypes.c_int]
        lib.oracle_tables_process.restype = ctypes.c_int
        lib.oracle_tables_to_half.argtypes = [cf]
        lib.oracle_tables_to_half.restype = cf
        lib.oracle_rl_record_doubles.argtypes = []
        lib.oracle_rl_record_doubles.restype = ctypes.c_int
        lib.oracle_rl_cost.argtypes = [cu, ctypes.c_int, c_dp, c_dp]
        lib.oracle_rl_cost.restype = None
        lib.oracle_rl_evaluate.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, cu, cf, cf, cf, cf, ctypes.c_double,
                                           c_dp, ctypes.c_int]
        lib.oracle_rl_evaluate.restype = ctypes.c_int
        lib.oracle_rfi_max_threads.argtypes = []
        lib.oracle_rfi_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def stokes(v8) -> np.ndarray:
    """(I,Q,U,V) as 8 reals from one sample's 8 reals (xx,xy,yx,yy interleaved re,im)."""
    v = np.ascontiguousarray(v8, dtype=np.float64).reshape(8)
    s = np.empty(8, dtype=np.float64)
    _load().oracle_rfi_stokes(_dp(v), _dp(s))
    return s


def window_stats(win, d: float):
    """(tau, r_re, r_im) of one window; win is [M,8] reals or [M,4] complex."""
    w = np.asarray(win)
    if np.iscomplexobj(w):
        w = np.ascontiguousarray(w.astype(np.complex128)).view(np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64).reshape(-1, 8)
    t, a, b = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _load().oracle_rfi_window_stats(_dp(w), w.shape[0], float(d),
                                    ctypes.byref(t), ctypes.byref(a), ctypes.byref(b))
    return t.value, a.value, b.value


def decide(tau, r_re, r_im, s_low, s_high, gamma) -> int:
    return _load().oracle_rfi_decide(float(tau), float(r_re), float(r_im),
                                     float(s_low), float(s_high), float(gamma))


@dataclass
class OracleResult:
    tau: np.ndarray      # [K, n_win, n_cells] float64
    r_re: np.ndarray     # [n_win, n_cells]
    r_im: np.ndarray     # [n_win, n_cells]
    flags: np.ndarray    # [K, n_win, n_cells] uint8, 1 = flagged
    avg: np.ndarray      # [K, n_out, n_cells, 4] complex128
    weight: np.ndarray   # [K, n_out, n_cells] int64


def process(vis, M: int, n_int: int, thresholds, n_threads: int = 0, want_stats: bool = True,
            F: int = 1) -> OracleResult:
    """Run the whole path.  Window footprint: M time samples x F adjacent cells (W = M*F).

    vis: real array [n_time, n_cells, 4, 2] (float16/32/64) or complex [n_time, n_cells, 4].
    thresholds: [K,4] rows of (d, s_low, s_high, gamma).
    """
    a = np.asarray(vis)
    if np.iscomplexobj(a):
        a = np.ascontiguousarray(a)
        a = a.view(np.float32 if a.dtype == np.complex64 else np.float64).reshape(*a.shape, 2)
    a = np.ascontiguousarray(a)
    if a.dtype not in _STORAGE:
        raise TypeError(f"unsupported storage dtype {a.dtype}")
    n_time, n_cells = a.shape[0], a.shape[1]
    assert a.shape[2:] == (4, 2), a.shape
    thr = np.ascontiguousarray(thresholds, dtype=np.float64).reshape(-1, 4)
    K = thr.shape[0]
    n_win, n_out = n_time // M, n_time // n_int
    tau = np.empty((K, n_win, n_cells), np.float64) if want_stats else None
    r_re = np.empty((n_win, n_cells), np.float64) if want_stats else None
    r_im = np.empty((n_win, n_cells), np.float64) if want_stats else None
    flags = np.empty((K, n_win, n_cells), np.uint8)
    avg = np.empty((K, n_out, n_cells, 8), np.float64)
    weight = np.empty((K, n_out, n_cells), np.int64)
    rc = _load().oracle_rfi_process_tf(
        a.ctypes.data, _STORAGE[a.dtype], n_time, n_cells, int(M), int(F), int(n_int), K, _dp(thr),
        _dp(tau), _dp(r_re), _dp(r_im), flags.ctypes.data, _dp(avg), weight.ctypes.data, int(n_threads))
    if rc != 0:
        raise ValueError("oracle_rfi_process: invalid arguments")
    return OracleResult(tau, r_re, r_im, flags, avg.view(np.complex128).reshape(K, n_out, n_cells, 4), weight)


def pack_flags(flags, n_baselines: int, n_chan: int) -> np.ndarray:
    """[rows, n_baselines*n_chan] bytes -> [rows, n_baselines, ceil(n_chan/32)] uint32 (include/rfi.h layout)."""
    f = np.ascontiguousarray(flags, dtype=np.uint8)
    rows = int(np.prod(f.shape[:-1])) if f.ndim > 1 else 1
    assert f.shape[-1] == n_baselines * n_chan
    wpb = (n_chan + 31) // 32
    out = np.empty((rows, n_baselines, wpb), np.uint32)
    rc = _load().oracle_rfi_pack_flags(f.ctypes.data, rows, n_baselines, n_chan, out.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_rfi_pack_flags: invalid arguments")
    return out.reshape(*f.shape[:-1], n_baselines, wpb)


def max_threads() -> int:
    return _load().oracle_rfi_max_threads()


# ---- paper-literal mixed-precision arithmetic (Tables 1-2, oracle/rfi_oracle_tables.cpp) -----------------------
def _fp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def tables_sk(xr, xi, d, s_low, s_high, mask):
    """Table 1 on one window of I = xr + j xi (float32).  Returns (tau, flag)."""
    xr = np.ascontiguousarray(xr, np.float32); xi = np.ascontiguousarray(xi, np.float32)
    t = ctypes.c_float()
    f = _load().oracle_tables_sk(_fp(xr), _fp(xi), len(xr), d, s_low, s_high, int(mask), ctypes.byref(t))
    return t.value, f


def tables_ds(q, u, v, gamma, mask):
    """Table 2 on one window of real (or imaginary) parts q, u, v (float32).  Returns (r, flag)."""
    q = np.ascontiguousarray(q, np.float32); u = np.ascontiguousarray(u, np.float32); v = np.ascontiguousarray(v, np.float32)
    r = ctypes.c_float()
    f = _load().oracle_tables_ds(_fp(q), _fp(u), _fp(v), len(q), gamma, int(mask), ctypes.byref(r))
    return r.value, f


def to_half(x: float) -> float:
    return _load().oracle_tables_to_half(float(x))


def tables_process(vis, M: int, n_int: int, threshold, mask: int, n_threads: int = 0) -> OracleResult:
    """The whole path in the tables' arithmetic.  vis float32 [n_time, n_cells, 4, 2]; threshold (d, s_low, s_high, gamma)."""
    a = np.ascontiguousarray(vis, np.float32)
    n_time, n_cells = a.shape[0], a.shape[1]
    assert a.shape[2:] == (4, 2), a.shape
    n_win, n_out = n_time // M, n_time // n_int
    tau = np.empty((n_win, n_cells), np.float32); r_re = np.empty_like(tau); r_im = np.empty_like(tau)
    flags = np.empty((n_win, n_cells), np.uint8)
    avg = np.empty((n_out, n_cells, 8), np.float64)
    weight = np.empty((n_out, n_cells), np.int64)
    d, lo, hi, g = [float(np.float32(x)) for x in threshold]
    rc = _load().oracle_tables_process(a.ctypes.data, n_time, n_cells, int(M), int(n_int), d, lo, hi, g, int(mask),
                                       tau.ctypes.data, r_re.ctypes.data, r_im.ctypes.data, flags.ctypes.data,
                                       _dp(avg), weight.ctypes.data, int(n_threads))
    if rc != 0:
        raise ValueError("oracle_tables_process: invalid arguments")
    return OracleResult(tau[None], r_re, r_im, flags[None], avg.view(np.complex128).reshape(1, n_out, n_cells, 4), weight[None])


RL_FIELDS = {"features": slice(0, 10), "bits": slice(10, 24), "errors": slice(24, 45), "op_cost": 45, "conversions": 46,
             "overflow": 47, "underflow": 48, "matches": 49, "reward": 50, "flags": 51}


def rl_cost(mask: int, W: int):
    """(operation cost, type conversions) of a precision mask for window size W (readings T10, T12)."""
    c, v = ctypes.c_double(), ctypes.c_double()
    _load().oracle_rl_cost(int(mask), int(W), ctypes.byref(c), ctypes.byref(v))
    return c.value, v.value


def rl_evaluate(windows, mask: int, threshold, rho: float = 3.0, n_threads: int = 0):
    """The RL environment of PAPER.md:149-172 on windows float32 [n, W, 4, 2]: returns float64 [n, 52] records
    (layout RL_FIELDS; readings T10-T15 in oracle/rfi_oracle_tables.cpp)."""
    a = np.ascontiguousarray(windows, np.float32)
    assert a.ndim == 4 and a.shape[2:] == (4, 2), a.shape
    n, W = a.shape[0], a.shape[1]
    rec = _load().oracle_rl_record_doubles()
    out = np.empty((n, rec), np.float64)
    d, lo, hi, g = [float(np.float32(x)) for x in threshold]
    rc = _load().oracle_rl_evaluate(a.ctypes.data, n, W, int(mask), d, lo, hi, g, float(rho), _dp(out), int(n_threads))
    if rc != 0:
        raise ValueError("oracle_rl_evaluate: invalid arguments")
    return out
