"""Thin ctypes binding of librfi.so (include/rfi.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module holds no arithmetic of
the method and there is no CPU fallback: if librfi.so is missing or no B200 is present the calls raise.
PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

from . import build as _build

RFI_FP32, RFI_FP16 = 0, 1
VARIANT_AUTO, VARIANT_DIRECT, VARIANT_TMA = 0, 1, 2
_VARIANTS = {"auto": 0, "direct": 1, "tma": 2, "split": 5}
ARITH_FAST, ARITH_TABLES = 0, 1
MASK_PAPER_LEARNED = 0x3C50      # Tables 3-4: Table 1 groups 5,7 and Table 2 groups 4-7 in half

EXPORTS = [
    "rfi_plan_create", "rfi_plan_set_integration", "rfi_plan_set_baseline_shard", "rfi_plan_set_window_freq", "rfi_plan_set_arithmetic", "rfi_plan_set_baseline_classes", "rfi_plan_set_layout", "rfi_set_thresholds",
    "rfi_plan_set_variant", "rfi_process_chunk", "rfi_get_flags", "rfi_confusion_counts", "rfi_plan_set_truth", "rfi_process_chunk_host", "rfi_plan_destroy",
    "rfi_strerror", "rfi_last_cuda_error", "rfi_flags_bytes", "rfi_avg_bytes", "rfi_weight_bytes",
    "rfi_stats_bytes", "rfi_vis_bytes", "rfi_plan_launch_count", "rfi_plan_last_variant", "rfi_version",
    "rfi_probe_read_bandwidth", "rfi_probe_mix_bandwidth", "rfi_sim42_generate", "rfi_sim42_vis_bytes", "rfi_sim42_truth_bytes",
    "rfi_sim42_generate_static", "rfi_sim42_static_bytes",
    "rfi_rl_evaluate", "rfi_rl_evaluate_masks", "rfi_plan_set_adaptive", "rfi_plan_set_adaptive_limit", "rfi_plan_set_adaptive_scope", "rfi_plan_set_stream_thresholds", "rfi_plan_get_stream_thresholds",
    "rfi_plan_get_stream_histograms", "rfi_plan_get_thresholds",
    "rfi_plan_get_adaptive_histogram",
]


class RfiThresholds(ctypes.Structure):
    _fields_ = [("d", ctypes.c_float), ("s_low", ctypes.c_float), ("s_high", ctypes.c_float),
                ("gamma", ctypes.c_float)]


SIM42_MAX_COMPONENTS = 16


class Sim42Config(ctypes.Structure):
    """rfi_sim42_config (include/rfi.h): the section-4.2 simulator of the paper."""
    _fields_ = [("n_time", ctypes.c_int), ("n_chan", ctypes.c_int), ("n_real", ctypes.c_int), ("n_sources", ctypes.c_int),
                ("n_broadband", ctypes.c_int), ("n_narrowband", ctypes.c_int), ("n_narrowdur", ctypes.c_int),
                ("polarized", ctypes.c_int), ("inr", ctypes.c_float), ("window_T", ctypes.c_int), ("window_F", ctypes.c_int),
                ("seed", ctypes.c_uint64)]


class Sim42Component(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("t0", ctypes.c_int), ("t1", ctypes.c_int), ("c0", ctypes.c_int), ("c1", ctypes.c_int),
                ("tries", ctypes.c_int), ("period", ctypes.c_double), ("J", ctypes.c_double * 8)]


class Sim42Realisation(ctypes.Structure):
    _fields_ = [("a", ctypes.c_double), ("u", ctypes.c_double), ("v", ctypes.c_double), ("w", ctypes.c_double),
                ("p_cel", ctypes.c_double), ("p_rfi", ctypes.c_double), ("gain", ctypes.c_double),
                ("n_comp", ctypes.c_int), ("reserved", ctypes.c_int), ("comp", Sim42Component * SIM42_MAX_COMPONENTS)]


class RfiError(RuntimeError):
    def __init__(self, code: int, where: str):
        lib = load_library()
        msg = lib.rfi_strerror(code).decode()
        cuda = lib.rfi_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})" + (f" [{cuda}]" if cuda and where.startswith(("rfi_process", "rfi_sim42", "rfi_probe", "rfi_rl")) else ""))
        self.code = code


_lib = None


def library_path() -> str:
    return _build.LIB


def load_library(build_if_missing: bool = True):
    """dlopen librfi.so (building it with nvcc first if absent or stale).  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if build_if_missing and (not os.path.exists(path) or _build.is_stale()):
        _build.build_library()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2412_14775_b200.build` (there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, sz, ci = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int
    lib.rfi_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ci]
    lib.rfi_plan_set_integration.argtypes = [vp, ci]
    lib.rfi_plan_set_baseline_shard.argtypes = [vp, ci, ci]
    lib.rfi_plan_set_window_freq.argtypes = [vp, ci]
    lib.rfi_plan_set_layout.argtypes = [vp, ci]
    lib.rfi_plan_set_layout.restype = ci
    lib.rfi_plan_set_baseline_classes.argtypes = [vp, ci, ctypes.c_char_p]
    lib.rfi_plan_set_baseline_classes.restype = ci
    lib.rfi_plan_set_arithmetic.argtypes = [vp, ci, ctypes.c_uint32]
    lib.rfi_set_thresholds.argtypes = [vp, ci, ctypes.POINTER(RfiThresholds)]
    lib.rfi_plan_set_variant.argtypes = [vp, ci]
    lib.rfi_plan_set_adaptive.argtypes = [vp, ctypes.c_float, ctypes.c_float]
    lib.rfi_plan_set_adaptive.restype = ci
    lib.rfi_plan_set_adaptive_limit.argtypes = [vp, ctypes.c_float]
    lib.rfi_plan_set_adaptive_limit.restype = ci
    lib.rfi_plan_set_adaptive_scope.argtypes = [vp, ci]
    lib.rfi_plan_set_adaptive_scope.restype = ci
    lib.rfi_plan_set_stream_thresholds.argtypes = [vp, ctypes.POINTER(RfiThresholds)]
    lib.rfi_plan_set_stream_thresholds.restype = ci
    lib.rfi_plan_get_stream_thresholds.argtypes = [vp, ctypes.POINTER(RfiThresholds)]
    lib.rfi_plan_get_stream_thresholds.restype = ci
    lib.rfi_plan_get_stream_histograms.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    lib.rfi_plan_get_stream_histograms.restype = ci
    lib.rfi_plan_get_thresholds.argtypes = [vp, ctypes.POINTER(RfiThresholds)]
    lib.rfi_plan_get_thresholds.restype = ci
    lib.rfi_plan_get_adaptive_histogram.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    lib.rfi_plan_get_adaptive_histogram.restype = ci
    lib.rfi_process_chunk.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.rfi_get_flags.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(sz)]
    lib.rfi_process_chunk_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.rfi_confusion_counts.argtypes = [vp, vp, vp, vp]
    lib.rfi_confusion_counts.restype = ci
    lib.rfi_plan_set_truth.argtypes = [vp, vp, vp]
    lib.rfi_plan_set_truth.restype = ci
    lib.rfi_plan_destroy.argtypes = [vp]
    lib.rfi_probe_read_bandwidth.argtypes = [vp, sz, ci, ctypes.POINTER(ctypes.c_float), vp]
    lib.rfi_probe_read_bandwidth.restype = ci
    lib.rfi_probe_mix_bandwidth.argtypes = [vp, sz, vp, sz, ci, ci, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(sz), vp]
    lib.rfi_probe_mix_bandwidth.restype = ci
    lib.rfi_rl_evaluate.argtypes = [vp, ctypes.c_int64, ci, ctypes.c_uint32, ctypes.POINTER(RfiThresholds), ctypes.c_double, vp, vp]
    lib.rfi_rl_evaluate_masks.argtypes = [vp, ctypes.c_int64, ci, vp, ctypes.POINTER(RfiThresholds), ctypes.c_double, vp, vp]
    lib.rfi_rl_evaluate_masks.restype = ci
    lib.rfi_rl_evaluate.restype = ci
    lib.rfi_sim42_generate.argtypes = [ctypes.POINTER(Sim42Config), vp, vp, vp, vp, vp]
    lib.rfi_sim42_generate.restype = ci
    lib.rfi_sim42_generate_static.argtypes = [ctypes.POINTER(Sim42Config), vp, vp, vp]
    lib.rfi_sim42_generate_static.restype = ci
    lib.rfi_sim42_static_bytes.argtypes = []
    lib.rfi_sim42_static_bytes.restype = sz
    for name in ("rfi_sim42_vis_bytes", "rfi_sim42_truth_bytes"):
        getattr(lib, name).argtypes = [ctypes.POINTER(Sim42Config)]
        getattr(lib, name).restype = sz
    for name in ("rfi_plan_create", "rfi_plan_set_integration", "rfi_plan_set_baseline_shard",
                 "rfi_plan_set_window_freq", "rfi_plan_set_arithmetic", "rfi_set_thresholds", "rfi_plan_set_variant",
                 "rfi_process_chunk", "rfi_get_flags", "rfi_confusion_counts", "rfi_process_chunk_host", "rfi_plan_destroy",
                 "rfi_plan_last_variant"):
        getattr(lib, name).restype = ci
    lib.rfi_strerror.argtypes = [ci]
    lib.rfi_strerror.restype = ctypes.c_char_p
    lib.rfi_last_cuda_error.argtypes = []
    lib.rfi_last_cuda_error.restype = ctypes.c_char_p
    lib.rfi_version.argtypes = []
    lib.rfi_version.restype = ctypes.c_char_p
    for name in ("rfi_flags_bytes", "rfi_avg_bytes", "rfi_weight_bytes", "rfi_stats_bytes", "rfi_vis_bytes"):
        getattr(lib, name).argtypes = [vp]
        getattr(lib, name).restype = sz
    lib.rfi_plan_launch_count.argtypes = [vp]
    lib.rfi_plan_launch_count.restype = ctypes.c_uint64
    lib.rfi_plan_last_variant.argtypes = [vp]
    _lib = lib
    return lib


def _check(code: int, where: str):
    if code != 0:
        raise RfiError(code, where)


class RfiPlan:
    """Python face of `rfi_plan` with the same call names as the C ABI."""

    def __init__(self, n_stations: int, n_baselines: int, n_chan: int, n_time: int, window_M: int,
                 precision: int = RFI_FP32, n_int: Optional[int] = None):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        _check(self._lib.rfi_plan_create(ctypes.byref(self._h), n_stations, n_baselines, n_chan, n_time,
                                         window_M, precision), "rfi_plan_create")
        self.n_stations, self.n_baselines, self.n_chan = n_stations, n_baselines, n_chan
        self.n_time, self.window_M, self.precision = n_time, window_M, precision
        self.n_int = n_time
        self.K = 0
        self.b_first = 0
        self.window_F = 1
        self.n_classes = 1
        self._n_baselines_total = n_baselines
        if n_int is not None:
            self.set_integration(n_int)

    # ---- shape helpers -------------------------------------------------------------------------
    @property
    def n_cells(self): return self.n_baselines * self.n_chan
    @property
    def n_win(self): return self.n_time // self.window_M
    @property
    def n_out(self): return self.n_time // self.n_int
    @property
    def wpb(self): return (self.n_chan + 31) // 32

    # ---- C ABI ---------------------------------------------------------------------------------
    def set_integration(self, n_int: int):
        _check(self._lib.rfi_plan_set_integration(self._h, n_int), "rfi_plan_set_integration")
        self.n_int = n_int

    def set_window_freq(self, F: int):
        """rfi_plan_set_window_freq: T x F footprints, W = window_M * F."""
        _check(self._lib.rfi_plan_set_window_freq(self._h, F), "rfi_plan_set_window_freq")
        self.window_F = F

    def set_layout(self, layout):
        """rfi_plan_set_layout: "time_major" (vis[t][b][c][pol], default) or "cell_major" (vis[b][c][t][pol])."""
        v = {"time_major": 0, "cell_major": 1}[layout] if isinstance(layout, str) else int(layout)
        _check(self._lib.rfi_plan_set_layout(self._h, v), "rfi_plan_set_layout")

    def set_arithmetic(self, mode, mask14: int = 0):
        """rfi_plan_set_arithmetic: "fast" (default) or "tables" (paper-literal Tables 1-2 with a 14-bit half-precision mask)."""
        m = {"fast": ARITH_FAST, "tables": ARITH_TABLES}[mode] if isinstance(mode, str) else int(mode)
        _check(self._lib.rfi_plan_set_arithmetic(self._h, m, mask14), "rfi_plan_set_arithmetic")

    def set_baseline_shard(self, b_first: int, b_count: int):
        """rfi_plan_set_baseline_shard: this plan processes baselines [b_first, b_first + b_count) only."""
        _check(self._lib.rfi_plan_set_baseline_shard(self._h, b_first, b_count), "rfi_plan_set_baseline_shard")
        self.b_first, self.n_baselines = b_first, b_count

    def set_baseline_classes(self, classes: Optional[Sequence[int]]):
        """rfi_plan_set_baseline_classes: classes[b] in {0, 1} for every baseline of the array (None: one class).
        Thresholds must be set again afterwards; with two classes set_thresholds takes [[set_class0, set_class1], ...]."""
        if classes is None:
            _check(self._lib.rfi_plan_set_baseline_classes(self._h, 1, None), "rfi_plan_set_baseline_classes")
            self.n_classes = 1
        else:
            buf = bytes(bytearray(int(c) for c in classes))
            if len(buf) != self._n_baselines_total:
                raise ValueError("classes must have one entry per baseline of the array")
            _check(self._lib.rfi_plan_set_baseline_classes(self._h, 2, buf), "rfi_plan_set_baseline_classes")
            self.n_classes = 2
        self.K = 0

    def set_thresholds(self, sets):
        """K sets (d, s_low, s_high, gamma); with two baseline classes K pairs [[class 0 set, class 1 set], ...]."""
        if self.n_classes == 2:
            flat = [s for pair in sets for s in pair]
            if len(flat) != 2 * len(sets):
                raise ValueError("with two baseline classes every entry must be a pair of sets")
        else:
            flat = list(sets)
        arr = (RfiThresholds * len(flat))(*[RfiThresholds(*map(float, s)) for s in flat])
        _check(self._lib.rfi_set_thresholds(self._h, len(sets), arr), "rfi_set_thresholds")
        self.K = len(sets)

    def set_adaptive(self, false_alarm: float, forget: float = 0.0):
        """rfi_plan_set_adaptive: hold `false_alarm` on RFI-free data by tracking the null quantiles of both statistics
        per baseline class, chunk by chunk, on the device (0 switches it off)."""
        _check(self._lib.rfi_plan_set_adaptive(self._h, float(false_alarm), float(forget)), "rfi_plan_set_adaptive")

    def set_adaptive_limit(self, max_loosen: Optional[float]):
        """rfi_plan_set_adaptive_limit: an update may loosen a threshold by at most max_loosen * |a-priori value|
        (None or a negative value: no bound).  Keeps the adaptation from drifting into the RFI when a stream's RFI
        occupancy exceeds the requested false-alarm rate."""
        _check(self._lib.rfi_plan_set_adaptive_limit(self._h, -1.0 if max_loosen is None else float(max_loosen)),
               "rfi_plan_set_adaptive_limit")

    def set_adaptive_scope(self, scope: str):
        """rfi_plan_set_adaptive_scope: "class" (one threshold set per baseline class) or "baseline" (every baseline
        stream adapts its own thresholds: the paper's "fine-tuning for each data stream")."""
        _check(self._lib.rfi_plan_set_adaptive_scope(self._h, {"class": 0, "baseline": 1}[scope]), "rfi_plan_set_adaptive_scope")

    def set_stream_thresholds(self, sets):
        """rfi_plan_set_stream_thresholds: sets[b] = (d, s_low, s_high, gamma) for every baseline of the plan's shard
        (None switches the table off).  K must be 1."""
        if sets is None:
            _check(self._lib.rfi_plan_set_stream_thresholds(self._h, None), "rfi_plan_set_stream_thresholds")
            return
        if len(sets) != self.n_baselines:
            raise ValueError("one threshold set per baseline of the plan is needed")
        arr = (RfiThresholds * self.n_baselines)(*[RfiThresholds(*map(float, t)) for t in sets])
        _check(self._lib.rfi_plan_set_stream_thresholds(self._h, arr), "rfi_plan_set_stream_thresholds")

    def get_stream_thresholds(self):
        """rfi_plan_get_stream_thresholds: float64 array [n_baselines, 4] = (d, s_low, s_high, gamma) per baseline stream."""
        import numpy as np
        arr = (RfiThresholds * self.n_baselines)()
        _check(self._lib.rfi_plan_get_stream_thresholds(self._h, arr), "rfi_plan_get_stream_thresholds")
        return np.array([(t.d, t.s_low, t.s_high, t.gamma) for t in arr], dtype=np.float64)

    def get_stream_histograms(self):
        """rfi_plan_get_stream_histograms: float64 array [n_baselines, 1152] (768 tau bins | 384 r bins), running counts."""
        import numpy as np
        buf = np.empty((self.n_baselines, 1152), dtype=np.float64)
        _check(self._lib.rfi_plan_get_stream_histograms(self._h, buf.ctypes.data_as(ctypes.POINTER(ctypes.c_double))),
               "rfi_plan_get_stream_histograms")
        return buf

    def get_thresholds(self):
        """rfi_plan_get_thresholds: [(d, s_low, s_high, gamma)] per baseline class, as currently in force."""
        arr = (RfiThresholds * self.n_classes)()
        _check(self._lib.rfi_plan_get_thresholds(self._h, arr), "rfi_plan_get_thresholds")
        return [(t.d, t.s_low, t.s_high, t.gamma) for t in arr]

    def get_adaptive_histogram(self):
        """rfi_plan_get_adaptive_histogram: list over the two classes of (tau histogram [768], r histogram [384]) as float64."""
        buf = (ctypes.c_double * (2 * 1152))()
        _check(self._lib.rfi_plan_get_adaptive_histogram(self._h, buf), "rfi_plan_get_adaptive_histogram")
        a = torch.tensor(list(buf), dtype=torch.float64).view(2, 1152)
        return [(a[c, :768].clone(), a[c, 768:].clone()) for c in range(2)]

    def set_variant(self, variant):
        v = _VARIANTS[variant] if isinstance(variant, str) else int(variant)
        _check(self._lib.rfi_plan_set_variant(self._h, v), "rfi_plan_set_variant")

    def alloc_outputs(self, device="cuda", stats: bool = False):
        K = max(self.K, 1)
        avg = torch.empty(K, self.n_out, self.n_baselines, self.n_chan, 4, 2, dtype=torch.float32, device=device)
        weight = torch.empty(K, self.n_out, self.n_baselines, self.n_chan, dtype=torch.int32, device=device)
        st = torch.empty(3, self.n_win, self.n_baselines, self.n_chan, dtype=torch.float32, device=device) if stats else None
        return avg, weight, st

    def process_chunk(self, vis: torch.Tensor, avg: torch.Tensor, weight: torch.Tensor,
                      stats: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None):
        """rfi_process_chunk on torch device tensors (asynchronous on `stream`, default: torch's current stream)."""
        for t, name in ((vis, "vis"), (avg, "avg"), (weight, "weight")):
            if not (t.is_cuda and t.is_contiguous()):
                raise ValueError(f"{name} must be a contiguous CUDA tensor")
        if vis.numel() * vis.element_size() != self._lib.rfi_vis_bytes(self._h):
            raise ValueError("vis has the wrong size for this plan")
        if avg.numel() * 4 != self._lib.rfi_avg_bytes(self._h) or weight.numel() * 4 != self._lib.rfi_weight_bytes(self._h):
            raise ValueError("avg/weight have the wrong size for this plan (set thresholds before allocating)")
        if stats is not None and stats.numel() * 4 != self._lib.rfi_stats_bytes(self._h):
            raise ValueError("stats has the wrong size for this plan")
        s = stream if stream is not None else torch.cuda.current_stream(vis.device)
        self._device = vis.device                         # the plan's flag buffer lives on this device
        _check(self._lib.rfi_process_chunk(self._h, vis.data_ptr(), avg.data_ptr(), weight.data_ptr(),
                                           stats.data_ptr() if stats is not None else None, s.cuda_stream),
               "rfi_process_chunk")

    def get_flags(self) -> torch.Tensor:
        """uint32-as-int32 tensor [K, n_win, n_baselines, wpb] aliasing the plan's device flag buffer."""
        ptr, n = ctypes.c_void_p(), ctypes.c_size_t()
        _check(self._lib.rfi_get_flags(self._h, ctypes.byref(ptr), ctypes.byref(n)), "rfi_get_flags")
        shape = (max(self.K, 1), self.n_win, self.n_baselines, self.wpb)
        assert n.value == shape[0] * shape[1] * shape[2] * shape[3]
        iface = {"shape": (n.value,), "typestr": "<i4", "data": (ptr.value, False), "version": 2}
        holder = type("_FlagView", (), {"__cuda_array_interface__": iface})()
        return torch.as_tensor(holder, device=getattr(self, "_device", "cuda")).view(shape)

    def confusion_counts(self, truth_words: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        """rfi_confusion_counts: truth_words = pack_flags(bool truth) on the device; returns int64 [K, 4] on the device."""
        if not (truth_words.is_cuda and truth_words.is_contiguous() and truth_words.dtype == torch.int32):
            raise ValueError("truth_words must be a contiguous int32 CUDA tensor (pack_flags)")
        if truth_words.numel() != self.n_win * self.n_baselines * self.wpb:
            raise ValueError("truth_words has the wrong size for this plan")
        counts = torch.empty(max(self.K, 1), 4, dtype=torch.int64, device=truth_words.device)
        s = stream if stream is not None else torch.cuda.current_stream(truth_words.device)
        _check(self._lib.rfi_confusion_counts(self._h, truth_words.data_ptr(), counts.data_ptr(), s.cuda_stream),
               "rfi_confusion_counts")
        return counts

    def set_truth(self, truth_words: Optional[torch.Tensor]) -> Optional[torch.Tensor]:
        """rfi_plan_set_truth: every following process_chunk also fills int64 counts[K, 4] = {false alarms, clean windows,
        missed detections, RFI windows} against truth_words (= pack_flags(bool truth) on the device); the K-set kernel
        counts in the same launch.  Returns the counts tensor (refilled by every call); None switches it off."""
        if truth_words is None:
            _check(self._lib.rfi_plan_set_truth(self._h, None, None), "rfi_plan_set_truth")
            self._truth = self._counts = None
            return None
        if not (truth_words.is_cuda and truth_words.is_contiguous() and truth_words.dtype == torch.int32):
            raise ValueError("truth_words must be a contiguous int32 CUDA tensor (pack_flags)")
        if truth_words.numel() != self.n_win * self.n_baselines * self.wpb:
            raise ValueError("truth_words has the wrong size for this plan")
        counts = torch.zeros(max(self.K, 1), 4, dtype=torch.int64, device=truth_words.device)
        _check(self._lib.rfi_plan_set_truth(self._h, truth_words.data_ptr(), counts.data_ptr()), "rfi_plan_set_truth")
        self._truth, self._counts = truth_words, counts                      # keep both alive
        return counts

    def process_chunk_host(self, vis: torch.Tensor, want_stats: bool = False):
        """rfi_process_chunk_host: vis is a (preferably pinned) CPU tensor; returns CPU tensors."""
        if vis.is_cuda or not vis.is_contiguous():
            raise ValueError("vis must be a contiguous CPU tensor")
        K = max(self.K, 1)
        pin = torch.cuda.is_available()
        avg = torch.empty(K, self.n_out, self.n_baselines, self.n_chan, 4, 2, dtype=torch.float32, pin_memory=pin)
        weight = torch.empty(K, self.n_out, self.n_baselines, self.n_chan, dtype=torch.int32, pin_memory=pin)
        flags = torch.empty(K, self.n_win, self.n_baselines, self.wpb, dtype=torch.int32, pin_memory=pin)
        stats = torch.empty(3, self.n_win, self.n_baselines, self.n_chan, dtype=torch.float32, pin_memory=pin) if want_stats else None
        self.process_chunk_host_into(vis, avg, weight, flags, stats)
        return avg, weight, flags, stats

    def process_chunk_host_into(self, vis, avg, weight, flags, stats=None):
        _check(self._lib.rfi_process_chunk_host(self._h, vis.data_ptr(), avg.data_ptr(), weight.data_ptr(),
                                                flags.data_ptr(), stats.data_ptr() if stats is not None else None),
               "rfi_process_chunk_host")

    @property
    def launch_count(self) -> int:
        return int(self._lib.rfi_plan_launch_count(self._h))

    @property
    def last_variant(self) -> str:
        v = self._lib.rfi_plan_last_variant(self._h)
        return {0: "none", 1: "direct", 2: "tma", 3: "batched", 4: "tables", 5: "split"}.get(v, str(v))

    def destroy(self):
        if self._h:
            self._lib.rfi_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


RL_RECORD_DOUBLES = 52
RL_FIELDS = {"features": slice(0, 10), "bits": slice(10, 24), "errors": slice(24, 45), "op_cost": 45, "conversions": 46,
             "overflow": 47, "underflow": 48, "matches": 49, "reward": 50, "flags": 51}


def rl_evaluate(windows: torch.Tensor, mask14: int, threshold, reward_per_match: float = 3.0,
                out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """rfi_rl_evaluate: the RL environment of PAPER.md:149-172 for a batch of windows and one precision mask -- or, with
    mask14 a CUDA int16 tensor [n], one mask per window (rfi_rl_evaluate_masks: a batch of (state, action) pairs).
    windows: contiguous CUDA float32 [n, W, 4, 2]; returns float64 [n, 52] (layout RL_FIELDS / include/rfi.h)."""
    if not (windows.is_cuda and windows.is_contiguous() and windows.dtype == torch.float32 and windows.dim() == 4
            and tuple(windows.shape[2:]) == (4, 2)):
        raise ValueError("windows must be a contiguous CUDA float32 tensor [n, W, 4, 2]")
    n, W = windows.shape[0], windows.shape[1]
    rec = out if out is not None else torch.empty(n, RL_RECORD_DOUBLES, dtype=torch.float64, device=windows.device)
    thr = RfiThresholds(*map(float, threshold))
    if isinstance(mask14, torch.Tensor):
        if not (mask14.is_cuda and mask14.is_contiguous() and mask14.dtype == torch.int16 and mask14.numel() == n):
            raise ValueError("per-window masks must be a contiguous CUDA int16 tensor [n]")
        with torch.cuda.device(windows.device):
            _check(load_library().rfi_rl_evaluate_masks(windows.data_ptr(), n, W, mask14.data_ptr(), ctypes.byref(thr),
                                                        float(reward_per_match), rec.data_ptr(),
                                                        torch.cuda.current_stream(windows.device).cuda_stream),
                   "rfi_rl_evaluate_masks")
        return rec
    with torch.cuda.device(windows.device):
        _check(load_library().rfi_rl_evaluate(windows.data_ptr(), n, W, int(mask14), ctypes.byref(thr), float(reward_per_match),
                                              rec.data_ptr(), torch.cuda.current_stream(windows.device).cuda_stream),
               "rfi_rl_evaluate")
    return rec


def sim42_generate(n_real: int, inr: float, seed: int = 1, n_time: int = 2000, n_chan: int = 512, n_sources: int = 200,
                   n_broadband: int = 5, n_narrowband: int = 1, n_narrowdur: int = 1, polarized: bool = True,
                   window_T: int = 10, window_F: int = 2, device="cuda", out: Optional[torch.Tensor] = None,
                   diagnostics: bool = False):
    """rfi_sim42_generate: the paper's section-4.2 simulator on the device.
    Returns (vis [n_time, n_real, n_chan, 4, 2] float32, truth_words [n_time/window_T, n_real, ceil(n_chan/32)] int32)
    and, with diagnostics=True, also the parameter table (list of Sim42Realisation) and the source coherence
    [n_real, n_chan, 2] float64.  Argument marshalling only: every number is drawn and computed by the CUDA kernels."""
    lib = load_library()
    cfg = Sim42Config(n_time, n_chan, n_real, n_sources, n_broadband, n_narrowband, n_narrowdur, 1 if polarized else 0,
                      float(inr), window_T, window_F, seed)
    dev = torch.device(device)
    vis = out if out is not None else torch.empty(n_time, n_real, n_chan, 4, 2, dtype=torch.float32, device=dev)
    if not (vis.is_cuda and vis.is_contiguous() and vis.numel() * 4 == lib.rfi_sim42_vis_bytes(ctypes.byref(cfg))):
        raise ValueError("out must be a contiguous CUDA float32 tensor of n_time * n_real * n_chan * 8 elements")
    truth = torch.empty(n_time // window_T, n_real, (n_chan + 31) // 32, dtype=torch.int32, device=vis.device)
    table = torch.empty(n_real * ctypes.sizeof(Sim42Realisation), dtype=torch.uint8, device=vis.device) if diagnostics else None
    src = torch.empty(n_real, n_chan, 2, dtype=torch.float64, device=vis.device) if diagnostics else None
    with torch.cuda.device(vis.device):
        _check(lib.rfi_sim42_generate(ctypes.byref(cfg), vis.data_ptr(), truth.data_ptr(),
                                      table.data_ptr() if diagnostics else None, src.data_ptr() if diagnostics else None,
                                      torch.cuda.current_stream(vis.device).cuda_stream), "rfi_sim42_generate")
    if not diagnostics:
        return vis, truth
    raw = table.cpu().numpy().tobytes()
    n = ctypes.sizeof(Sim42Realisation)
    tab = [Sim42Realisation.from_buffer_copy(raw[i * n:(i + 1) * n]) for i in range(n_real)]
    return vis, truth, tab, src


SIM42_STATIC_MAX_REAL = 512
SIM42_STATIC_MAX_CELLS = 262144


def sim42_generate_static(vis: torch.Tensor, truth: Optional[torch.Tensor], inr: float, seed: int = 1, n_sources: int = 200,
                          n_broadband: int = 5, n_narrowband: int = 1, n_narrowdur: int = 1, polarized: bool = True,
                          window_T: int = 10, window_F: int = 2) -> None:
    """rfi_sim42_generate_static: the section-4.2 generator for callers that may not allocate device memory (a plug-in
    inside a process that has handed the whole GPU to its own pool, a loop running beside live streams that a
    cudaMalloc / cudaFree would stall).  Its work arrays sit in a fixed array inside librfi.so, so the call allocates
    nothing -- and neither does this wrapper: the caller brings both outputs.
      vis    [n_time, n_real, n_chan, 4, 2] float32, contiguous, CUDA: filled in place
      truth  [n_time // window_T, n_real, ceil(n_chan / 32)] int32, contiguous, same device; or None
    Limits: n_real <= SIM42_STATIC_MAX_REAL, n_real * n_chan <= SIM42_STATIC_MAX_CELLS (RfiError otherwise).  Calls on
    one device share the array: keep them ordered on one stream.  Runs on vis's current stream; asynchronous."""
    if not (vis.is_cuda and vis.is_contiguous() and vis.dtype == torch.float32 and vis.dim() == 5 and vis.shape[3:] == (4, 2)):
        raise ValueError("vis must be a contiguous CUDA float32 tensor [n_time, n_real, n_chan, 4, 2]")
    n_time, n_real, n_chan = int(vis.shape[0]), int(vis.shape[1]), int(vis.shape[2])
    if truth is not None and not (truth.is_cuda and truth.device == vis.device and truth.is_contiguous() and truth.dtype == torch.int32
                                  and window_T > 0 and tuple(truth.shape) == (n_time // window_T, n_real, (n_chan + 31) // 32)):
        raise ValueError("truth must be a contiguous int32 tensor [n_time // window_T, n_real, ceil(n_chan / 32)] on vis's device")
    lib = load_library()
    cfg = Sim42Config(n_time, n_chan, n_real, n_sources, n_broadband, n_narrowband, n_narrowdur, 1 if polarized else 0,
                      float(inr), window_T, window_F, seed)
    with torch.cuda.device(vis.device):
        _check(lib.rfi_sim42_generate_static(ctypes.byref(cfg), vis.data_ptr(), truth.data_ptr() if truth is not None else None,
                                             torch.cuda.current_stream(vis.device).cuda_stream), "rfi_sim42_generate_static")


def probe_read_bandwidth(buf: torch.Tensor, repeats: int = 10) -> float:
    """rfi_probe_read_bandwidth: read-only streaming GB/s of buf's device (diagnostics; the denominator that suits a
    one-touch read stream).  buf: contiguous CUDA tensor, 32-byte aligned."""
    if not (buf.is_cuda and buf.is_contiguous()):
        raise ValueError("buf must be a contiguous CUDA tensor")
    lib = load_library()
    ms = ctypes.c_float()
    nbytes = buf.numel() * buf.element_size()
    with torch.cuda.device(buf.device):
        _check(lib.rfi_probe_read_bandwidth(buf.data_ptr(), nbytes, repeats, ctypes.byref(ms),
                                            torch.cuda.current_stream(buf.device).cuda_stream), "rfi_probe_read_bandwidth")
    return (nbytes // 32 * 32) / (ms.value * 1e-3) / 1e9


def probe_mix_bandwidth(buf: torch.Tensor, out_bytes: int, repeats: int = 10) -> float:
    """rfi_probe_mix_bandwidth: GB/s (read + written) of a zero-arithmetic stream that reads buf and writes about
    out_bytes, 1 KiB row per `reads_per_write` rows read -- the ceiling for a K-set pass with that output volume.
    buf: contiguous CUDA tensor, 32-byte aligned."""
    if not (buf.is_cuda and buf.is_contiguous()):
        raise ValueError("buf must be a contiguous CUDA tensor")
    lib = load_library()
    nbytes = buf.numel() * buf.element_size()
    rpw = max(1, round(nbytes / max(out_bytes, 1)))
    out = torch.empty(nbytes // (rpw * 1024) * 1024 + 1024, dtype=torch.uint8, device=buf.device)
    ms, moved = ctypes.c_float(), ctypes.c_size_t()
    with torch.cuda.device(buf.device):
        _check(lib.rfi_probe_mix_bandwidth(buf.data_ptr(), nbytes, out.data_ptr(), out.numel(), rpw, repeats, ctypes.byref(ms),
                                           ctypes.byref(moved), torch.cuda.current_stream(buf.device).cuda_stream),
               "rfi_probe_mix_bandwidth")
    return moved.value / (ms.value * 1e-3) / 1e9


def unpack_flags(flags: torch.Tensor, n_chan: int) -> torch.Tensor:
    """[.., n_baselines, wpb] int32 words -> bool [.., n_baselines, n_chan] (layout of include/rfi.h)."""
    bits = torch.arange(32, device=flags.device, dtype=torch.int32)
    b = ((flags.unsqueeze(-1) >> bits) & 1).bool()
    return b.flatten(-2)[..., :n_chan]


def pack_flags(mask: torch.Tensor) -> torch.Tensor:
    """bool [.., n_baselines, n_chan] -> int32 words [.., n_baselines, ceil(n_chan/32)] (inverse of unpack_flags)."""
    n_chan = mask.shape[-1]
    wpb = (n_chan + 31) // 32
    pad = wpb * 32 - n_chan
    m = torch.nn.functional.pad(mask.to(torch.int64), (0, pad)).reshape(*mask.shape[:-1], wpb, 32)
    w = (m << torch.arange(32, device=mask.device, dtype=torch.int64)).sum(-1)
    return torch.where(w >= 2 ** 31, w - 2 ** 32, w).to(torch.int32)
