"""B200-native fused spectral-kurtosis + polarization-alignment flag-and-average pass (arxiv 2412.14775).

`RfiPlan` mirrors the C ABI of include/rfi.h (librfi.so, hand-written sm_100a CUDA); `synth` holds the
seeded input generators.  There is no CPU implementation in this package.
"""
from .binding import (RFI_FP16, RFI_FP32, RfiError, RfiPlan, load_library, library_path,  # noqa: F401
                      pack_flags, probe_mix_bandwidth, probe_read_bandwidth, rl_evaluate, sim42_generate, sim42_generate_static, unpack_flags)
from . import synth  # noqa: F401
