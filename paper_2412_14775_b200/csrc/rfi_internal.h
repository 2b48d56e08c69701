// rfi_internal.h -- host-side declarations shared by the translation units of librfi.so (not installed).
#pragma once

#include "../../include/rfi.h"

#include <cstdio>
#include <cstdlib>

#include "rfi_common.cuh"

namespace rfi_host {

extern thread_local char g_cuda_err[512];

inline bool cuda_ok(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
    return false;
}
#define RFI_CUDA(call)                                            \
    do {                                                          \
        if (!rfi_host::cuda_ok((call), #call)) return RFI_ECUDA;  \
    } while (0)

inline int env_int(const char* name, int dflt) {
    const char* s = getenv(name);
    return (s && *s) ? atoi(s) : dflt;
}

inline int largest_divisor_le(int M, int cap) {
    for (int r = cap; r >= 1; --r)
        if (M % r == 0) return r;
    return 1;
}

// Rows merged per block by the register-staged kernels (direct and batched): the largest divisor of the
// window length that keeps 128 B per thread in flight (4 rows fp32, 8 rows fp16); RFI_DIRECT_ROWS lowers the cap.
inline int pick_rows(int M, bool fp16) {
    const int max_r = fp16 ? 8 : 4;
    int cap = env_int("RFI_DIRECT_ROWS", max_r);
    if (cap < 1) cap = 1;
    if (cap > max_r) cap = max_r;
    return largest_divisor_le(M, cap);
}

// Each returns RFI_OK or RFI_ECUDA / RFI_EINVAL; all only enqueue work on `st`.
int launch_direct(bool fp16, const rfi::KParams& kp, cudaStream_t st);
int launch_tma(bool fp16, const rfi::KParams& kp, const CUtensorMap* map, int R, int sm_count, int smem_optin,
               cudaStream_t st);
int tma_rows(int M);                                   // rows per TMA stage for window length M
int launch_batched(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, cudaStream_t st);
bool batched_tma_supported(bool fp16, const rfi::KParams& kp, int R);
int launch_batched_tma(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int R,
                       int sm_count, int smem_optin, cudaStream_t st);

}  // namespace rfi_host
