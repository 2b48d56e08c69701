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

// Rows merged per block by the register-staged kernels (direct and batched): a divisor of the window length T.
// fp16: the largest divisor <= 8 (16 B rows, 4 CTAs of 4 warps per SM).  fp32: rows are 32 B = 8 registers per
// buffered row, so R <= 4 runs 4 CTAs/SM (16 warps), R = 5 three (12 warps), R = 6..8 two (8 warps); pick the divisor
// with the most bytes in flight per SM, R * warps(R), smaller R on ties.  T = 16 -> 4, T = 10 -> 5, T = 5 -> 5,
// T = 7 -> 7, T = 6 -> 3.  `cap` bounds R (the batched kernels are instantiated up to 4 / 8 only);
// RFI_DIRECT_ROWS lowers it further.
inline int direct_warps_per_sm(int R, bool fp16) { return (fp16 || R <= 4) ? 16 : (R == 5 ? 12 : 8); }
inline int pick_rows(int M, bool fp16, int cap = 8) {
    const int max_r = fp16 ? 8 : 8;
    int lim = env_int("RFI_DIRECT_ROWS", max_r);
    if (lim < 1) lim = 1;
    if (lim > max_r) lim = max_r;
    if (lim > cap) lim = cap;
    int best = 1, best_score = 0;
    for (int r = 1; r <= lim; ++r) {
        if (M % r) continue;
        const int score = r * direct_warps_per_sm(r, fp16);
        if (score > best_score) { best = r; best_score = score; }
    }
    return best;
}

// Each returns RFI_OK or RFI_ECUDA / RFI_EINVAL; all only enqueue work on `st`.
int launch_direct(bool fp16, const rfi::KParams& kp, cudaStream_t st);
int launch_split(bool fp16, const rfi::KParams& kp, int smem_optin, cudaStream_t st);   // small chunks, low latency
int launch_tma(bool fp16, const rfi::KParams& kp, const CUtensorMap* map, int R, int sm_count, int smem_optin,
               cudaStream_t st);
int launch_tma_cellmajor(bool fp16, const rfi::KParams& kp, const CUtensorMap* map, int sm_count, int smem_optin,
                         cudaStream_t st);
int tma_rows(int M);                                   // rows per TMA stage for window length M
int launch_batched(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, cudaStream_t st);
int launch_tables(const rfi::KParams& kp, cudaStream_t st);
int launch_tables_ps(const rfi::KParams& kp, cudaStream_t st);          // R = 4, per-sample groups compile-time (256 variants)

int launch_batched_tma_cellmajor(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map,
                                 int sm_count, int smem_optin, cudaStream_t st);
int launch_adapt_update(uint32_t* d_hist, double* d_acc, rfi::Thr* d_thr, rfi_thresholds* d_raw, const rfi_thresholds* d_prior,
                        double max_loosen, int n_classes, double alpha, double forget, cudaStream_t st);
int launch_confusion(const uint32_t* d_flags, const uint32_t* d_truth, uint64_t* d_counts, int K, size_t n_words,
                     int wpb, int n_chan, int sm_count, cudaStream_t st);
bool batched_tma_supported(bool fp16, const rfi::KParams& kp, int R);

int launch_batched_tma(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int R,
                       int sm_count, int smem_optin, cudaStream_t st);

// second-generation batched kernel (rfi_batched_mask.cuh): whole-word tiles only (n_chan % 32 == 0)
int launch_batched_mask_f32(const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int R, bool cell_major,
                            int sm_count, int smem_optin, cudaStream_t st);
int launch_batched_mask_f16(const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int R, bool cell_major,
                            int sm_count, int smem_optin, cudaStream_t st);
inline bool batched_mask_supported(const rfi::KParams& kp) {
    return kp.n_chan % 32 == 0 && env_int("RFI_BT_MASK", 1) != 0;
}
inline bool batched_mask_rows(bool fp16, int R) {          // block lengths it is instantiated for
    return fp16 ? (R == 8 || R == 5 || R == 4 || R == 2) : (R == 5 || R == 4 || R == 2);
}

}  // namespace rfi_host
