// rfi_launch_batched_tma.cu -- instantiations and launcher of the TMA-staged batched-threshold kernel.
#include "rfi_internal.h"
#include "rfi_batched_tma.cuh"

namespace rfi_host {
namespace {

template <int R, bool FP16, int SPW, bool CM = false>
int launch_rs(const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int sm_count, int smem_optin,
              cudaStream_t st) {
    constexpr int NW = rfi::kBtWarps;
    const int row_bytes = FP16 ? 512 : 1024;
    const int stage_bytes = CM ? 4096 : R * row_bytes;
    const int rec_bytes = 2 * NW * 32 * rfi::kRecBytes;
    const int budget = smem_optin - 1024 - rec_bytes - 256;
    int stages = env_int("RFI_BT_STAGES", 0);
    if (stages <= 0) stages = 8;
    while (stages > 1 && NW * stages * (stage_bytes + 16) > budget) --stages;
    if (NW * stages * (stage_bytes + 16) > budget) return RFI_EINVAL;
    const size_t smem = (size_t)NW * stages * (stage_bytes + 16) + rec_bytes + 1024;
    const int n_tiles = (kp.n_cells + 31) / 32;
    const long n_units = (long)n_tiles * kp.n_out_slab;
    long grid = n_units < sm_count ? n_units : sm_count;
    // whole 32-channel flag words (one word per tile, no invalid lane) take the ballot-per-round store;
    // anything else the generic per-word store
    if (kp.n_chan % 32 == 0) {
        auto kern = rfi::rfi_batched_tma_kernel<R, FP16, SPW, true, CM>;
        RFI_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<(unsigned)grid, NW * 32, smem, st>>>(*map, kp, bt, stages);
    } else {
        auto kern = rfi::rfi_batched_tma_kernel<R, FP16, SPW, false, CM>;
        RFI_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<(unsigned)grid, NW * 32, smem, st>>>(*map, kp, bt, stages);
    }
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

template <int R, bool FP16, bool CM = false>
int launch_r(const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int sm_count, int smem_optin,
             cudaStream_t st) {
    // sets per warp: 16 warps x {1, 2, 4} covers K <= 16, 32, 64
    if (kp.K <= rfi::kBtWarps) return launch_rs<R, FP16, 1, CM>(kp, bt, map, sm_count, smem_optin, st);
    if (kp.K <= 2 * rfi::kBtWarps) return launch_rs<R, FP16, 2, CM>(kp, bt, map, sm_count, smem_optin, st);
    return launch_rs<R, FP16, 4, CM>(kp, bt, map, sm_count, smem_optin, st);
}

}  // namespace

// Shapes the TMA-staged batched kernel covers: a block length it is instantiated for (and, checked by the caller,
// a cell count the tensor map can describe).  Everything else runs the register-staged batched kernel.
bool batched_tma_supported(bool fp16, const rfi::KParams& kp, int R) {
    if (env_int("RFI_BATCHED_TMA", 1) == 0) return false;
    return fp16 ? (R == 8 || R == 4 || R == 2) : (R == 4 || R == 2);
}

// Cell-major input: R = samples per 128-byte line (4 fp32 / 8 fp16), transposing tensor map.
int launch_batched_tma_cellmajor(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map,
                                 int sm_count, int smem_optin, cudaStream_t st) {
    if (kp.K < 1 || kp.K > rfi::kMaxBatch) return RFI_EINVAL;
    return fp16 ? launch_r<8, true, true>(kp, bt, map, sm_count, smem_optin, st)
                : launch_r<4, false, true>(kp, bt, map, sm_count, smem_optin, st);
}

int launch_batched_tma(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, const CUtensorMap* map, int R,
                       int sm_count, int smem_optin, cudaStream_t st) {
    if (kp.K < 1 || kp.K > rfi::kMaxBatch) return RFI_EINVAL;
    if (!fp16) {
        if (R == 4) return launch_r<4, false>(kp, bt, map, sm_count, smem_optin, st);
        if (R == 2) return launch_r<2, false>(kp, bt, map, sm_count, smem_optin, st);
        return RFI_EINVAL;
    }
    if (R == 8) return launch_r<8, true>(kp, bt, map, sm_count, smem_optin, st);
    if (R == 4) return launch_r<4, true>(kp, bt, map, sm_count, smem_optin, st);
    if (R == 2) return launch_r<2, true>(kp, bt, map, sm_count, smem_optin, st);
    return RFI_EINVAL;
}

}  // namespace rfi_host
