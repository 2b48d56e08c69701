// rfi_launch_tma.cu -- instantiations and launcher of the TMA (cp.async.bulk.tensor) single-set kernel.
#include "rfi_internal.h"
#include "rfi_kernels.cuh"

namespace rfi_host {
namespace {

template <int R, bool FP16, bool CM = false>
int launch_r(const rfi::KParams& kp, const CUtensorMap* map, int sm_count, int smem_optin, cudaStream_t st) {
    const int row_bytes = FP16 ? 512 : 1024;
    const int stage_bytes = CM ? 4096 : R * row_bytes;
    int warps = env_int("RFI_TMA_WARPS", 16);
    int stages = env_int("RFI_TMA_STAGES", 0);
    if (warps < 1) warps = 1;
    if (warps > 16) warps = 16;
    const int budget = smem_optin - 1024 - 256;
    if (stages <= 0) {
        stages = budget / (warps * (stage_bytes + 16));
        if (stages > 6) stages = 6;
    }
    while (stages > 1 && warps * stages * (stage_bytes + 16) > budget) --stages;
    while (warps > 1 && warps * stages * (stage_bytes + 16) > budget) --warps;
    const size_t smem = (size_t)warps * stages * (stage_bytes + 16) + 1024;
    const int n_tiles = (kp.n_cells + 31) / 32;
    const long n_units = (long)n_tiles * kp.n_out_slab;
    long grid = (n_units + warps - 1) / warps;
    const int ctas_per_sm = env_int("RFI_TMA_CTAS_PER_SM", 1);
    if (grid > (long)sm_count * ctas_per_sm) grid = (long)sm_count * ctas_per_sm;
    auto kern = rfi::rfi_tma_kernel<R, FP16, CM>;
    RFI_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)grid, warps * 32, smem, st>>>(*map, kp, stages);
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

template <bool FP16>
int launch_f(const rfi::KParams& kp, const CUtensorMap* map, int R, int sm_count, int smem_optin, cudaStream_t st) {
    switch (R) {
        case 1: return launch_r<1, FP16>(kp, map, sm_count, smem_optin, st);
        case 2: return launch_r<2, FP16>(kp, map, sm_count, smem_optin, st);
        case 3: return launch_r<3, FP16>(kp, map, sm_count, smem_optin, st);
        case 4: return launch_r<4, FP16>(kp, map, sm_count, smem_optin, st);
        case 5: return launch_r<5, FP16>(kp, map, sm_count, smem_optin, st);
        case 6: return launch_r<6, FP16>(kp, map, sm_count, smem_optin, st);
        case 7: return launch_r<7, FP16>(kp, map, sm_count, smem_optin, st);
        default: return launch_r<8, FP16>(kp, map, sm_count, smem_optin, st);
    }
}

}  // namespace

// Cell-major input (vis[b][c][t][pol]): the same kernel behind a transposing tensor map; R = samples per 128-byte line.
int launch_tma_cellmajor(bool fp16, const rfi::KParams& kp, const CUtensorMap* map, int sm_count, int smem_optin,
                         cudaStream_t st) {
    return fp16 ? launch_r<8, true, true>(kp, map, sm_count, smem_optin, st)
                : launch_r<4, false, true>(kp, map, sm_count, smem_optin, st);
}

int tma_rows(int M) {
    const int cap = env_int("RFI_TMA_ROWS", 8);
    return largest_divisor_le(M, cap < 1 ? 1 : (cap > 8 ? 8 : cap));
}

int launch_tma(bool fp16, const rfi::KParams& kp, const CUtensorMap* map, int R, int sm_count, int smem_optin,
               cudaStream_t st) {
    return fp16 ? launch_f<true>(kp, map, R, sm_count, smem_optin, st)
                : launch_f<false>(kp, map, R, sm_count, smem_optin, st);
}

}  // namespace rfi_host
