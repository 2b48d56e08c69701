// rfi_launch_split.cu -- instantiations and launcher of the small-chunk low-latency kernel (rfi_split.cuh).
#include "rfi_internal.h"
#include "rfi_split.cuh"

namespace rfi_host {
namespace {

template <int R, bool FP16>
int launch_r(const rfi::KParams& kp, int smem_optin, cudaStream_t st) {
    const int nb = kp.n_int / R;
    const size_t smem = ((size_t)nb * rfi::kSplitPartFloats + (size_t)kp.wpo * rfi::kSplitRecFloats) * 32 * sizeof(float);
    if (nb > rfi::kSplitMaxBlocks) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "RFI_VARIANT_SPLIT is for small chunks: n_int / %d = %d blocks per unit exceed %d "
                 "(use RFI_VARIANT_AUTO)", R, nb, rfi::kSplitMaxBlocks);
        return RFI_EINVAL;
    }
    if ((long)smem > smem_optin) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "RFI_VARIANT_SPLIT is for small chunks: %d blocks and %d windows per unit need %zu bytes of "
                 "shared memory, the device offers %d (use RFI_VARIANT_AUTO)", nb, kp.wpo, smem, smem_optin);
        return RFI_EINVAL;
    }
    const int n_tiles = (kp.n_cells + 31) / 32;
    const unsigned grid = (unsigned)((long)n_tiles * kp.n_out_slab);
    int warps = nb < kp.wpo ? kp.wpo : nb;
    if (warps > 16) warps = 16;
    const bool a32 = FP16 || (reinterpret_cast<uintptr_t>(kp.vis) % 32 == 0);
    if (a32) {
        auto kern = rfi::rfi_split_kernel<R, FP16, true>;
        RFI_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<grid, warps * 32, smem, st>>>(kp);
    } else {
        auto kern = rfi::rfi_split_kernel<R, FP16, false>;
        RFI_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<grid, warps * 32, smem, st>>>(kp);
    }
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

template <bool FP16>
int launch_f(const rfi::KParams& kp, int R, int smem_optin, cudaStream_t st) {
    switch (R) {
        case 1: return launch_r<1, FP16>(kp, smem_optin, st);
        case 2: return launch_r<2, FP16>(kp, smem_optin, st);
        case 3: return launch_r<3, FP16>(kp, smem_optin, st);
        case 4: return launch_r<4, FP16>(kp, smem_optin, st);
        case 5: return launch_r<5, FP16>(kp, smem_optin, st);
        case 6: return launch_r<6, FP16>(kp, smem_optin, st);
        case 7: return launch_r<7, FP16>(kp, smem_optin, st);
        default: return launch_r<8, FP16>(kp, smem_optin, st);
    }
}

}  // namespace

int launch_split(bool fp16, const rfi::KParams& kp, int smem_optin, cudaStream_t st) {
    const int R = pick_rows(kp.M, fp16);                      // the direct kernel's block length: same block statistics
    return fp16 ? launch_f<true>(kp, R, smem_optin, st) : launch_f<false>(kp, R, smem_optin, st);
}

}  // namespace rfi_host
