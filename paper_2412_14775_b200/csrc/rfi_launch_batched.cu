// rfi_launch_batched.cu -- instantiations and launcher of the batched-threshold kernel (K <= 64 sets per launch).
#include "rfi_internal.h"
#include "rfi_batched.cuh"

namespace rfi_host {
namespace {

template <int R, bool FP16, int SPW>
int launch_rs(const rfi::KParams& kp, const rfi::BatchThr& bt, cudaStream_t st) {
    const int n_tiles = (kp.n_cells + 31) / 32;
    const unsigned grid = (unsigned)((long)n_tiles * kp.n_out_slab);
    const bool a32 = FP16 || (reinterpret_cast<uintptr_t>(kp.vis) % 32 == 0);
    if (a32) rfi::rfi_batched_kernel<R, FP16, true, SPW><<<grid, rfi::kBatchWarps * 32, 0, st>>>(kp, bt);
    else     rfi::rfi_batched_kernel<R, FP16, false, SPW><<<grid, rfi::kBatchWarps * 32, 0, st>>>(kp, bt);
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

template <int R, bool FP16>
int launch_r(const rfi::KParams& kp, const rfi::BatchThr& bt, cudaStream_t st) {
    // sets per warp: 16 warps x {1, 4} covers K <= 16 and K <= 64
    if (kp.K <= rfi::kBatchWarps) return launch_rs<R, FP16, 1>(kp, bt, st);
    return launch_rs<R, FP16, 4>(kp, bt, st);
}

}  // namespace

int launch_batched(bool fp16, const rfi::KParams& kp, const rfi::BatchThr& bt, cudaStream_t st) {
    if (kp.K < 1 || kp.K > rfi::kMaxBatch) return RFI_EINVAL;
    const int R = pick_rows(kp.M, fp16, fp16 ? 8 : 4);
    if (!fp16) {
        switch (R) {
            case 1: return launch_r<1, false>(kp, bt, st);
            case 2: return launch_r<2, false>(kp, bt, st);
            case 3: return launch_r<3, false>(kp, bt, st);
            default: return launch_r<4, false>(kp, bt, st);
        }
    }
    switch (R) {
        case 1: return launch_r<1, true>(kp, bt, st);
        case 2: return launch_r<2, true>(kp, bt, st);
        case 3: return launch_r<3, true>(kp, bt, st);
        case 4: return launch_r<4, true>(kp, bt, st);
        case 5: return launch_r<5, true>(kp, bt, st);
        case 6: return launch_r<6, true>(kp, bt, st);
        case 7: return launch_r<7, true>(kp, bt, st);
        default: return launch_r<8, true>(kp, bt, st);
    }
}

}  // namespace rfi_host
