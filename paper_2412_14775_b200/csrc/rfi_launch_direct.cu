// rfi_launch_direct.cu -- instantiations and launcher of the register-staged single-set kernel.
#include "rfi_internal.h"
#include "rfi_kernels.cuh"

namespace rfi_host {
namespace {

template <int R, bool FP16>
int launch_r(const rfi::KParams& kp, cudaStream_t st) {
    const int n_tiles = (kp.n_cells + 31) / 32;
    const long n_units = (long)n_tiles * kp.n_out_slab;
    const unsigned grid = (unsigned)((n_units + 3) / 4);
    // 256-bit loads need a 32-byte aligned sample: base % 32 == 0 (the sample stride is 32 B)
    const bool a32 = FP16 || (reinterpret_cast<uintptr_t>(kp.vis) % 32 == 0);
    if (kp.d_thr && kp.adapt_streams == 2) {                   // static thresholds per baseline stream (rfi_plan_set_stream_thresholds)
        if (a32) rfi::rfi_direct_kernel<R, FP16, true, 3><<<grid, 128, 0, st>>>(kp);
        else     rfi::rfi_direct_kernel<R, FP16, false, 3><<<grid, 128, 0, st>>>(kp);
    } else if (kp.d_thr && kp.adapt_streams) {                 // on-line adaptation per baseline stream
        if (a32) rfi::rfi_direct_kernel<R, FP16, true, 2><<<grid, 128, 0, st>>>(kp);
        else     rfi::rfi_direct_kernel<R, FP16, false, 2><<<grid, 128, 0, st>>>(kp);
    } else if (kp.d_thr) {                                     // on-line threshold adaptation per class (rfi_plan_set_adaptive)
        if (a32) rfi::rfi_direct_kernel<R, FP16, true, 1><<<grid, 128, 0, st>>>(kp);
        else     rfi::rfi_direct_kernel<R, FP16, false, 1><<<grid, 128, 0, st>>>(kp);
    } else {
        if (a32) rfi::rfi_direct_kernel<R, FP16, true><<<grid, 128, 0, st>>>(kp);
        else     rfi::rfi_direct_kernel<R, FP16, false><<<grid, 128, 0, st>>>(kp);
    }
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

}  // namespace

int launch_direct(bool fp16, const rfi::KParams& kp, cudaStream_t st) {
    const int R = pick_rows(kp.M, fp16);
    if (!fp16) {
        switch (R) {
            case 1: return launch_r<1, false>(kp, st);
            case 2: return launch_r<2, false>(kp, st);
            case 3: return launch_r<3, false>(kp, st);
            case 4: return launch_r<4, false>(kp, st);
            case 5: return launch_r<5, false>(kp, st);
            case 6: return launch_r<6, false>(kp, st);
            case 7: return launch_r<7, false>(kp, st);
            default: return launch_r<8, false>(kp, st);
        }
    }
    switch (R) {
        case 1: return launch_r<1, true>(kp, st);
        case 2: return launch_r<2, true>(kp, st);
        case 3: return launch_r<3, true>(kp, st);
        case 4: return launch_r<4, true>(kp, st);
        case 5: return launch_r<5, true>(kp, st);
        case 6: return launch_r<6, true>(kp, st);
        case 7: return launch_r<7, true>(kp, st);
        default: return launch_r<8, true>(kp, st);
    }
}

}  // namespace rfi_host
