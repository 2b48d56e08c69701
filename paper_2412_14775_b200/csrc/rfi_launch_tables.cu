// rfi_launch_tables.cu -- instantiations and launcher of the paper-literal mixed-precision kernel (rfi_tables.cuh).
#include "rfi_internal.h"
#include "rfi_tables.cuh"

namespace rfi_host {
namespace {

template <int R, int MASK>
int launch_rm(const rfi::KParams& kp, cudaStream_t st) {
    const int n_tiles = (kp.n_cells + 31) / 32;
    const long n_units = (long)n_tiles * kp.n_out_slab;
    const unsigned grid = (unsigned)((n_units + 3) / 4);
    rfi::rfi_tables_kernel<R, MASK><<<grid, 128, 0, st>>>(kp);
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

template <int R>
int launch_r(const rfi::KParams& kp, cudaStream_t st) {
    // compile-time masks: all single, and the assignment the paper's agent learned (Tables 3-4, PAPER.md:196-214:
    // Table 1 groups 5 and 7 in half, Table 2 groups 4-7 in half); anything else reads the mask at run time
    if (kp.arith_mask == 0u) return launch_rm<R, 0>(kp, st);
    if (kp.arith_mask == 0x3C50u) return launch_rm<R, 0x3C50>(kp, st);
    return launch_rm<R, -1>(kp, st);
}

}  // namespace

int launch_tables(const rfi::KParams& kp, cudaStream_t st) {
    switch (pick_rows(kp.M, false, 4)) {
        case 1: return launch_r<1>(kp, st);
        case 2: return launch_r<2>(kp, st);
        case 3: return launch_r<3>(kp, st);
        default: return launch_r<4>(kp, st);
    }
}

}  // namespace rfi_host
