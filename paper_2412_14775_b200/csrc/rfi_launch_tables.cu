// rfi_launch_tables.cu -- instantiations and launcher of the paper-literal mixed-precision kernel (rfi_tables.cuh).
#include "rfi_internal.h"
#include "rfi_tables.cuh"

namespace rfi_host {

int launch_tables_ps_part0(int idx, const rfi::KParams& kp, cudaStream_t st);
int launch_tables_ps_part1(int idx, const rfi::KParams& kp, cudaStream_t st);
int launch_tables_ps_part2(int idx, const rfi::KParams& kp, cudaStream_t st);
int launch_tables_ps_part3(int idx, const rfi::KParams& kp, cudaStream_t st);

int launch_tables_ps(const rfi::KParams& kp, cudaStream_t st) {
    const int i = (int)((kp.arith_mask & 15u) | (((kp.arith_mask >> 7) & 15u) << 4));   // the 8 per-sample bits
    switch (i >> 6) {
        case 0: return launch_tables_ps_part0(i & 63, kp, st);
        case 1: return launch_tables_ps_part1(i & 63, kp, st);
        case 2: return launch_tables_ps_part2(i & 63, kp, st);
        default: return launch_tables_ps_part3(i & 63, kp, st);
    }
}

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
    // Table 1 groups 5 and 7 in half, Table 2 groups 4-7 in half)
    if (kp.arith_mask == 0u) return launch_rm<R, 0>(kp, st);
    if (kp.arith_mask == 0x3C50u) return launch_rm<R, 0x3C50>(kp, st);
    // any other mask: block length 2 has one instantiation per assignment of the 8 per-sample groups (the per-window
    // tail reads its 6 bits at run time); other block lengths read the whole mask at run time
    if (R == 2 && env_int("RFI_TABLES_PS", 1)) return launch_tables_ps(kp, st);
    return launch_rm<R, -1>(kp, st);
}

}  // namespace

int launch_tables(const rfi::KParams& kp, cudaStream_t st) {
    // The arithmetic runs sample by sample whatever the block length (sums are sequential, rfi_tables.cuh), and this mode
    // is bound by instruction issue (nine IEEE divisions / square roots per sample), not by bytes in flight: short blocks
    // leave registers for more resident warps (R = 2: 24 warps per SM instead of 16, measured 4.18 -> 3.90 ms).
    int R = kp.M % 2 == 0 ? 2 : 1;
    const int force = env_int("RFI_TABLES_ROWS", 0);
    if (force >= 1 && force <= 4 && kp.M % force == 0) R = force;
    switch (R) {
        case 1: return launch_r<1>(kp, st);
        case 2: return launch_r<2>(kp, st);
        case 3: return launch_r<3>(kp, st);
        default: return launch_r<4>(kp, st);
    }
}

}  // namespace rfi_host
