// rfi_batched.cuh -- batched-threshold kernel: K <= 64 threshold sets evaluated in ONE pass over the data.
//
// The statistics (x = W S2/S1^2 - 1, r_re, r_im) and the window sums do not depend on the thresholds; only
// the decision and the masked accumulation do.  K x 8 accumulators per cell do not
// fit in one thread's registers, so a CTA of NW = 16 warps shares one 32-cell tile:
//
//   stream phase    warp j computes window (round*NW + j) of the tile's output integration, one thread per
//                   cell exactly as in the single-set kernel, and leaves an 11-float record per cell
//                   (x, r_re, r_im, window sum[8]) in shared memory;
//   contract phase  thread (warp j, lane l) owns cell l and the SPW sets j*SPW .. j*SPW+SPW-1: it walks the
//                   round's NW records, decides per set, packs the flag word with a warp ballot and adds the
//                   window sum into its per-set accumulators (SPW x 8 fp32 registers + SPW counters).
//
// One __syncthreads per round (records are double-buffered).  The loads of a warp's next window are already in
// flight while the CTA contracts, so HBM stays busy during the ALU-heavy phase.  Thresholds travel as a
// by-value kernel parameter (constant bank).
#pragma once

#include "rfi_kernels.cuh"

namespace rfi {

constexpr int kBatchWarps = 16;
constexpr int kRecFloats = 11;

template <int R, bool FP16, bool ALIGN32, int SPW>
__global__ void __launch_bounds__(kBatchWarps * 32, 1)
rfi_batched_kernel(const KParams p, const __grid_constant__ BatchThr bt) {
    constexpr int NW = kBatchWarps;
    constexpr int SAMPLE_BYTES = FP16 ? 16 : 32;
    __shared__ float rec[2][NW][kRecFloats][32];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int n_tiles = (p.n_cells + 31) >> 5;
    const int unit = blockIdx.x;
    const int o_local = unit / n_tiles;
    const int tile = unit - o_local * n_tiles;
    const int o_global = p.o_first + o_local;
    const LaneGeom g = lane_geom(p, tile, lane);
    const float inv_M = p.inv_W;                             // 1/W, W = T*F
    const size_t row_stride = (size_t)p.n_cells * SAMPLE_BYTES;
    const size_t blk_stride = row_stride * R;
    const size_t win_jump = blk_stride + (size_t)(NW - 1) * p.M * row_stride;   // last block of a window -> first block of window + NW
    const int bpw = p.M / R;
    const int n_rounds = (p.wpo + NW - 1) / NW;
    const int my_n = warp < p.wpo ? (p.wpo - 1 - warp) / NW + 1 : 0;             // windows streamed by this warp
    const int total = my_n * bpw;

    const uint8_t* nptr = static_cast<const uint8_t*>(p.vis) + ((size_t)o_local * p.n_int + (size_t)warp * p.M) * row_stride
                          + (size_t)g.cell * SAMPLE_BYTES;
    int ld_b = 0;
    auto advance = [&]() {
        if (++ld_b == bpw) { ld_b = 0; nptr += win_jump; } else { nptr += blk_stride; }
    };

    f2 acc[SPW][4];
    uint32_t wt[SPW];
#pragma unroll
    for (int i = 0; i < SPW; ++i) {
        wt[i] = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[i][q] = 0ull;
    }

    Win w;
    w.reset();
    int blk = 0, b_in_win = 0;
    Raw<FP16> A[R], B[R];
    if (total > 0) {
        load_block<R, FP16, ALIGN32>(nptr, row_stride, A);
        advance();
    }
    auto step = [&](Raw<FP16> (&cur)[R], Raw<FP16> (&nxt)[R]) {
        if (blk + 1 < total) {
            load_block<R, FP16, ALIGN32>(nptr, row_stride, nxt);
            advance();
        }
        accumulate_block<R, FP16>(w, cur, b_in_win);
        ++blk;
        ++b_in_win;
    };

    for (int round = 0; round < n_rounds; ++round) {
        const int buf = round & 1;
        // ---- stream phase: this warp's window of the round ----
        if (round < my_n) {
            for (int b = 0; b < bpw; ++b) {
                if (blk & 1) step(B, A); else step(A, B);
            }
            float x, r_re, r_im;
            if (p.F > 1) combine_group(w, p.F, p.M);
            window_stats(w, inv_M, x, r_re, r_im);
            float (*my)[32] = rec[buf][warp];
            my[0][lane] = x;
            my[1][lane] = r_re;
            my[2][lane] = r_im;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float lo, hi;
                unpack2(w.s[q], lo, hi);
                my[3 + 2 * q][lane] = lo;
                my[4 + 2 * q][lane] = hi;
            }
            if (p.k_first == 0) store_stats(p, g, o_global * p.wpo + round * NW + warp, (g.cls ? p.thr1.c : p.thr0.c) * x, r_re, r_im);
            w.reset();
            b_in_win = 0;
        }
        __syncthreads();
        // ---- contract phase: this thread's sets over the round's windows ----
        const int n_w = min(NW, p.wpo - round * NW);
        for (int j = 0; j < n_w; ++j) {
            const float (*rj)[32] = rec[buf][j];
            const float x = rj[0][lane], r_re = rj[1][lane], r_im = rj[2][lane];
            f2 s[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) s[q] = pack2(rj[3 + 2 * q][lane], rj[4 + 2 * q][lane]);
            const int w_global = o_global * p.wpo + round * NW + j;
#pragma unroll
            for (int i = 0; i < SPW; ++i) {
                const int k = warp * SPW + i;
                if (k < p.K) {                                         // warp-uniform
                    const bool flag = decide(x, max_nan(r_re, r_im), g.cls ? bt.t1[k] : bt.t[k]);
                    store_flags(p, g, p.k_first + k, w_global, flag);
                    if (!flag) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) acc[i][q] = add2(acc[i][q], s[q]);
                        wt[i] += (uint32_t)p.M;
                    }
                }
            }
        }
    }
#pragma unroll
    for (int i = 0; i < SPW; ++i) {
        const int k = warp * SPW + i;
        if (k < p.K) store_output(p, g, p.k_first + k, o_global, acc[i], wt[i]);
    }
}

}  // namespace rfi
