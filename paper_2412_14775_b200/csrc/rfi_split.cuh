// rfi_split.cuh -- low-latency variant for SMALL chunks (RFI_VARIANT_SPLIT): the rows of a unit are split over the
// warps of a CTA.
//
// The streaming kernels give one warp a whole (32-cell tile, output integration) unit and let it walk the unit's
// n_int rows with a few blocks in flight: perfect for chunks with thousands of units (HBM-bound), but a chunk with a
// handful of units (BASELINE.json configs[0]: 48 units of 64 rows) leaves 140 SMs idle while 48 warps each wait for
// 16 dependent memory round trips.  The paper keeps its windows small for latency; this variant keeps
// the kernel's latency small when the chunk is small: one CTA per unit, up to 16 warps,
//
//   phase 1  warp j takes blocks j, j+16, ... of R rows: ALL rows of the unit are in flight at once (one memory round
//            trip); per block it leaves the block statistics of |I| (mean, centred second moment) and the block's
//            partial sums (unit vectors, samples) in shared memory;
//   phase 2  warp v takes windows v, v+16, ...: merges the window's blocks IN ORDER (Chan merge: the same operations
//            in the same order as merge_block, so x is bit-identical to the direct kernel; the unit-vector and sample
//            sums are added block-wise, which differs from the direct kernel's sample-wise order in the last bits),
//            window tail, decision, flag word, statistics planes, and a window record (flag, sums) in shared memory;
//   phase 3  warp 0 adds the kept windows in order and stores the output.
//
// K = 1, RFI_ARITH_FAST, time-major layout, at most kSplitMaxBlocks blocks per unit (shared memory).
#pragma once

#include "rfi_kernels.cuh"

namespace rfi {

constexpr int kSplitMaxBlocks = 96;                           // 96 x 2 KiB of block partials
constexpr int kSplitPartFloats = 16;                          // mb, m2b, q/u/v (re,im parts), 8 sample sums
constexpr int kSplitRecFloats = 9;                            // flag, 8 sample sums

template <int R, bool FP16, bool ALIGN32>
__global__ void __launch_bounds__(512, 1) rfi_split_kernel(const KParams p) {
    constexpr int SAMPLE_BYTES = FP16 ? 16 : 32;
    extern __shared__ float sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int n_tiles = (p.n_cells + 31) >> 5;
    const int unit = blockIdx.x;
    const int o_local = unit / n_tiles;
    const int tile = unit - o_local * n_tiles;
    const int o_global = p.o_first + o_local;
    const LaneGeom g = lane_geom(p, tile, lane);
    const int nb = p.n_int / R, bpw = p.M / R;
    float* part = sm;                                         // [nb][kSplitPartFloats][32]
    float* rec = sm + (size_t)nb * kSplitPartFloats * 32;     // [wpo][kSplitRecFloats][32]
    const size_t row_stride = (size_t)p.n_cells * SAMPLE_BYTES;
    const uint8_t* base = static_cast<const uint8_t*>(p.vis) + (size_t)o_local * p.n_int * row_stride + (size_t)g.cell * SAMPLE_BYTES;

    // ---- phase 1: blocks ----
    for (int blk = warp; blk < nb; blk += nwarps) {
        Raw<FP16> buf[R];
        load_block<R, FP16, ALIGN32>(base + (size_t)blk * R * row_stride, row_stride, buf);
        Win w;
        w.reset();
        float z[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            f2 x[4];
            widen(buf[r], x);
            z[r] = accumulate_sample(w, x);
        }
        float mb, m2b;
        block_stats<R>(z, mb, m2b);
        float* o = part + (size_t)blk * kSplitPartFloats * 32 + lane;
        o[0] = mb; o[32] = m2b;
        float a, b;
        unpack2(w.q, a, b); o[2 * 32] = a; o[3 * 32] = b;
        unpack2(w.u, a, b); o[4 * 32] = a; o[5 * 32] = b;
        unpack2(w.v, a, b); o[6 * 32] = a; o[7 * 32] = b;
#pragma unroll
        for (int q = 0; q < 4; ++q) { unpack2(w.s[q], a, b); o[(8 + 2 * q) * 32] = a; o[(9 + 2 * q) * 32] = b; }
    }
    __syncthreads();

    // ---- phase 2: windows ----
    for (int wl = warp; wl < p.wpo; wl += nwarps) {
        Win w;
        w.reset();
        for (int b = 0; b < bpw; ++b) {
            const float* o = part + (size_t)(wl * bpw + b) * kSplitPartFloats * 32 + lane;
            merge_stats<R>(w, o[0], o[32], b);
            w.q = add2(w.q, pack2(o[2 * 32], o[3 * 32]));
            w.u = add2(w.u, pack2(o[4 * 32], o[5 * 32]));
            w.v = add2(w.v, pack2(o[6 * 32], o[7 * 32]));
#pragma unroll
            for (int q = 0; q < 4; ++q) w.s[q] = add2(w.s[q], pack2(o[(8 + 2 * q) * 32], o[(9 + 2 * q) * 32]));
        }
        float x, r_re, r_im;
        if (p.F > 1) combine_group(w, p.F, p.M);
        window_stats(w, p.inv_W, x, r_re, r_im);
        const Thr& t = g.cls ? p.thr1 : p.thr0;
        const bool flag = decide(x, max_nan(r_re, r_im), t);
        const int w_global = o_global * p.wpo + wl;
        store_flags(p, g, p.k_first, w_global, flag);
        store_stats(p, g, w_global, t.c * x, r_re, r_im);
        float* o = rec + (size_t)wl * kSplitRecFloats * 32 + lane;
        o[0] = flag ? 1.f : 0.f;
#pragma unroll
        for (int q = 0; q < 4; ++q) { float a, b; unpack2(w.s[q], a, b); o[(1 + 2 * q) * 32] = a; o[(2 + 2 * q) * 32] = b; }
    }
    __syncthreads();

    // ---- phase 3: the output integration: kept windows in order ----
    if (warp == 0) {
        f2 acc[4] = {0ull, 0ull, 0ull, 0ull};
        uint32_t wt = 0;
        for (int wl = 0; wl < p.wpo; ++wl) {
            const float* o = rec + (size_t)wl * kSplitRecFloats * 32 + lane;
            if (o[0] == 0.f) {
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[q] = add2(acc[q], pack2(o[(1 + 2 * q) * 32], o[(2 + 2 * q) * 32]));
                wt += (uint32_t)p.M;
            }
        }
        store_output(p, g, p.k_first, o_global, acc, wt);
    }
}

}  // namespace rfi
