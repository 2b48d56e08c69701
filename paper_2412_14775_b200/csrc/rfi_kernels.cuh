// rfi_kernels.cuh -- the single-set streaming kernels (K = 1) of the fused flag-and-average pass.
//
// A "unit" of work is (32-cell tile, output integration); one warp owns one unit at a time and walks its
// n_int time samples in blocks of R rows (R divides the window length M).
#pragma once

#include <type_traits>

#include "rfi_window.cuh"

namespace rfi {

// ------------------------------------------------------------------------------------------------
// Variant DIRECT: per-thread streaming loads, no shared memory.  Two register buffers of R raw samples
// (ping-pong): the loads of block i+1 are in flight while block i is consumed, i.e. R x 32 B (fp32) or
// R x 16 B (fp16) per thread, 128 B with the default R (4 / 8).
// ------------------------------------------------------------------------------------------------
template <int R, bool FP16, bool ALIGN32>
__device__ __forceinline__ void load_block(const uint8_t* ptr, size_t row_stride, Raw<FP16> (&buf)[R]) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if constexpr (!FP16 && !ALIGN32) ldg_stream_16B(ptr + (size_t)r * row_stride, buf[r]);
        else                             ldg_stream(ptr + (size_t)r * row_stride, buf[r]);
    }
}

// One (tile, integration) unit of the direct kernel.  ADAPT (on-line threshold adaptation, rfi_adapt.cu): the lane's
// thresholds are read from device memory once per unit and every window is counted in the CTA's histogram.
template <int R, bool FP16, bool ALIGN32, int ADAPT>
__device__ __forceinline__ void direct_unit(const KParams& p, const int unit, const int n_tiles, uint32_t* sh_hist) {
    constexpr int SAMPLE_BYTES = FP16 ? 16 : 32;
    const int lane = threadIdx.x & 31;
    const int o_local = unit / n_tiles;
    const int tile = unit - o_local * n_tiles;
    const LaneGeom g = lane_geom(p, tile, lane);
    const float inv_M = p.inv_W;                             // 1/W, W = T*F
    const size_t row_stride = (size_t)p.n_cells * SAMPLE_BYTES;
    const size_t blk_stride = row_stride * R;
    const uint8_t* ptr = static_cast<const uint8_t*>(p.vis) + (size_t)o_local * p.n_int * row_stride
                         + (size_t)g.cell * SAMPLE_BYTES;
    const int o_global = p.o_first + o_local;
    const int bpw = p.M / R;                          // blocks per window
    const int total = p.n_int / R;                    // blocks per unit
    int w_global = o_global * p.wpo;

    f2 acc[4] = {0ull, 0ull, 0ull, 0ull};
    uint32_t wt = 0;
    Win w;
    w.reset();
    int blk = 0, b_in_win = 0;

    Thr thr_dev;
    // ADAPT = 1: thresholds and histograms per baseline class; ADAPT = 2: per baseline STREAM (the tile lies in one baseline:
    // n_chan % 32 == 0, checked by the host), histogram private to the warp and flushed at the end of the unit; ADAPT = 3:
    // per-stream thresholds given by the caller, no histogram
    const int stream = ADAPT >= 2 ? (tile * 32) / p.n_chan : g.cls;
    if constexpr (ADAPT != 0) thr_dev = p.d_thr[stream];
    Raw<FP16> A[R], B[R];
    auto window_end = [&]() {
        ++blk;
        if (++b_in_win == bpw) {
            finish_window<ADAPT>(p, g, w, inv_M, w_global, acc, wt, &thr_dev, sh_hist);
            ++w_global;
            b_in_win = 0;
            w.reset();
        }
    };
    if constexpr (FP16) {
        // Row-granular register ring of 2R rows: a row's registers are refilled (row + 2R) right after the row
        // is consumed, so between R and 2R-1 rows (128..240 B) per thread are in flight instead of exactly R.
        // Measured on B200 (profiles/): fp16 1.445 -> 1.321 ms; fp32 loses 1.5 % to spills and keeps the ping-pong.
        load_block<R, FP16, ALIGN32>(ptr, row_stride, A);
        if (total > 1) load_block<R, FP16, ALIGN32>(ptr + blk_stride, row_stride, B);
        ptr += 2 * blk_stride;                        // address of the row that refills A[0]
        auto step = [&](auto always, Raw<FP16> (&cur)[R]) {
            const bool refill = decltype(always)::value || blk + 2 < total;
            float z[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                f2 x[4];
                widen(cur[r], x);
                if (refill) ldg_stream(ptr + (size_t)r * row_stride, cur[r]);
                z[r] = accumulate_sample(w, x);
            }
            ptr += blk_stride;
            merge_block<R>(w, z, b_in_win);
            window_end();
        };
        while (blk + 4 <= total) {                    // both steps refill unconditionally
            step(std::true_type{}, A);
            step(std::true_type{}, B);
        }
        while (blk + 2 <= total) {
            step(std::false_type{}, A);
            step(std::false_type{}, B);
        }
        if (blk < total) step(std::false_type{}, A);
    } else {
        // Ping-pong: the loads of block i+1 are issued before block i is consumed.
        load_block<R, FP16, ALIGN32>(ptr, row_stride, A);
        ptr += blk_stride;
        auto step = [&](Raw<FP16> (&cur)[R], Raw<FP16> (&nxt)[R]) {
            if (blk + 1 < total) {
                load_block<R, FP16, ALIGN32>(ptr, row_stride, nxt);
                ptr += blk_stride;
            }
            accumulate_block<R, FP16>(w, cur, b_in_win);
            window_end();
        };
        while (blk + 2 <= total) {
            step(A, B);
            step(B, A);
        }
        if (blk < total) step(A, B);
    }
    store_output(p, g, p.k_first, o_global, acc, wt);
    if constexpr (ADAPT == 2) {
        __syncwarp();
        uint32_t* dst = p.hist + (size_t)stream * kAdaptBins;
        for (int i = lane; i < kAdaptBins; i += 32) {
            const uint32_t c = sh_hist[i];
            if (c) { atomicAdd(dst + i, c); sh_hist[i] = 0u; }
        }
        __syncwarp();
    }
}

template <int R, bool FP16, bool ALIGN32, int ADAPT = 0>
__global__ void __launch_bounds__(128, (FP16 || R <= 4) ? 4 : (R == 5 ? 3 : 2)) rfi_direct_kernel(const KParams p) {
    const int n_tiles = (p.n_cells + 31) >> 5;
    const int unit = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if constexpr (ADAPT == 0) {
        if (unit < n_tiles * p.n_out_slab) direct_unit<R, FP16, ALIGN32, 0>(p, unit, n_tiles, nullptr);
    } else if constexpr (ADAPT == 1) {
        __shared__ uint32_t sh_hist[2 * kAdaptBins];          // [class][tau bins | r bins], flushed once per CTA
        for (int i = threadIdx.x; i < 2 * kAdaptBins; i += blockDim.x) sh_hist[i] = 0u;
        __syncthreads();
        if (unit < n_tiles * p.n_out_slab) direct_unit<R, FP16, ALIGN32, 1>(p, unit, n_tiles, sh_hist);
        __syncthreads();
        for (int i = threadIdx.x; i < 2 * kAdaptBins; i += blockDim.x) {
            const uint32_t c = sh_hist[i];
            if (c) atomicAdd(p.hist + i, c);
        }
    } else if constexpr (ADAPT == 3) {
        if (unit < n_tiles * p.n_out_slab) direct_unit<R, FP16, ALIGN32, 3>(p, unit, n_tiles, nullptr);
    } else {
        __shared__ uint32_t sh_hist[4 * kAdaptBins];          // one [tau bins | r bins] histogram per warp (= per unit = one stream)
        uint32_t* mine = sh_hist + (threadIdx.x >> 5) * kAdaptBins;
        for (int i = threadIdx.x & 31; i < kAdaptBins; i += 32) mine[i] = 0u;
        __syncwarp();
        if (unit < n_tiles * p.n_out_slab) direct_unit<R, FP16, ALIGN32, 2>(p, unit, n_tiles, mine);
    }
}

// ------------------------------------------------------------------------------------------------
// Variant TMA: persistent CTAs; every warp owns a private ring of `stages` shared-memory stages.
// Lane 0 issues one cp.async.bulk.tensor per stage (R time rows x 32 cells), the warp waits on the
// stage's mbarrier, consumes it from shared memory, and lane 0 refills the stage.  No CTA-wide
// synchronisation exists after setup; bytes in flight are bounded by shared memory, not registers.
//
// fp32: 3-D tensor {32 floats = 4 cells, n_cells/4, n_time}, box {32, 8, R}, SWIZZLE_128B: the 16-byte
//       chunk index is XORed with the 128-byte line index (mod 8), which makes the two 128-bit
//       shared loads of a lane (32-byte stride between lanes) bank-conflict free.
// fp16: 2-D tensor {n_cells*4 words, n_time}, box {128, R}: lanes read consecutive 16 B, no swizzle needed.
//
// CM = true: the CELL-MAJOR input layout vis[b][c][t][pol] (each cell's time series contiguous).  The same kernel
// with a transposing tensor map: 3-D tensor {32 words = 128 B = R samples of one cell, n_time/R, n_cells}, box
// {32, 1, 32 cells}, SWIZZLE_128B.  A stage is 32 lines of 128 B, line l = the R samples of the tile's cell l; lane l
// reads its own line, chunk index XOR (l mod 8): conflict free per quarter warp.  After that a thread owns a cell
// and R consecutive samples exactly as in the time-major kernels, so the results are bit-identical to them.
// R is fixed by the 128-byte line: 4 (fp32) or 8 (fp16).
// ------------------------------------------------------------------------------------------------
template <int R, bool FP16, bool CM = false>
__global__ void __launch_bounds__(512, 1) rfi_tma_kernel(const __grid_constant__ CUtensorMap tmap,
                                                           const KParams p, const int stages) {
    static_assert(!CM || R == (FP16 ? 8 : 4), "cell-major stages hold one 128-byte line per cell");
    constexpr int ROW_BYTES = FP16 ? 512 : 1024;
    constexpr int STAGE_BYTES = CM ? 4096 : R * ROW_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const uint32_t ring = smem_base + (uint32_t)warp * stages * STAGE_BYTES;
    // per warp: `stages` "full" barriers (count 1 + TMA bytes) followed by `stages` "empty" barriers (count 32)
    const uint32_t bars = smem_base + (uint32_t)nwarps * stages * STAGE_BYTES + (uint32_t)warp * stages * 16;
    const uint32_t ebars = bars + (uint32_t)stages * 8;

    const int n_tiles = (p.n_cells + 31) >> 5;
    const int n_units = n_tiles * p.n_out_slab;
    const int gw = blockIdx.x * nwarps + warp;
    const int GW = gridDim.x * nwarps;
    if (gw >= n_units) return;                                // warp-private pipeline: safe to leave
    const int my_units = (n_units - 1 - gw) / GW + 1;
    const int bpu = p.n_int / R;                              // blocks (stages) per unit
    const int total = my_units * bpu;
    const int bpw = p.M / R;
    const float inv_M = p.inv_W;                             // 1/W, W = T*F

    if (lane == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(bars + 8 * s, 1); mbar_init(ebars + 8 * s, 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    // producer cursor (lane 0 only uses it)
    uint64_t pol = 0;
    int pr_unit = gw, pr_blk = 0, pr_tile = 0, pr_row0 = 0, pr_i = 0;
    auto pr_locate = [&]() {
        const int o_local = pr_unit / n_tiles;
        pr_tile = pr_unit - o_local * n_tiles;
        pr_row0 = o_local * p.n_int;
    };
    auto pr_issue = [&]() {
        const int s = pr_i % stages;
        const uint32_t bar = bars + 8 * s;
        const uint32_t dst = ring + (uint32_t)s * STAGE_BYTES;
        mbar_expect_tx(bar, STAGE_BYTES);
        if constexpr (CM)        tma_load_3d(dst, &tmap, 0, pr_row0 / R + pr_blk, pr_tile * 32, bar, pol);
        else if constexpr (FP16) tma_load_2d(dst, &tmap, pr_tile * 128, pr_row0 + pr_blk * R, bar, pol);
        else                     tma_load_3d(dst, &tmap, 0, pr_tile * 8, pr_row0 + pr_blk * R, bar, pol);
        ++pr_i;
        if (++pr_blk == bpu) { pr_blk = 0; pr_unit += GW; pr_locate(); }
    };
    if (lane == 0) {
        pol = l2_evict_first_policy();
        pr_locate();
        const int pre = total < stages ? total : stages;
        for (int i = 0; i < pre; ++i) pr_issue();
    }

    // lane-constant shared-memory offsets of this lane's sample inside one row
    uint32_t off0, off1;
    if constexpr (FP16) {
        off0 = (uint32_t)lane * 16u;
        off1 = 0;
    } else {
        const uint32_t grp = (uint32_t)lane >> 2;             // 128-byte line within the row
        const uint32_t chunk = ((uint32_t)lane & 3u) * 2u;    // 16-byte chunk of the first half
        off0 = grp * 128u + ((chunk ^ grp) << 4);
        off1 = grp * 128u + (((chunk + 1u) ^ grp) << 4);
    }

    int it = 0, stage = 0;
    uint32_t parity = 0;
    for (int j = 0; j < my_units; ++j) {
        const int unit = gw + j * GW;
        const int o_local = unit / n_tiles;
        const int tile = unit - o_local * n_tiles;
        const int o_global = p.o_first + o_local;
        const LaneGeom g = lane_geom(p, tile, lane);
        f2 acc[4] = {0ull, 0ull, 0ull, 0ull};
        uint32_t wt = 0;

        for (int wl = 0; wl < p.wpo; ++wl) {
            Win w;
            w.reset();
            for (int b = 0; b < bpw; ++b) {
                mbar_wait(bars + 8 * stage, parity);
                const uint32_t sbase = ring + (uint32_t)stage * STAGE_BYTES;
                Raw<FP16> buf[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if constexpr (CM) {
                        const uint32_t line = sbase + (uint32_t)lane * 128u, x = (uint32_t)lane & 7u;
                        if constexpr (FP16) lds_raw(line + (((uint32_t)r ^ x) << 4), 0, buf[r]);
                        else                lds_raw(line + (((uint32_t)(2 * r) ^ x) << 4), line + (((uint32_t)(2 * r + 1) ^ x) << 4), buf[r]);
                    } else {
                        lds_raw(sbase + r * ROW_BYTES + off0, sbase + r * ROW_BYTES + off1, buf[r]);
                    }
                }
                // hand the stage back (rfi_common.cuh): every lane arrives after its loads of the stage, the producer
                // lane waits for the 32 arrivals (same phase parity as the fill just consumed), fences the proxies, refills
                mbar_arrive(ebars + 8 * stage);
                if (lane == 0 && it + stages < total) {
                    mbar_wait(ebars + 8 * stage, parity);
                    fence_proxy_async();
                    pr_issue();
                }
                accumulate_block<R, FP16>(w, buf, b);
                ++it;
                if (++stage == stages) { stage = 0; parity ^= 1u; }
            }
            finish_window(p, g, w, inv_M, o_global * p.wpo + wl, acc, wt);
        }
        store_output(p, g, p.k_first, o_global, acc, wt);
    }
}

}  // namespace rfi
