// rfi_batched_tma.cuh -- batched-threshold kernel, TMA-staged: K <= 64 threshold sets in ONE pass over the data.
//
// Same function as rfi_batched.cuh (the register-staged fallback for ragged shapes); this is the fast path for
// n_chan % 32 == 0 (every 32-cell tile is exactly one flag word and has no invalid lane).
//
// The statistics (x = W S2/S1^2 - 1, r_re, r_im) and the window sums do not depend on the thresholds; only the
// decision and the masked accumulation do.  K x 8 accumulators per cell do not fit in
// one thread, so a persistent CTA of 16 warps shares one (32-cell tile, output integration) unit at a time:
//
//   stream    warp j owns window (round*16 + j) of the unit.  Its samples arrive through a warp-private ring of
//             cp.async.bulk.tensor stages (R time rows x 32 cells each; the ring runs ahead across rounds and
//             units, so HBM stays busy while the CTA contracts).  One thread per cell computes the window's
//             statistics exactly as the single-set kernels do and leaves a 48-byte record per cell in shared
//             memory: x, max(r_re, r_im), window sum[8]   (3 x 128-bit, stride 48 B: bank-conflict free).
//   contract  thread (warp j, lane l) owns cell l and the sets j*SPW .. j*SPW+SPW-1.  Per record and set:
//             3 compares, 1 ballot (the flag word of that window and set), 4 predicated packed adds and a
//             predicated count.  Lane i keeps the ballot of the round's i-th window, so the flag words of a
//             round leave with one store instruction per set.
//
// One __syncthreads per round (records are double-buffered).  Thresholds travel as a by-value kernel
// parameter (constant bank), already divided by c (rfi_window.cuh: decide).
#pragma once

#include "rfi_kernels.cuh"

namespace rfi {

constexpr int kBtWarps = 16;
constexpr int kRecBytes = 48;

// One record against one threshold set (Eq.(5), Eq.(10), then the exclusion of PAPER.md:75).
// keep = (x >= x_low) && (x <= x_high) && (r_max <= gamma): ordered compares, so a NaN statistic is not kept.
// Same decision as decide() in rfi_window.cuh.  The masked add is acc = fma(sum, keep ? 1 : 0, acc): exactly
// acc + sum when kept, exactly acc when not (one packed instruction per pair; a predicated packed add costs
// three).  This needs finite sums: the stream side stores zeros for a window whose sums are not finite -- such
// a window has NaN statistics and is flagged by every set anyway.
// Returns the warp's flag word (bit l = lane l flagged); cnt counts kept windows (exact in fp32 below 2^24).
__device__ __forceinline__ uint32_t contract_one(float x, float r_max, float x_low, float x_high, float gamma,
                                                 f2 (&a)[4], float& cnt, const f2 (&s)[4]) {
    uint32_t word;
    float kf;
    asm volatile(
        "{\n\t.reg .pred k;\n\t"
        "setp.ge.f32 k, %2, %4;\n\t"
        "setp.le.and.f32 k, %2, %5, k;\n\t"
        "setp.le.and.f32 k, %3, %6, k;\n\t"
        "vote.sync.ballot.b32 %0, !k, 0xffffffff;\n\t"
        "selp.f32 %1, 0f3F800000, 0f00000000, k;\n\t}"
        : "=r"(word), "=f"(kf)
        : "f"(x), "f"(r_max), "f"(x_low), "f"(x_high), "f"(gamma));
    const f2 kk = pack2(kf, kf);
#pragma unroll
    for (int q = 0; q < 4; ++q) a[q] = fma2(s[q], kk, a[q]);
    cnt += kf;
    return word;
}

__device__ __forceinline__ bool finite2(f2 v) {
    float lo, hi;
    unpack2(v, lo, hi);
    return fabsf(lo) <= 3.402823466e38f && fabsf(hi) <= 3.402823466e38f;
}

__device__ __forceinline__ void sts128(uint32_t addr, float a, float b, float c, float d) {
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void sts128_f2(uint32_t addr, f2 a, f2 b) {
    asm volatile("st.shared.v2.b64 [%0], {%1,%2};" ::"r"(addr), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void lds128_f2(uint32_t addr, f2& a, f2& b) {
    asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}
__device__ __forceinline__ void lds128_head(uint32_t addr, float& a, float& b) {   // 128-bit keeps the 48 B stride conflict-free
    float c, d;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "r"(addr));
}

template <int R, bool FP16, int SPW, bool FULLWORD, bool CM = false>
__global__ void __launch_bounds__(kBtWarps * 32, 1)
rfi_batched_tma_kernel(const __grid_constant__ CUtensorMap tmap, const KParams p,
                       const __grid_constant__ BatchThr bt, const int stages) {
    constexpr int NW = kBtWarps;
    constexpr int ROW_BYTES = FP16 ? 512 : 1024;
    static_assert(!CM || R == (FP16 ? 8 : 4), "cell-major stages hold one 128-byte line per cell");
    constexpr int STAGE_BYTES = CM ? 4096 : R * ROW_BYTES;   // CM: cell-major input, see rfi_tma_kernel
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const uint32_t ring = smem_base + (uint32_t)warp * stages * STAGE_BYTES;
    const uint32_t rec_base = smem_base + (uint32_t)NW * stages * STAGE_BYTES;          // [2][NW][32 lanes][48 B]
    // per warp: `stages` "full" barriers followed by `stages` "empty" barriers (consumer -> producer hand-off)
    const uint32_t bars = rec_base + 2u * NW * 32u * kRecBytes + (uint32_t)warp * stages * 16;
    const uint32_t ebars = bars + (uint32_t)stages * 8;

    const int n_tiles = (p.n_cells + 31) >> 5;                // FULLWORD (n_chan % 32 == 0): whole tiles only; else the
                                                              // last tile is ragged (TMA zero-fills, invalid lanes are masked)
    const int n_units = n_tiles * p.n_out_slab;
    if ((int)blockIdx.x >= n_units) return;
    const int my_units = (n_units - 1 - (int)blockIdx.x) / (int)gridDim.x + 1;
    const int bpw = p.M / R;                                  // stages per window
    const int n_rounds = (p.wpo + NW - 1) / NW;
    const int my_n = warp < p.wpo ? (p.wpo - 1 - warp) / NW + 1 : 0;     // windows of a unit streamed by this warp
    const int total = my_units * my_n * bpw;                  // stages this warp consumes in its lifetime
    const float inv_M = p.inv_W;                             // 1/W, W = T*F
    const size_t flag_words_per_win = (size_t)p.n_baselines * p.wpb;
    const size_t flag_set_stride = (size_t)p.n_win_total * flag_words_per_win;

    if (lane == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(bars + 8 * s, 1); mbar_init(ebars + 8 * s, 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    // ---- producer cursor (lane 0 only): unit -> window (warp, warp+NW, ...) -> stage ----
    uint64_t pol = 0;
    int pr_unit = blockIdx.x, pr_wl = warp, pr_b = 0, pr_tile = 0, pr_row0 = 0, pr_i = 0;
    auto pr_locate = [&]() {
        const int o_local = pr_unit / n_tiles;
        pr_tile = pr_unit - o_local * n_tiles;
        pr_row0 = o_local * p.n_int;
    };
    auto pr_issue = [&]() {
        const int s = pr_i % stages;
        const uint32_t bar = bars + 8 * s;
        const uint32_t dst = ring + (uint32_t)s * STAGE_BYTES;
        const int row = pr_row0 + pr_wl * p.M + pr_b * R;
        mbar_expect_tx(bar, STAGE_BYTES);
        if constexpr (CM)        tma_load_3d(dst, &tmap, 0, row / R, pr_tile * 32, bar, pol);
        else if constexpr (FP16) tma_load_2d(dst, &tmap, pr_tile * 128, row, bar, pol);
        else                     tma_load_3d(dst, &tmap, 0, pr_tile * 8, row, bar, pol);
        ++pr_i;
        if (++pr_b == bpw) {
            pr_b = 0;
            pr_wl += NW;
            if (pr_wl >= p.wpo) { pr_wl = warp; pr_unit += gridDim.x; pr_locate(); }
        }
    };
    if (lane == 0 && total > 0) {
        pol = l2_evict_first_policy();
        pr_locate();
        const int pre = total < stages ? total : stages;
        for (int i = 0; i < pre; ++i) pr_issue();
    }

    // lane-constant shared-memory offsets of this lane's sample inside one row (see rfi_tma_kernel)
    uint32_t off0, off1;
    if constexpr (FP16) {
        off0 = (uint32_t)lane * 16u;
        off1 = 0;
    } else {
        const uint32_t grp = (uint32_t)lane >> 2;
        const uint32_t chunk = ((uint32_t)lane & 3u) * 2u;
        off0 = grp * 128u + ((chunk ^ grp) << 4);
        off1 = grp * 128u + (((chunk + 1u) ^ grp) << 4);
    }

    int it = 0, stage = 0;
    uint32_t parity = 0, gr = 0;
    for (int ui = 0; ui < my_units; ++ui) {
        const int unit = blockIdx.x + ui * gridDim.x;
        const int o_local = unit / n_tiles;
        const int tile = unit - o_local * n_tiles;
        const int o_global = p.o_first + o_local;
        LaneGeom g;
        if constexpr (FULLWORD) {
            g.cell = tile * 32 + lane;
            g.valid = true;
            g.word = tile; g.bit = lane; g.group = 0xffffffffu; g.leader = lane == 0;
            g.cls = p.cls ? (int)p.cls[p.b_first + (tile * 32) / p.n_chan] : 0;   // a whole-word tile lies in one baseline
        } else {
            g = lane_geom(p, tile, lane);                      // several flag words per tile, ragged last tile
        }

        // this lane's flag word of set warp*SPW, window (round 0, lane): later sets / rounds are fixed strides away
        uint32_t* const flag_ptr = p.flags + ((size_t)(p.k_first + warp * SPW) * p.n_win_total
                                              + (size_t)o_global * p.wpo + lane) * flag_words_per_win + tile;
        f2 acc[SPW][4];
        float cnt[SPW];
#pragma unroll
        for (int i = 0; i < SPW; ++i) {
            cnt[i] = 0.f;
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][q] = 0ull;
        }

        for (int round = 0; round < n_rounds; ++round, ++gr) {
            const uint32_t rbuf = rec_base + (gr & 1u) * (NW * 32u * kRecBytes);
            const int wl = round * NW + warp;
            // ---- stream: this warp's window of the round ----
            if (wl < p.wpo) {
                Win w;
                w.reset();
                for (int b = 0; b < bpw; ++b) {
                    mbar_wait(bars + 8 * stage, parity);
                    const uint32_t sbase = ring + (uint32_t)stage * STAGE_BYTES;
                    Raw<FP16> buf[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if constexpr (CM) {
                            const uint32_t line = sbase + (uint32_t)lane * 128u, sx = (uint32_t)lane & 7u;
                            if constexpr (FP16) lds_raw(line + (((uint32_t)r ^ sx) << 4), 0, buf[r]);
                            else                lds_raw(line + (((uint32_t)(2 * r) ^ sx) << 4), line + (((uint32_t)(2 * r + 1) ^ sx) << 4), buf[r]);
                        } else {
                            lds_raw(sbase + r * ROW_BYTES + off0, sbase + r * ROW_BYTES + off1, buf[r]);
                        }
                    }
                    // stage hand-off (rfi_common.cuh): 32 arrivals after the loads, wait, proxy fence, refill
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
                float x, r_re, r_im;
                if (p.F > 1) combine_group(w, p.F, p.M);
            window_stats(w, inv_M, x, r_re, r_im);
                const uint32_t ra = rbuf + ((uint32_t)warp * 32u + lane) * kRecBytes;
                sts128(ra, x, max_nan(r_re, r_im), 0.f, 0.f);
                const bool fin = finite2(w.s[0]) && finite2(w.s[1]) && finite2(w.s[2]) && finite2(w.s[3]);
                sts128_f2(ra + 16, fin ? w.s[0] : 0ull, fin ? w.s[1] : 0ull);
                sts128_f2(ra + 32, fin ? w.s[2] : 0ull, fin ? w.s[3] : 0ull);
                if (p.k_first == 0) store_stats(p, g, o_global * p.wpo + wl, (g.cls ? p.thr1.c : p.thr0.c) * x, r_re, r_im);
            }
            __syncthreads();
            // ---- contract: this thread's sets against the round's records ----
            const int n_w = min(NW, p.wpo - round * NW);
            float xl[SPW], xh[SPW], gm[SPW];
            uint32_t myw[SPW];
#pragma unroll
            for (int i = 0; i < SPW; ++i) {
                const Thr t = g.cls ? bt.t1[warp * SPW + i] : bt.t[warp * SPW + i];   // the lane's baseline class
                xl[i] = t.x_low; xh[i] = t.x_high; gm[i] = t.gamma;
                myw[i] = 0;
            }
            uint32_t ra = rbuf + (uint32_t)lane * kRecBytes;
#pragma unroll 2
            for (int j = 0; j < n_w; ++j, ra += 32u * kRecBytes) {
                float x, r_max;
                f2 s[4];
                lds128_head(ra, x, r_max);
                lds128_f2(ra + 16, s[0], s[1]);
                lds128_f2(ra + 32, s[2], s[3]);
                const bool mine = lane == j;
#pragma unroll
                for (int i = 0; i < SPW; ++i) {
                    const uint32_t word = contract_one(x, r_max, xl[i], xh[i], gm[i], acc[i], cnt[i], s);
                    if constexpr (FULLWORD) {
                        myw[i] = mine ? word : myw[i];
                    } else {
                        // the lanes of one flag word are contiguous: the leader shifts its group's bits into place
                        const int k = warp * SPW + i;
                        if (g.leader && k < p.K) {
                            const uint32_t v = ((word & g.group) >> lane) << g.bit;
                            uint32_t* dst = p.flags + ((size_t)(p.k_first + k) * p.n_win_total + (size_t)o_global * p.wpo
                                                       + round * NW + j) * flag_words_per_win + g.word;
                            if (p.flags_atomic) atomicOr(dst, v); else *dst = v;
                        }
                    }
                }
            }
            if (FULLWORD && lane < n_w) {
                uint32_t* fp = flag_ptr + (size_t)round * NW * flag_words_per_win;
#pragma unroll
                for (int i = 0; i < SPW; ++i, fp += flag_set_stride)
                    if (warp * SPW + i < p.K) *fp = myw[i];
            }
        }
#pragma unroll
        for (int i = 0; i < SPW; ++i) {
            const int k = warp * SPW + i;
            if (k < p.K) store_output(p, g, p.k_first + k, o_global, acc[i], (uint32_t)cnt[i] * (uint32_t)p.M);
        }
    }
}

}  // namespace rfi
