// rfi_batched_mask.cuh -- batched-threshold kernel, second generation: K <= 64 threshold sets in ONE pass over the
// data, for whole-word tiles (n_chan % 32 == 0).  Same function and same bits as rfi_batched_tma.cuh (which remains for
// ragged channel counts); what differs is where the K decisions are taken and when the masked sums are formed.
//
//   decide    once per (window, cell), by the thread that streamed the window: the K decisions of Eq.(5) / Eq.(10)
//              are three rank queries.  With the sets sorted by s_low / s_high / gamma (done once
//             per CTA, in shared memory), {k : x >= x_low[k]} is a prefix of the first order, {k : x <= x_high[k]} a
//             suffix of the second, {k : r <= gamma[k]} a suffix of the third; each prefix is a 64-bit set mask looked
//             up by its length, and the window's keep mask is the AND of the three: 21 probes instead of 192 compares.
//             The probes are the same float comparisons as decide() in rfi_window.cuh (NaN statistic -> empty mask).
//   flags     the 32 keep masks of a window (lane = cell, bit = set) are transposed inside the warp (5 butterfly
//             steps per 32 sets), so lane k holds set k's 32-cell flag word and stores it: no ballot per (set, window).
//   contract  thread (warp j, lane l) owns cell l and the sets j*SPW .. j*SPW+SPW-1.  Per record: one predicate per
//             set from the mask bits, a 0/1 factor, 4 packed fma (exactly acc + sum or acc: see contract_one in
//             rfi_batched_tma.cuh), a predicated count.
//   pipeline  the contraction of round g-1 is interleaved, block by block, with the streaming of round g (records are
//             double-buffered, one CTA barrier per round): the TMA ring keeps refilling while the warp contracts, so
//             HBM does not idle during the contraction as it does when the two phases alternate.
//
// The sums are added per set in window order, as in the single-set kernels: K sets equal K single-set runs bit for bit.
#pragma once

#include "rfi_batched_tma.cuh"

namespace rfi {

constexpr int kBmRecBytes = 1280;                 // per (round buffer, window): mask[2][32] u32, s01[32] 16 B, s23[32] 16 B
constexpr int kBmTblBytes = 3 * 64 * 4 + 3 * 65 * 8;   // per class: sorted x_low, x_high, gamma; prefix masks by rank

__device__ __forceinline__ float lds_f32(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void lds_u32x2(uint32_t a, uint32_t& lo, uint32_t& hi) {
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(a));
}
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_u32x2(uint32_t a, uint32_t lo, uint32_t hi) {
    asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(a), "r"(lo), "r"(hi) : "memory");
}

// 32 x 32 bit-matrix transpose across a warp: lane l enters with row l (bit k = M[l][k]) and leaves with column l
// (bit k = M[k][l]).  Recursive block transpose, one shuffle per level.
__device__ __forceinline__ uint32_t warp_transpose32(uint32_t x, int lane) {
#pragma unroll
    for (int j = 16; j >= 1; j >>= 1) {
        const uint32_t m = j == 16 ? 0x0000FFFFu : j == 8 ? 0x00FF00FFu : j == 4 ? 0x0F0F0F0Fu : j == 2 ? 0x33333333u : 0x55555555u;
        const uint32_t y = __shfl_xor_sync(0xffffffffu, x, j);
        x = (lane & j) ? ((x & ~m) | ((y >> j) & m)) : ((x & m) | ((y << j) & ~m));
    }
    return x;
}

// Keep mask of one (window, cell) against the 64 sets: bit k = (x >= x_low[k]) && (x <= x_high[k]) && (r <= gamma[k]).
// `tbl` = the lane's class table in shared memory.  Branch-free rank queries on the three sorted arrays, interleaved.
__device__ __forceinline__ void keep_mask(uint32_t tbl, float x, float r_max, uint32_t& m_lo, uint32_t& m_hi) {
    uint32_t pa = tbl, pb = tbl + 256, pc = tbl + 512;
#pragma unroll
    for (int step = 32; step >= 1; step >>= 1) {
        const float va = lds_f32(pa + (step - 1) * 4), vb = lds_f32(pb + (step - 1) * 4), vc = lds_f32(pc + (step - 1) * 4);
        pa += (va <= x) ? step * 4 : 0;                         // a = #{k : x_low[k] <= x}; NaN x -> 0 -> empty mask
        pb += (vb < x) ? step * 4 : 0;                          // b = #{k : x_high[k] < x}
        pc += !(vc >= r_max) ? step * 4 : 0;                    // c = #{k : !(gamma[k] >= r)}; NaN r -> 64 -> empty mask
    }
    {
        const float va = lds_f32(pa), vb = lds_f32(pb), vc = lds_f32(pc);
        pa += (va <= x) ? 4 : 0;
        pb += (vb < x) ? 4 : 0;
        pc += !(vc >= r_max) ? 4 : 0;
    }
    // byte offset of a rank inside its float array = 4 * rank; the 64-bit masks sit at 8 * rank
    uint32_t a0, a1, b0, b1, c0, c1;
    lds_u32x2(tbl + 768 + 2 * (pa - tbl), a0, a1);                          // sets with x_low <= x
    lds_u32x2(tbl + 768 + 520 + 2 * (pb - (tbl + 256)), b0, b1);            // sets with x_high >= x (complement stored)
    lds_u32x2(tbl + 768 + 1040 + 2 * (pc - (tbl + 512)), c0, c1);           // sets with gamma >= r   (complement stored)
    m_lo = a0 & b0 & c0;
    m_hi = a1 & b1 & c1;
}

// Records [j0, j1) of one round buffer against this thread's SPW sets.  `msel` = byte offset of the mask word holding
// the warp's sets, `align` = left shift that brings them to the top SPW bits.
template <int SPW>
__device__ __forceinline__ void contract_records(uint32_t rbuf, int j0, int j1, int lane, uint32_t msel, int align,
                                                 f2 (&acc)[SPW][4], uint32_t (&cnt)[SPW]) {
    uint32_t ra = rbuf + (uint32_t)j0 * kBmRecBytes;
#pragma unroll 2
    for (int j = j0; j < j1; ++j, ra += kBmRecBytes) {
        const uint32_t top = lds_u32(ra + msel + (uint32_t)lane * 4u) << align;
        f2 s[4];
        lds128_f2(ra + 256 + (uint32_t)lane * 16u, s[0], s[1]);
        lds128_f2(ra + 768 + (uint32_t)lane * 16u, s[2], s[3]);
#pragma unroll
        for (int i = 0; i < SPW; ++i) {
            const bool keep = (top & (1u << (32 - SPW + i))) != 0u;
            const float kf = keep ? 1.0f : 0.0f;
            const f2 kk = pack2(kf, kf);
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][q] = fma2(s[q], kk, acc[i][q]);
            if (keep) ++cnt[i];
        }
    }
}

template <int R, bool FP16, int SPW, bool CM, bool PIPE>
__global__ void __launch_bounds__(kBtWarps * 32, 1)
rfi_batched_mask_kernel(const __grid_constant__ CUtensorMap tmap, const KParams p,
                        const __grid_constant__ BatchThr bt, const int stages) {
    constexpr int NW = kBtWarps;
    constexpr int ROW_BYTES = FP16 ? 512 : 1024;
    static_assert(!CM || R == (FP16 ? 8 : 4), "cell-major stages hold one 128-byte line per cell");
    constexpr int STAGE_BYTES = CM ? 4096 : R * ROW_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const uint32_t ring = smem_base + (uint32_t)warp * stages * STAGE_BYTES;
    const uint32_t rec_base = smem_base + (uint32_t)NW * stages * STAGE_BYTES;          // [2][NW] records
    const uint32_t tbl_base = rec_base + 2u * NW * kBmRecBytes;                          // [2 classes] tables
    const uint32_t perm_base = tbl_base + 2u * kBmTblBytes;                              // [6][64] u8 sort permutations
    const uint32_t bars = perm_base + 384u + (uint32_t)warp * stages * 16;               // per warp: full[], empty[]
    const uint32_t ebars = bars + (uint32_t)stages * 8;

    const int n_tiles = p.n_cells >> 5;                       // whole tiles only (n_chan % 32 == 0)
    const int n_units = n_tiles * p.n_out_slab;
    if ((int)blockIdx.x >= n_units) return;
    const int my_units = (n_units - 1 - (int)blockIdx.x) / (int)gridDim.x + 1;
    const int bpw = p.M / R;                                  // stages per window
    const int n_rounds = (p.wpo + NW - 1) / NW;
    const int my_n = warp < p.wpo ? (p.wpo - 1 - warp) / NW + 1 : 0;     // windows of a unit streamed by this warp
    const int total = my_units * my_n * bpw;                  // stages this warp consumes in its lifetime
    const float inv_M = p.inv_W;                              // 1/W, W = T*F
    const size_t fwpw = (size_t)p.n_baselines * p.wpb;        // flag words per window
    const size_t flag_set_stride = (size_t)p.n_win_total * fwpw;

    if (lane == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(bars + 8 * s, 1); mbar_init(ebars + 8 * s, 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    // ---- producer cursor (lane 0 only): unit -> window (warp, warp+NW, ...) -> stage; no divisions on the way ----
    uint64_t pol = 0;
    const int step_o = (int)gridDim.x / n_tiles, step_t = (int)gridDim.x - step_o * n_tiles;   // unit += gridDim.x
    int pr_left = total, pr_wl = warp, pr_b = 0;
    int pr_o = (int)blockIdx.x / n_tiles, pr_tile = (int)blockIdx.x - pr_o * n_tiles;
    auto pr_issue = [&](int s) {
        const uint32_t bar = bars + 8 * s;
        const uint32_t dst = ring + (uint32_t)s * STAGE_BYTES;
        const int row = pr_o * p.n_int + pr_wl * p.M + pr_b * R;
        mbar_expect_tx(bar, STAGE_BYTES);
        if constexpr (CM)        tma_load_3d(dst, &tmap, 0, row / R, pr_tile * 32, bar, pol);
        else if constexpr (FP16) tma_load_2d(dst, &tmap, pr_tile * 128, row, bar, pol);
        else                     tma_load_3d(dst, &tmap, 0, pr_tile * 8, row, bar, pol);
        --pr_left;
        if (++pr_b == bpw) {
            pr_b = 0;
            pr_wl += NW;
            if (pr_wl >= p.wpo) {
                pr_wl = warp;
                pr_o += step_o;
                pr_tile += step_t;
                if (pr_tile >= n_tiles) { pr_tile -= n_tiles; ++pr_o; }
            }
        }
    };
    if (lane == 0 && total > 0) {
        pol = l2_evict_first_policy();
        const int pre = total < stages ? total : stages;
        for (int i = 0; i < pre; ++i) pr_issue(i);
    }

    // ---- per-CTA threshold tables: the K sets sorted by x_low, x_high, gamma; prefix masks by rank ----
    {
        const int t = threadIdx.x;
        if (t < 384) {
            const int a = t >> 6, i = t & 63, cls = a / 3, kind = a - 3 * cls;
            auto val = [&](int j) -> float {
                if (j >= p.K) return 0.f;                     // unused sets: their mask bits are never read
                const Thr& th = cls ? bt.t1[j] : bt.t[j];
                return kind == 0 ? th.x_low : (kind == 1 ? th.x_high : th.gamma);
            };
            const float v = val(i);
            int rank = 0;
            for (int j = 0; j < 64; ++j) {
                const float u = val(j);
                rank += (u < v || (u == v && j < i)) ? 1 : 0;
            }
            sts_f32(tbl_base + cls * kBmTblBytes + kind * 256 + rank * 4, v);
            asm volatile("st.shared.u8 [%0], %1;" ::"r"(perm_base + a * 64 + rank), "r"(i) : "memory");
        }
        __syncthreads();
        if (t < 390) {
            const int a = t / 65, n = t - a * 65, cls = a / 3, kind = a - 3 * cls;
            unsigned long long m = 0ull;
            for (int j = 0; j < n; ++j) {
                uint32_t k;
                asm volatile("ld.shared.u8 %0, [%1];" : "=r"(k) : "r"(perm_base + a * 64 + j));
                m |= 1ull << k;
            }
            if (kind != 0) m = ~m;                            // x_high, gamma: the sets NOT in the prefix are kept
            sts_u32x2(tbl_base + cls * kBmTblBytes + 768 + kind * 520 + n * 8, (uint32_t)m, (uint32_t)(m >> 32));
        }
        __syncthreads();
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

    // contract side: this warp's sets sit at bits warp*SPW .. of the 64-bit keep mask
    const uint32_t msel = (uint32_t)((warp * SPW) >> 5) * 128u;
    const int align = 32 - SPW - ((warp * SPW) & 31);
    f2 acc[SPW][4];
    uint32_t cnt[SPW];
    auto reset_acc = [&]() {
#pragma unroll
        for (int i = 0; i < SPW; ++i) {
            cnt[i] = 0u;
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][q] = 0ull;
        }
    };
    auto store_unit = [&](int tile, int o_global) {           // the unit's K averaged outputs
        LaneGeom g;
        g.cell = tile * 32 + lane;
        g.valid = true;
#pragma unroll
        for (int i = 0; i < SPW; ++i) {
            const int k = warp * SPW + i;
            if (k < p.K) store_output(p, g, p.k_first + k, o_global, acc[i], cnt[i] * (uint32_t)p.M);
        }
    };
    reset_acc();

    // stream side: lane k stores the flag words of sets k and 32 + k
    uint32_t* const flag_lo = p.flags + (size_t)(p.k_first + lane) * flag_set_stride;
    uint32_t* const flag_hi = flag_lo + 32 * flag_set_stride;

    int stage = 0;
    uint32_t parity = 0;
    int o_local = (int)blockIdx.x / n_tiles, tile = (int)blockIdx.x - o_local * n_tiles;
    int prev_tile = 0, prev_o_global = 0, prev_n = 0;         // the round whose records wait to be contracted
    bool prev_last = false;
    uint32_t gr = 0;
    for (int ui = 0; ui < my_units; ++ui) {
        const int o_global = p.o_first + o_local;
        const int cls = p.cls ? (int)p.cls[p.b_first + (tile * 32) / p.n_chan] : 0;     // a whole-word tile lies in one baseline
        const uint32_t tbl = tbl_base + (uint32_t)cls * kBmTblBytes;
        LaneGeom g;
        g.cell = tile * 32 + lane;
        g.valid = true;

        for (int round = 0; round < n_rounds; ++round, ++gr) {
            const uint32_t wbuf = rec_base + (gr & 1u) * (NW * kBmRecBytes);
            const uint32_t pbuf = rec_base + ((gr & 1u) ^ 1u) * (NW * kBmRecBytes);
            const int wl = round * NW + warp;
            const int n_w = min(NW, p.wpo - round * NW);
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
                    if (lane == 0 && pr_left > 0) {
                        mbar_wait(ebars + 8 * stage, parity);
                        fence_proxy_async();
                        pr_issue(stage);
                    }
                    accumulate_block<R, FP16>(w, buf, b);
                    if (++stage == stages) { stage = 0; parity ^= 1u; }
                    if constexpr (PIPE) {                      // a slice of the previous round's records
                        contract_records<SPW>(pbuf, (b * prev_n) / bpw, ((b + 1) * prev_n) / bpw, lane, msel, align, acc, cnt);
                    }
                }
                float x, r_re, r_im;
                if (p.F > 1) combine_group(w, p.F, p.M);
                window_stats(w, inv_M, x, r_re, r_im);
                const int w_global = o_global * p.wpo + wl;
                uint32_t m_lo, m_hi;
                keep_mask(tbl, x, max_nan(r_re, r_im), m_lo, m_hi);
                // record: keep mask + window sums (zeros if not finite: such a window is kept by no set, and
                // fma(NaN, 0, acc) would poison the accumulator)
                const uint32_t ra = wbuf + (uint32_t)warp * kBmRecBytes;
                sts_u32(ra + (uint32_t)lane * 4u, m_lo);
                sts_u32(ra + 128u + (uint32_t)lane * 4u, m_hi);
                const bool fin = finite2(w.s[0]) && finite2(w.s[1]) && finite2(w.s[2]) && finite2(w.s[3]);
                sts128_f2(ra + 256u + (uint32_t)lane * 16u, fin ? w.s[0] : 0ull, fin ? w.s[1] : 0ull);
                sts128_f2(ra + 768u + (uint32_t)lane * 16u, fin ? w.s[2] : 0ull, fin ? w.s[3] : 0ull);
                // flag words: transpose (cell, set) -> (set, cell); flagged = not kept
                {
                    const size_t wo = (size_t)w_global * fwpw + tile;
                    const uint32_t t_lo = warp_transpose32(m_lo, lane);
                    if (lane < p.K) flag_lo[wo] = ~t_lo;
                    if (p.K > 32) {
                        const uint32_t t_hi = warp_transpose32(m_hi, lane);
                        if (lane + 32 < p.K) flag_hi[wo] = ~t_hi;
                    }
                }
                if (p.k_first == 0) store_stats(p, g, w_global, (cls ? p.thr1.c : p.thr0.c) * x, r_re, r_im);
            } else if constexpr (PIPE) {
                contract_records<SPW>(pbuf, 0, prev_n, lane, msel, align, acc, cnt);
            }
            if constexpr (PIPE) {
                if (prev_last) { store_unit(prev_tile, prev_o_global); reset_acc(); }
                prev_n = n_w; prev_tile = tile; prev_o_global = o_global; prev_last = round == n_rounds - 1;
                __syncthreads();
            } else {
                __syncthreads();
                contract_records<SPW>(wbuf, 0, n_w, lane, msel, align, acc, cnt);
            }
        }
        if constexpr (!PIPE) { store_unit(tile, o_global); reset_acc(); }
        o_local += step_o;
        tile += step_t;
        if (tile >= n_tiles) { tile -= n_tiles; ++o_local; }
    }
    if constexpr (PIPE) {                                      // drain: the last round's records
        contract_records<SPW>(rec_base + ((gr & 1u) ^ 1u) * (NW * kBmRecBytes), 0, prev_n, lane, msel, align, acc, cnt);
        store_unit(prev_tile, prev_o_global);
    }
}

}  // namespace rfi
