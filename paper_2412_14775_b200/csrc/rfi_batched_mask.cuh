// rfi_batched_mask.cuh -- batched-threshold kernel, second generation: K <= 64 threshold sets in ONE pass over the
// data, for whole-word tiles (n_chan % 32 == 0).  Same function and same bits as rfi_batched_tma.cuh (which remains for
// ragged channel counts); what differs is where the K decisions are taken and how the flag words leave.
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
//   staging   the flag layout has the tile index fastest (include/rfi.h), so one tile's words are 4 isolated bytes per
//             (set, window): 32 distinct lines per store instruction, measured at 0.3 ms of a 3.4 ms K = 64 pass.  A CTA
//             therefore takes G adjacent tiles of one integration in a row (G = 8 when the row length allows) and every
//             stream warp parks the flag words of its own windows in tensor memory (tcgen05.st, 32 lanes x one column
//             per word: TMEM is otherwise unused by this path and shared memory is full); after the G-th tile the same
//             warp reads them back (tcgen05.ld.x8) and stores whole 32-byte sectors.  No cross-warp hand-off.
//
// The sums are added per set in window order, as in the single-set kernels: K sets equal K single-set runs bit for bit.
#pragma once

#include "rfi_batched_tma.cuh"

namespace rfi {

constexpr int kBmRecBytes = 1280;                 // per (round buffer, window): mask[2][32] u32, s01[32] 16 B, s23[32] 16 B
constexpr int kBmTblBytes = 3 * 64 * 4 + 3 * 65 * 8;   // per class: sorted x_low, x_high, gamma; prefix masks by rank
constexpr int kBmCntBytes = kBtWarps * 6 * 32 * 4;     // per warp: {fa, md} x {sets k, 32+k}, clean, rfi; one word per lane

__device__ __forceinline__ float lds_f32(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void lds_u32x2(uint32_t a, uint32_t& lo, uint32_t& hi) {
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(a));
}
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void red_shared_add(uint32_t a, uint32_t v) { asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
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

// ---- tensor memory as per-warp scratch (flag-word staging) ----
__device__ __forceinline__ void tmem_alloc(uint32_t smem_slot, uint32_t cols) {          // one whole warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_slot), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {             // one whole warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void tmem_st1(uint32_t taddr, uint32_t v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(v) : "memory");
}
template <int G>
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&r)[G]) {
    static_assert(G == 2 || G == 4 || G == 8, "group sizes");
    if constexpr (G == 8)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr) : "memory");
    else if constexpr (G == 4)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
    else
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
template <int G>
__device__ __forceinline__ void stg_words(uint32_t* dst, const uint32_t (&r)[G]) {        // dst aligned to 4 G bytes
    if constexpr (G == 8)
        asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(dst), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]),
                     "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
    else if constexpr (G == 4)
        asm volatile("st.global.cs.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(dst), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
    else
        asm volatile("st.global.cs.v2.b32 [%0], {%1,%2};" ::"l"(dst), "r"(r[0]), "r"(r[1]) : "memory");
}

// One warp's parked flag words of a finished tile group: for each of its windows (round ri, window ri*NW + warp) and
// each half of the sets (lane k: set k, set 32 + k), G consecutive TMEM columns = the words of tiles tile0 .. tile0+G-1.
template <int G>
__device__ __forceinline__ void flush_group_flags(const KParams& p, uint32_t tcol, int n_rounds, int warp, int lane,
                                                  uint32_t* flag_lo, size_t flag_set_stride, size_t fwpw, int o_global, int tile0) {
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    const int halves = p.K > 32 ? 2 : 1;
    for (int ri = 0; ri < n_rounds; ++ri) {
        const int wl = ri * kBtWarps + warp;
        if (wl >= p.wpo) break;
        for (int h = 0; h < halves; ++h) {
            uint32_t r[G];
            tmem_ld<G>(tcol + (uint32_t)((ri * 2 + h) * G), r);
            if (lane + 32 * h < p.K) {
                uint32_t* dst = flag_lo + (size_t)(32 * h) * flag_set_stride + ((size_t)o_global * p.wpo + wl) * fwpw + tile0;
                stg_words<G>(dst, r);
            }
        }
    }
}

template <int R, bool FP16, int SPW, bool CM>
__global__ void __launch_bounds__(kBtWarps * 32, 1)
rfi_batched_mask_kernel(const __grid_constant__ CUtensorMap tmap, const KParams p,
                        const __grid_constant__ BatchThr bt, const int stages, const int G, const int tm_cols) {
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
    const uint32_t cnt_base = perm_base + 384u;                                          // [NW][6][32] u32 confusion counters
    const uint32_t tm_slot = cnt_base + kBmCntBytes;                                           // TMEM base address (one word)
    const uint32_t round_bar = tm_slot + 8u;                                             // records of a round complete (all threads arrive)
    const uint32_t bars = tm_slot + 16u + (uint32_t)warp * stages * 16;                  // per warp: full[], empty[]
    const uint32_t ebars = bars + (uint32_t)stages * 8;

    // Work list: super-unit = (group of G adjacent tiles, output integration); its tiles are units taken in a row.
    const int n_tiles = p.n_cells >> 5;                       // whole tiles only (n_chan % 32 == 0)
    const int n_groups = n_tiles / G;                         // G divides the flag row length = n_tiles (launcher)
    const int n_su = n_groups * p.n_out_slab;
    if ((int)blockIdx.x >= n_su) return;
    const int bpw = p.M / R;                                  // stages per window
    const int n_rounds = (p.wpo + NW - 1) / NW;
    const float inv_M = p.inv_W;                              // 1/W, W = T*F
    const size_t fwpw = (size_t)p.n_baselines * p.wpb;        // flag words per window
    const size_t flag_set_stride = (size_t)p.n_win_total * fwpw;
    const int step_o = (int)gridDim.x / n_groups, step_g = (int)gridDim.x - step_o * n_groups;   // su += gridDim.x

    if (threadIdx.x == 0) mbar_init(round_bar, NW * 32);
    if (lane == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(bars + 8 * s, 1); mbar_init(ebars + 8 * s, 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    // ---- producer cursor (lane 0 only): super-unit -> tile of the group -> window (warp, warp+NW, ...) -> stage ----
    uint64_t pol = 0;
    bool pr_active = warp < p.wpo;
    int pr_su = blockIdx.x, pr_o = (int)blockIdx.x / n_groups, pr_grp = (int)blockIdx.x - pr_o * n_groups;
    int pr_j = 0, pr_wl = warp, pr_b = 0;
    auto pr_issue = [&](int s) {
        const uint32_t bar = bars + 8 * s;
        const uint32_t dst = ring + (uint32_t)s * STAGE_BYTES;
        const int row = pr_o * p.n_int + pr_wl * p.M + pr_b * R;
        const int tile = pr_grp * G + pr_j;
        mbar_expect_tx(bar, STAGE_BYTES);
        if constexpr (CM)        tma_load_3d(dst, &tmap, 0, row / R, tile * 32, bar, pol);
        else if constexpr (FP16) tma_load_2d(dst, &tmap, tile * 128, row, bar, pol);
        else                     tma_load_3d(dst, &tmap, 0, tile * 8, row, bar, pol);
        if (++pr_b == bpw) {
            pr_b = 0;
            pr_wl += NW;
            if (pr_wl >= p.wpo) {
                pr_wl = warp;
                if (++pr_j == G) {
                    pr_j = 0;
                    pr_su += gridDim.x;
                    pr_o += step_o;
                    pr_grp += step_g;
                    if (pr_grp >= n_groups) { pr_grp -= n_groups; ++pr_o; }
                    pr_active = pr_su < n_su;
                }
            }
        }
    };
    if (lane == 0 && pr_active) {
        pol = l2_evict_first_policy();
        for (int i = 0; i < stages && pr_active; ++i) pr_issue(i);
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
        if (p.truth)
            for (int i = t; i < kBmCntBytes / 4; i += NW * 32) sts_u32(cnt_base + 4u * i, 0u);
        if (warp == NW - 1 && G > 1) tmem_alloc(tm_slot, (uint32_t)tm_cols);    // flag staging (warp NW-1 is idle above)
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
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
    const uint32_t tm_base = G > 1 ? lds_u32(tm_slot) : 0u;
    // this warp's TMEM window: its lane quarter (warp % 4), columns [(warp / 4) * n_rounds * 2 G, +n_rounds * 2 G)
    const uint32_t tcol = tm_base + ((uint32_t)(warp & 3) << 21) + (uint32_t)((warp >> 2) * n_rounds * 2 * G);

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

    // stream side: lane k handles the flag words of sets k and 32 + k
    uint32_t* const flag_lo = p.flags + (size_t)(p.k_first + lane) * flag_set_stride;

    int stage = 0;
    uint32_t parity = 0, gr = 0;
    int o_local = (int)blockIdx.x / n_groups, grp = (int)blockIdx.x - o_local * n_groups;
    for (int su = blockIdx.x; su < n_su; su += gridDim.x) {
        const int o_global = p.o_first + o_local;
        const int tile0 = grp * G;
        for (int j = 0; j < G; ++j) {
            const int tile = tile0 + j;
            const int cls = p.cls ? (int)p.cls[p.b_first + (tile * 32) / p.n_chan] : 0;     // a whole-word tile lies in one baseline
            const uint32_t tbl = tbl_base + (uint32_t)cls * kBmTblBytes;
            LaneGeom g;
            g.cell = tile * 32 + lane;
            g.valid = true;
#pragma unroll
            for (int i = 0; i < SPW; ++i) {
                cnt[i] = 0u;
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[i][q] = 0ull;
            }

            for (int round = 0; round < n_rounds; ++round, ++gr) {
                const uint32_t rbuf = rec_base + (gr & 1u) * (NW * kBmRecBytes);
                const int wl = round * NW + warp;
                if (wl < p.wpo) {
                    Win w;
                    w.reset();
                    // the window's ground-truth word, if counters are wanted: asked for now, used after the statistics
                    const uint32_t tw = p.truth ? __ldg(p.truth + ((size_t)o_global * p.wpo + wl) * fwpw + tile) : 0u;
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
                        if (lane == 0 && pr_active) {
                            mbar_wait(ebars + 8 * stage, parity);
                            fence_proxy_async();
                            pr_issue(stage);
                        }
                        accumulate_block<R, FP16>(w, buf, b);
                        if (++stage == stages) { stage = 0; parity ^= 1u; }
                    }
                    float x, r_re, r_im;
                    if (p.F > 1) combine_group(w, p.F, p.M);
                    window_stats(w, inv_M, x, r_re, r_im);
                    const int w_global = o_global * p.wpo + wl;
                    uint32_t m_lo, m_hi;
                    keep_mask(tbl, x, max_nan(r_re, r_im), m_lo, m_hi);
                    // record: keep mask + window sums (zeros if not finite: such a window is kept by no set, and
                    // fma(NaN, 0, acc) would poison the accumulator)
                    const uint32_t ra = rbuf + (uint32_t)warp * kBmRecBytes;
                    sts_u32(ra + (uint32_t)lane * 4u, m_lo);
                    sts_u32(ra + 128u + (uint32_t)lane * 4u, m_hi);
                    const bool fin = finite2(w.s[0]) && finite2(w.s[1]) && finite2(w.s[2]) && finite2(w.s[3]);
                    sts128_f2(ra + 256u + (uint32_t)lane * 16u, fin ? w.s[0] : 0ull, fin ? w.s[1] : 0ull);
                    sts128_f2(ra + 768u + (uint32_t)lane * 16u, fin ? w.s[2] : 0ull, fin ? w.s[3] : 0ull);
                    // The record is out: arrive on the round barrier, then do what nobody waits for.
                    mbar_arrive(round_bar);
                    // flag words: transpose (cell, set) -> (set, cell); flagged = not kept
                    {
                        const uint32_t f_lo = ~warp_transpose32(m_lo, lane);
                        const uint32_t f_hi = p.K > 32 ? ~warp_transpose32(m_hi, lane) : 0u;
                        if (p.truth) {                         // confusion counters of sets k and 32 + k (rfi_plan_set_truth)
                            const uint32_t cw = cnt_base + (uint32_t)warp * 768u + (uint32_t)lane * 4u;
                            red_shared_add(cw, __popc(f_lo & ~tw));
                            red_shared_add(cw + 128u, __popc(~f_lo & tw));
                            red_shared_add(cw + 256u, __popc(f_hi & ~tw));
                            red_shared_add(cw + 384u, __popc(~f_hi & tw));
                            red_shared_add(cw + 512u, __popc(~tw));
                            red_shared_add(cw + 640u, __popc(tw));
                        }
                        if (G > 1) {                           // park them until the group's last tile
                            tmem_st1(tcol + (uint32_t)((round * 2) * G + j), f_lo);
                            if (p.K > 32) tmem_st1(tcol + (uint32_t)((round * 2 + 1) * G + j), f_hi);
                        } else {
                            const size_t wo = (size_t)w_global * fwpw + tile;
                            if (lane < p.K) flag_lo[wo] = f_lo;
                            if (lane + 32 < p.K) flag_lo[32 * flag_set_stride + wo] = f_hi;
                        }
                    }
                    if (p.k_first == 0) store_stats(p, g, w_global, (cls ? p.thr1.c : p.thr0.c) * x, r_re, r_im);
                } else {
                    mbar_arrive(round_bar);
                }
                mbar_wait(round_bar, gr & 1u);                 // every warp's record of this round is in shared memory
                contract_records<SPW>(rbuf, 0, min(NW, p.wpo - round * NW), lane, msel, align, acc, cnt);
            }
#pragma unroll
            for (int i = 0; i < SPW; ++i) {                     // the unit's averaged outputs
                const int k = warp * SPW + i;
                if (k < p.K) store_output(p, g, p.k_first + k, o_global, acc[i], cnt[i] * (uint32_t)p.M);
            }
        }
        if (G > 1) {
            if (G == 8)      flush_group_flags<8>(p, tcol, n_rounds, warp, lane, flag_lo, flag_set_stride, fwpw, o_global, tile0);
            else if (G == 4) flush_group_flags<4>(p, tcol, n_rounds, warp, lane, flag_lo, flag_set_stride, fwpw, o_global, tile0);
            else             flush_group_flags<2>(p, tcol, n_rounds, warp, lane, flag_lo, flag_set_stride, fwpw, o_global, tile0);
        }
        o_local += step_o;
        grp += step_g;
        if (grp >= n_groups) { grp -= n_groups; ++o_local; }
    }
    if (p.truth) {                                             // this warp's counters: lane k -> sets k and 32 + k
        const uint32_t cw = cnt_base + (uint32_t)warp * 768u + (uint32_t)lane * 4u;
        const unsigned long long clean = lds_u32(cw + 512u), rfi_n = lds_u32(cw + 640u);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int k = lane + 32 * h;
            if (k < p.K) {
                unsigned long long* c = p.counts + (size_t)(p.k_first + k) * 4;
                atomicAdd(c + 0, (unsigned long long)lds_u32(cw + 256u * h));
                atomicAdd(c + 1, clean);
                atomicAdd(c + 2, (unsigned long long)lds_u32(cw + 256u * h + 128u));
                atomicAdd(c + 3, rfi_n);
            }
        }
    }
    if (G > 1) {                                               // every warp is done with its columns
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (warp == NW - 1) tmem_dealloc(tm_base, (uint32_t)tm_cols);
    }
}

}  // namespace rfi
