// rfi_kernels.cuh -- sm_100a device code of the fused flag-and-average pass.
//
// What is computed is defined in include/rfi.h (equations of PAPER.md cited there).  This file is
// the product path: it shares nothing with oracle/.
//
// Mapping: one thread = one (baseline, channel) cell, a warp = 32 consecutive cells.  With the
// time-slowest layout a warp's row of one time step is 1 KiB (fp32) / 512 B (fp16) contiguous, so
// every global access is a whole-line, fully used request.  A "unit" of work is (32-cell tile,
// output integration); statistics never cross lanes, the only warp collective is the ballot that
// packs the flag bits.
//
// SK in centred form: Eq.(4)'s  W*S2/S1^2 - 1  equals  sum (z_i - zbar)^2 / (W zbar^2)  with z_i = |I_i|.
// The running mean / centred second moment (Welford) recurrence evaluates it without the
// cancellation of the raw-moment form in fp32.
#pragma once

#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace rfi {

constexpr int kInvNTable = 4096;
__constant__ float c_inv_n[kInvNTable];          // c_inv_n[i] = 1/(i+1), uploaded once per device

struct Thr {                                      // one threshold set, device form
    float c;                                      // (W d + 1)/(W - 1), Eq.(4) prefactor
    float s_low, s_high, gamma;
};

struct KParams {
    const void* vis;          // slab base: [rows][n_cells] samples
    float* avg;               // [K][n_out_total][n_cells][8]
    uint32_t* weight;         // [K][n_out_total][n_cells]
    float* stats;             // [3][n_win_total][n_cells] or nullptr
    uint32_t* flags;          // [K][n_win_total][n_baselines*wpb]
    const Thr* thr_table;     // K sets (batched kernel)
    Thr thr0;                 // set 0 (single-set kernels; stats use its c)
    int n_cells, n_chan, n_baselines, wpb;
    int M, n_int, wpo;        // window, samples per output, windows per output
    int n_out_slab;           // outputs contained in this slab
    int o_first;              // global index of the slab's first output
    int n_out_total, n_win_total;
    int K;
    int flags_atomic;         // 1: flag words may be shared between warps -> atomicOr into a zeroed buffer
};

// ------------------------------------------------------------------------------------------------
// small PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// 256-bit streaming load: read-once data, keep it out of L1 and mark it evict-first in L2
__device__ __forceinline__ void ldg256_stream(const void* p, float (&v)[8]) {
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "l"(p));
}
__device__ __forceinline__ uint4 ldg128_stream(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint4 lds128(uint32_t saddr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(saddr));
    return r;
}
__device__ __forceinline__ void half8_to_float(const uint4& h, float (&v)[8]) {
    const __half2* p = reinterpret_cast<const __half2*>(&h);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float2 f = __half22float2(p[i]);
        v[2 * i] = f.x;
        v[2 * i + 1] = f.y;
    }
}
__device__ __forceinline__ void u4x2_to_float(const uint4& a, const uint4& b, float (&v)[8]) {
    v[0] = __uint_as_float(a.x); v[1] = __uint_as_float(a.y); v[2] = __uint_as_float(a.z); v[3] = __uint_as_float(a.w);
    v[4] = __uint_as_float(b.x); v[5] = __uint_as_float(b.y); v[6] = __uint_as_float(b.z); v[7] = __uint_as_float(b.w);
}

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2,
                                            uint32_t bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(pol)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1,
                                            uint32_t bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar), "l"(pol)
        : "memory");
}

// ------------------------------------------------------------------------------------------------
// per-window state and per-sample update (one thread = one cell)
// ------------------------------------------------------------------------------------------------
struct Win {
    float mean, m2;            // running mean and centred second moment of z = |I|   (Eq.(3))
    float qr, ur, vr;          // sum of unit vectors, real parts of (Q,U,V)            (Eq.(8))
    float qi, ui, vi;          // the same for the imaginary parts
    float s[8];                // plain sum of the window's samples (for the average)
    __device__ __forceinline__ void reset() {
        mean = m2 = qr = ur = vr = qi = ui = vi = 0.f;
#pragma unroll
        for (int p = 0; p < 8; ++p) s[p] = 0.f;
    }
};

// v = {xx.re, xx.im, xy.re, xy.im, yx.re, yx.im, yy.re, yy.im};  inv_n = 1/(index of this sample in the window, from 1)
__device__ __forceinline__ void accumulate(Win& w, const float (&v)[8], float inv_n) {
    // Eq.(2): I = xx+yy, Q = xx-yy, U = xy+yx, V = j(xy-yx) -> Re V = -Im(xy-yx), Im V = Re(xy-yx).
    // The sign of V cannot change r (it enters through v^2 and (sum v)^2), so D = xy - yx is used as is.
    const float Ir = v[0] + v[6], Ii = v[1] + v[7];
    const float Qr = v[0] - v[6], Qi = v[1] - v[7];
    const float Ur = v[2] + v[4], Ui = v[3] + v[5];
    const float Dr = v[2] - v[4], Di = v[3] - v[5];
    // Table 1 groups 1-4: y = |I|^2, z = |I|, then the centred recurrence
    const float y = fmaf(Ir, Ir, Ii * Ii);
    const float z = sqrt_approx(y);
    const float delta = z - w.mean;
    w.mean = fmaf(delta, inv_n, w.mean);
    w.m2 = fmaf(delta, z - w.mean, w.m2);
    // Table 2 groups 1-4, real parts: (Qr, Ur, -Di); imaginary parts: (Qi, Ui, Dr)
    const float p2r = fmaf(Qr, Qr, fmaf(Ur, Ur, Di * Di));
    const float p2i = fmaf(Qi, Qi, fmaf(Ui, Ui, Dr * Dr));
    // exact-zero guard: p = 0 means q = u = v = 0, and 0 * rsqrt(FLT_MIN) = 0
    const float ir = rsqrt_approx(fmaxf(p2r, 1.17549435e-38f));
    const float ii = rsqrt_approx(fmaxf(p2i, 1.17549435e-38f));
    w.qr = fmaf(Qr, ir, w.qr);
    w.ur = fmaf(Ur, ir, w.ur);
    w.vr = fmaf(Di, ir, w.vr);
    w.qi = fmaf(Qi, ii, w.qi);
    w.ui = fmaf(Ui, ii, w.ui);
    w.vi = fmaf(Dr, ii, w.vi);
#pragma unroll
    for (int p = 0; p < 8; ++p) w.s[p] += v[p];
}

// Window tail: Eq.(4) in centred form and Eq.(9).  x = W*S2/S1^2 - 1; tau = c * x.
__device__ __forceinline__ void window_stats(const Win& w, float fM, float& x, float& r_re, float& r_im) {
    // all-zero window: S1 = 0 -> x = -1 (the eps -> 0 limit of Table 1 row 7)
    x = (w.mean == 0.f) ? -1.f : w.m2 / (fM * w.mean * w.mean);
    r_re = sqrtf(fmaf(w.qr, w.qr, fmaf(w.ur, w.ur, w.vr * w.vr))) / fM;
    r_im = sqrtf(fmaf(w.qi, w.qi, fmaf(w.ui, w.ui, w.vi * w.vi))) / fM;
}

// Eq.(5), Eq.(10), OR-combined; negated so that NaN flags.
__device__ __forceinline__ bool decide(float x, float r_re, float r_im, const Thr& t) {
    const float tau = t.c * x;
    return !(tau >= t.s_low && tau <= t.s_high) || !(r_re <= t.gamma) || !(r_im <= t.gamma);
}

// Per-unit lane geometry: which cell, which flag word / bit.
struct LaneGeom {
    int cell;          // clamped to a valid cell for loads
    bool valid;
    int word;          // b * wpb + c/32
    int bit;           // c % 32
    unsigned group;    // lanes of this warp that share `word`
    bool leader;       // lowest lane of the group
};

__device__ __forceinline__ LaneGeom lane_geom(const KParams& p, int tile, int lane) {
    LaneGeom g;
    const int cell = tile * 32 + lane;
    g.valid = cell < p.n_cells;
    g.cell = g.valid ? cell : p.n_cells - 1;
    const int b = g.cell / p.n_chan;
    const int c = g.cell - b * p.n_chan;
    g.word = g.valid ? b * p.wpb + (c >> 5) : -1 - lane;      // invalid lanes form singleton groups
    g.bit = c & 31;
    g.group = __match_any_sync(0xffffffffu, g.word);
    g.leader = g.valid && ((__ffs(g.group) - 1) == lane);
    return g;
}

// Pack the warp's flag bits into the mask (layout in include/rfi.h).
__device__ __forceinline__ void store_flags(const KParams& p, const LaneGeom& g, int k, int w_global, bool flag) {
    const unsigned mine = (flag && g.valid) ? (1u << g.bit) : 0u;
    const unsigned word = __reduce_or_sync(g.group, mine);
    if (g.leader) {
        uint32_t* dst = p.flags + ((size_t)k * p.n_win_total + w_global) * ((size_t)p.n_baselines * p.wpb) + g.word;
        if (p.flags_atomic) atomicOr(dst, word); else *dst = word;
    }
}

__device__ __forceinline__ void store_stats(const KParams& p, const LaneGeom& g, int w_global,
                                            float tau, float r_re, float r_im) {
    if (p.stats && g.valid) {
        const size_t plane = (size_t)p.n_win_total * p.n_cells;
        const size_t i = (size_t)w_global * p.n_cells + g.cell;
        p.stats[i] = tau;
        p.stats[plane + i] = r_re;
        p.stats[2 * plane + i] = r_im;
    }
}

__device__ __forceinline__ void store_output(const KParams& p, const LaneGeom& g, int k, int o_global,
                                             const float (&acc)[8], uint32_t wt) {
    if (!g.valid) return;
    const size_t oi = ((size_t)k * p.n_out_total + o_global) * p.n_cells + g.cell;
    float4 a, b;
    if (wt) {
        const float fw = (float)wt;
        a = make_float4(acc[0] / fw, acc[1] / fw, acc[2] / fw, acc[3] / fw);
        b = make_float4(acc[4] / fw, acc[5] / fw, acc[6] / fw, acc[7] / fw);
    } else {
        a = b = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float4* dst = reinterpret_cast<float4*>(p.avg + oi * 8);
    dst[0] = a;
    dst[1] = b;
    p.weight[oi] = wt;
}

// ------------------------------------------------------------------------------------------------
// Variant DIRECT: per-thread streaming loads, R samples in flight per thread (double-buffered).
// One warp = one unit.  R divides M.
// ------------------------------------------------------------------------------------------------
template <bool FP16, bool V8>
__device__ __forceinline__ void load_sample(const uint8_t* ptr, float (&v)[8]) {
    if constexpr (FP16) {
        half8_to_float(ldg128_stream(ptr), v);
    } else if constexpr (V8) {
        ldg256_stream(ptr, v);
    } else {
        u4x2_to_float(ldg128_stream(ptr), ldg128_stream(ptr + 16), v);
    }
}

template <int R, bool FP16, bool V8>
__global__ void __launch_bounds__(128) rfi_direct_kernel(const KParams p) {
    constexpr int SAMPLE_BYTES = FP16 ? 16 : 32;
    const int lane = threadIdx.x & 31;
    const int n_tiles = (p.n_cells + 31) >> 5;
    const int unit = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (unit >= n_tiles * p.n_out_slab) return;
    const int o_local = unit / n_tiles;
    const int tile = unit - o_local * n_tiles;
    const LaneGeom g = lane_geom(p, tile, lane);
    const float fM = (float)p.M;
    const size_t row_stride = (size_t)p.n_cells * SAMPLE_BYTES;
    const uint8_t* ptr = static_cast<const uint8_t*>(p.vis) + (size_t)o_local * p.n_int * row_stride
                         + (size_t)g.cell * SAMPLE_BYTES;
    const int o_global = p.o_first + o_local;
    const int blocks_per_win = p.M / R;

    float acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.f;
    uint32_t wt = 0;

    float cur[R][8], nxt[R][8];
#pragma unroll
    for (int r = 0; r < R; ++r) load_sample<FP16, V8>(ptr + (size_t)r * row_stride, cur[r]);
    const int total_blocks = p.n_int / R;
    int blk = 0;

    for (int wl = 0; wl < p.wpo; ++wl) {
        Win w;
        w.reset();
        for (int b = 0; b < blocks_per_win; ++b, ++blk) {
            if (blk + 1 < total_blocks) {
                const uint8_t* np = ptr + (size_t)(blk + 1) * R * row_stride;
#pragma unroll
                for (int r = 0; r < R; ++r) load_sample<FP16, V8>(np + (size_t)r * row_stride, nxt[r]);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int n = b * R + r;
                const float inv_n = (n < kInvNTable) ? c_inv_n[n] : 1.f / (float)(n + 1);
                accumulate(w, cur[r], inv_n);
            }
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int q = 0; q < 8; ++q) cur[r][q] = nxt[r][q];
        }
        float x, r_re, r_im;
        window_stats(w, fM, x, r_re, r_im);
        const bool flag = decide(x, r_re, r_im, p.thr0);
        const int w_global = o_global * p.wpo + wl;
        store_flags(p, g, 0, w_global, flag);
        store_stats(p, g, w_global, p.thr0.c * x, r_re, r_im);
        if (!flag) {
#pragma unroll
            for (int q = 0; q < 8; ++q) acc[q] += w.s[q];
            wt += (uint32_t)p.M;
        }
    }
    store_output(p, g, 0, o_global, acc, wt);
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
// ------------------------------------------------------------------------------------------------
template <int R, bool FP16>
__global__ void __launch_bounds__(512, 1) rfi_tma_kernel(const __grid_constant__ CUtensorMap tmap,
                                                           const KParams p, const int stages) {
    constexpr int ROW_BYTES = FP16 ? 512 : 1024;
    constexpr int STAGE_BYTES = R * ROW_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const uint32_t ring = smem_base + (uint32_t)warp * stages * STAGE_BYTES;
    const uint32_t bars = smem_base + (uint32_t)nwarps * stages * STAGE_BYTES + (uint32_t)warp * stages * 8;

    const int n_tiles = (p.n_cells + 31) >> 5;
    const int n_units = n_tiles * p.n_out_slab;
    const int gw = blockIdx.x * nwarps + warp;
    const int GW = gridDim.x * nwarps;
    if (gw >= n_units) return;                                // warp-private pipeline: safe to leave
    const int my_units = (n_units - 1 - gw) / GW + 1;
    const int bpu = p.n_int / R;                              // blocks (stages) per unit
    const int total = my_units * bpu;
    const int blocks_per_win = p.M / R;
    const float fM = (float)p.M;

    if (lane == 0) {
        for (int s = 0; s < stages; ++s) mbar_init(bars + 8 * s, 1);
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
        if constexpr (FP16) tma_load_2d(dst, &tmap, pr_tile * 128, pr_row0 + pr_blk * R, bar, pol);
        else                tma_load_3d(dst, &tmap, 0, pr_tile * 8, pr_row0 + pr_blk * R, bar, pol);
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
        float acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.f;
        uint32_t wt = 0;

        for (int wl = 0; wl < p.wpo; ++wl) {
            Win w;
            w.reset();
            for (int b = 0; b < blocks_per_win; ++b) {
                mbar_wait(bars + 8 * stage, parity);
                const uint32_t sbase = ring + (uint32_t)stage * STAGE_BYTES;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float v[8];
                    if constexpr (FP16) {
                        half8_to_float(lds128(sbase + r * ROW_BYTES + off0), v);
                    } else {
                        u4x2_to_float(lds128(sbase + r * ROW_BYTES + off0), lds128(sbase + r * ROW_BYTES + off1), v);
                    }
                    const int n = b * R + r;
                    const float inv_n = (n < kInvNTable) ? c_inv_n[n] : 1.f / (float)(n + 1);
                    accumulate(w, v, inv_n);
                }
                __syncwarp();                                  // all lanes have read the stage
                if (lane == 0 && it + stages < total) pr_issue();
                ++it;
                if (++stage == stages) { stage = 0; parity ^= 1u; }
            }
            float x, r_re, r_im;
            window_stats(w, fM, x, r_re, r_im);
            const bool flag = decide(x, r_re, r_im, p.thr0);
            const int w_global = o_global * p.wpo + wl;
            store_flags(p, g, 0, w_global, flag);
            store_stats(p, g, w_global, p.thr0.c * x, r_re, r_im);
            if (!flag) {
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] += w.s[q];
                wt += (uint32_t)p.M;
            }
        }
        store_output(p, g, 0, o_global, acc, wt);
    }
}

}  // namespace rfi
