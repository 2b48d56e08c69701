// rfi_common.cuh -- sm_100a device helpers shared by the kernels of the fused flag-and-average pass:
// PTX wrappers (packed f32x2 arithmetic, streaming loads, mbarrier/TMA), the per-sample moment
// accumulation, the window tail and the output stores.
//
// What is computed is defined in include/rfi.h (equations of PAPER.md cited there).  This file is
// the product path: it shares nothing with oracle/.
//
// Mapping used by every kernel: one thread = one (baseline, channel) cell, a warp = 32 consecutive
// cells.  With the time-slowest layout a warp's row of one time step is 1 KiB (fp32) / 512 B (fp16)
// contiguous, so every global access is a whole-line, fully used request.  Statistics never cross
// lanes; the only warp collective is the ballot that packs the flag bits.
//
// Arithmetic is fp32.  Pairs (re, im) are kept in 64-bit registers and processed with the
// Blackwell packed instructions FADD2 / FMUL2 / FFMA2 (PTX add/mul/fma.rn.f32x2), which halves the
// issue slots of the Stokes formation (Eq.(2)), the unit-vector sums (Eq.(8)) and the window sums.
//
// SK in centred form: Eq.(4)'s  W*S2/S1^2 - 1  equals  sum (z_i - zbar)^2 / (W zbar^2), z_i = |I_i|.
// The centred second moment is built block-wise (R samples at a time: block mean, block centred
// moment, then the pairwise merge of Chan et al.), which has none of the cancellation of the raw-moment
// form in fp32 and no per-sample dependent chain.
#pragma once

#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace rfi {

typedef unsigned long long f2;                    // two packed floats {lo = re, hi = im}

struct Thr {                                      // one threshold set, device form
    float c;                                      // (W d + 1)/(W - 1), Eq.(4) prefactor: tau = c * x
    float x_low, x_high;                          // s_low / c, s_high / c: Eq.(5) decided on x = W S2/S1^2 - 1
    float gamma;                                  // Eq.(10)
};

constexpr int kMaxBatch = 64;                     // threshold sets evaluated by one batched launch

struct KParams {
    const void* vis;          // slab base: [rows][n_cells] samples
    float* avg;               // [K][n_out_total][n_cells][8]
    uint32_t* weight;         // [K][n_out_total][n_cells]
    float* stats;             // [3][n_win_total][n_cells] or nullptr
    uint32_t* flags;          // [K][n_win_total][n_baselines*wpb]
    Thr thr0;                 // set 0, baseline class 0 (single-set kernels; stats use its c)
    Thr thr1;                 // set 0, baseline class 1 (= thr0 when the plan has one class)
    const uint8_t* cls;       // [n_baselines of the whole array] class of each baseline (0/1), or nullptr: all class 0
    int b_first;              // first baseline of this plan's shard (index into cls)
    int n_cells, n_chan, n_baselines, wpb;
    int M, n_int, wpo;        // window length in time (T), samples per output, windows per output
    int F;                    // window extent in frequency: F adjacent channels (lanes), power of two <= 32
    float inv_W;              // 1 / (T * F), W of Eq.(4) and Eq.(9)
    int n_out_slab;           // outputs contained in this slab
    int o_first;              // global index of the slab's first output
    int n_out_total, n_win_total;
    int K;                    // sets handled by this launch (batched kernel: <= kMaxBatch)
    int k_first;              // global index of this launch's first set
    int flags_atomic;         // 1: flag words may be shared between warps -> atomicOr into a zeroed buffer
    // on-line threshold adaptation (rfi_plan_set_adaptive; rfi_adapt.cu): thresholds of the two classes in device memory
    // (updated between chunks by a device kernel) and this chunk's histograms of tau and max(r_re, r_im); null otherwise
    const Thr* d_thr;
    uint32_t* hist;
    int adapt_streams;        // 0: thresholds / histograms per baseline class ([2]); 1: per baseline stream ([n_baselines]);
                              // 2: per-stream thresholds given by the caller, no adaptation
    // in-kernel confusion counters (rfi_plan_set_truth; K-set kernel only): ground-truth mask laid out like one set of the
    // flag mask, and uint64 counts[K][4] = {false alarms, clean windows, missed detections, RFI windows}; null otherwise
    const uint32_t* truth;
    unsigned long long* counts;
    // paper-literal tables mode (rfi_tables.cuh) only: raw thresholds of set 0 and the 14-bit precision mask
    float d, s_low, s_high;
    float d1, s_low1, s_high1;   // class 1
    uint32_t arith_mask;
};

// Histogram bins of the adaptation (reading A2): geometric, 64 linear sub-bins per octave, read
// off the float's bit pattern; tau in [2^-8, 2^4) -> 768 bins, max(r_re, r_im) in [2^-6, 1) -> 384 bins.
constexpr int kAdaptTauBins = 768, kAdaptRBins = 384, kAdaptBins = kAdaptTauBins + kAdaptRBins;
constexpr int kAdaptTauLoExp = -8, kAdaptRLoExp = -6;
__device__ __forceinline__ int adapt_bin(float v, int lo_exp, int n_bins) {
    if (!(v > 0.f)) return 0;                                 // zero and negative values: first bin (NaN is never binned)
    const int idx = (int)(__float_as_uint(v) >> 17) - ((127 + lo_exp) << 6);
    return min(max(idx, 0), n_bins - 1);
}

struct BatchThr { Thr t[kMaxBatch]; Thr t1[kMaxBatch]; };   // by-value kernel parameter (constant bank), 2 KiB: class 0, class 1

// ------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ f2 pack2(float lo, float hi) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { f2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
    f2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
// max that returns NaN if either operand is NaN (so that a NaN statistic still flags, reading G6)
__device__ __forceinline__ float max_nan(float a, float b) { float r; asm("max.NaN.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// One 4-pol sample in registers as it sits in memory: fp32 -> 4 x (re,im) pairs, fp16 -> 4 x half2.
template <bool FP16> struct Raw;
template <> struct Raw<false> { f2 p[4]; };
template <> struct Raw<true> { uint32_t p[4]; };

// Streaming global loads: read-once data, not allocated in L1 (and evict-first in L2 where PTX allows the
// qualifier, i.e. on the 256-bit form).
__device__ __forceinline__ void ldg_stream(const void* ptr, Raw<false>& r) {      // one 256-bit request
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v4.b64 {%0,%1,%2,%3}, [%4];"
                 : "=l"(r.p[0]), "=l"(r.p[1]), "=l"(r.p[2]), "=l"(r.p[3]) : "l"(ptr));
}
__device__ __forceinline__ void ldg_stream_16B(const void* ptr, Raw<false>& r) {  // 16-byte-aligned base only
    asm volatile("ld.global.nc.L1::no_allocate.v2.b64 {%0,%1}, [%2];"
                 : "=l"(r.p[0]), "=l"(r.p[1]) : "l"(ptr));
    asm volatile("ld.global.nc.L1::no_allocate.v2.b64 {%0,%1}, [%2+16];"
                 : "=l"(r.p[2]), "=l"(r.p[3]) : "l"(ptr));
}
__device__ __forceinline__ void ldg_stream(const void* ptr, Raw<true>& r) {       // one 128-bit request
    asm volatile("ld.global.nc.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.p[0]), "=r"(r.p[1]), "=r"(r.p[2]), "=r"(r.p[3]) : "l"(ptr));
}
__device__ __forceinline__ void lds_raw(uint32_t a0, uint32_t a1, Raw<false>& r) {
    asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(r.p[0]), "=l"(r.p[1]) : "r"(a0));
    asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(r.p[2]), "=l"(r.p[3]) : "r"(a1));
}
__device__ __forceinline__ void lds_raw(uint32_t a0, uint32_t, Raw<true>& r) {
    asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r.p[0]), "=r"(r.p[1]), "=r"(r.p[2]), "=r"(r.p[3]) : "r"(a0));
}

// Stage reuse (a stage is read by the generic proxy, then overwritten by the async proxy).  The hand-off is an
// explicit consumer -> producer barrier per stage (an "empty" mbarrier, count 32): every lane arrives right after its
// own shared-memory loads of the stage -- mbarrier.arrive.release orders the lane's reads before the arrival (in
// hardware the LDS and the SYNCS.ARRIVE go through the same in-order shared-memory pipe, so the stage has been read
// when the arrival is performed) -- the producer lane waits for all 32 arrivals (acquire), orders generic-proxy reads
// before the async-proxy write with fence.proxy.async (SASS: MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC) and only then issues
// the TMA refill.  Refilling BEFORE the arithmetic on the loaded registers keeps a whole block time of prefetch lead:
// with two stages per warp (all the K-set kernel has room for) arriving after accumulate_block measured 5 % slower.
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Widen one sample to four fp32 (re,im) pairs: xx, xy, yx, yy (row-major Eq.(1)).
__device__ __forceinline__ void widen(const Raw<false>& r, f2 (&x)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) x[i] = r.p[i];
}
__device__ __forceinline__ void widen(const Raw<true>& r, f2 (&x)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&r.p[i]));   // exact
        x[i] = pack2(f.x, f.y);
    }
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

}  // namespace rfi
