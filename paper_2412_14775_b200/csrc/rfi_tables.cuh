// rfi_tables.cuh -- the paper-literal mixed-precision arithmetic mode.
//
// Tables 1 and 2 of the paper executed group by group, each of the 14 groups in
// single or half precision as a mask says (a[i] >= 0.5 -> group i in 16 bit).
// This is the arithmetic the paper's reinforcement-learning environment evaluates; the fast kernels
// (rfi_kernels.cuh) compute the same statistics in a reformulated, all-single form.  Same data layout, same
// outputs, same fused structure: one thread per cell, one pass, flags + masked average in the kernel.
//
// Every operation is an IEEE-754 round-to-nearest-even operation of the group's format, never contracted:
// single = __fadd_rn / __fmul_rn / __fdiv_rn / __fsqrt_rn; half = the same on operands converted to half, result
// rounded to half (the correctly rounded half operation: the float result of two half operands carries enough
// bits for the second rounding to be innocuous).  Sums run sequentially in sample order.  The results are
// therefore bit-identical to the step-by-step CPU restatement in oracle/ -- which shares no code with this file.
//
// Mask: bit g-1 = Table 1 group g in half; bit 7+g-1 = Table 2 group g in half (same bits for the real-part and
// the imaginary-part pass).  The kernel takes two compile-time masks: SMASK for the per-sample groups (Table 1
// groups 1-4, Table 2 groups 1-4: where the time goes) and TMASK for the per-window tail (groups 5-7); a negative
// value means "read the bits from the kernel parameters".  Instantiated: all-single <0,0>, the paper's learned
// assignment <0x3C50,0x3C50>, every one of the 256 per-sample assignments with a run-time tail <ps,-1> (so that ANY of
// the 2^14 masks an RL search visits runs at compile-time-mask speed, rfi_launch_tables_ps*.cu), and the fully
// run-time <-1,-1> for odd window lengths.  Block length R = 2 (1 for odd windows): the arithmetic is sequential in the
// samples whatever R is, and the mode is bound by instruction issue, so the registers go to resident warps (24 per SM)
// rather than to bytes in flight.
// Readings T1-T7 of DESIGN.md section 11 (eps = machine epsilon of the group's format, Eq.(4) brackets, ...).
#pragma once

#include "rfi_kernels.cuh"

namespace rfi {

struct Fmt {
    bool half;
    __device__ __forceinline__ float cv(float x) const { return half ? __half2float(__float2half_rn(x)) : x; }
    __device__ __forceinline__ float add(float a, float b) const { return cv(__fadd_rn(cv(a), cv(b))); }
    __device__ __forceinline__ float sub(float a, float b) const { return cv(__fsub_rn(cv(a), cv(b))); }
    __device__ __forceinline__ float mul(float a, float b) const { return cv(__fmul_rn(cv(a), cv(b))); }
    __device__ __forceinline__ float div(float a, float b) const { return cv(__fdiv_rn(cv(a), cv(b))); }
    __device__ __forceinline__ float sqrt(float a) const { return cv(__fsqrt_rn(cv(a))); }
    __device__ __forceinline__ float eps() const { return half ? 9.765625e-4f : 1.1920928955078125e-7f; }   // 2^-10, 2^-23
};

template <int MASK>
__device__ __forceinline__ Fmt table_fmt(uint32_t runtime_mask, int bit) {
    if constexpr (MASK >= 0) return Fmt{((MASK >> bit) & 1) != 0};
    else                     return Fmt{((runtime_mask >> bit) & 1u) != 0};
}

// Running state of one window: Table 1 groups 3-4 and Table 2 group 4 (for both parts), plus the window sum.
struct TabWin {
    float s1, s2;
    float qs[2], us[2], vs[2];
    f2 s[4];
    __device__ __forceinline__ void reset() {
        s1 = s2 = 0.f;
        qs[0] = qs[1] = us[0] = us[1] = vs[0] = vs[1] = 0.f;
#pragma unroll
        for (int p = 0; p < 4; ++p) s[p] = 0ull;
    }
};

// One sample through the per-sample groups (Table 1 groups 1-4, Table 2 groups 1-4).
template <int MASK>
__device__ __forceinline__ void tables_sample(TabWin& w, const f2 (&x)[4], uint32_t mask) {
    float xxr, xxi, xyr, xyi, yxr, yxi, yyr, yyi;
    unpack2(x[0], xxr, xxi);
    unpack2(x[1], xyr, xyi);
    unpack2(x[2], yxr, yxi);
    unpack2(x[3], yyr, yyi);
    // Eq.(2) in single precision (the tables' inputs are single)
    const float Ir = __fadd_rn(xxr, yyr), Ii = __fadd_rn(xxi, yyi);
    const float Q[2] = {__fsub_rn(xxr, yyr), __fsub_rn(xxi, yyi)};
    const float U[2] = {__fadd_rn(xyr, yxr), __fadd_rn(xyi, yxi)};
    const float V[2] = {-__fsub_rn(xyi, yxi), __fsub_rn(xyr, yxr)};          // V = j (xy - yx)
    const Fmt g1 = table_fmt<MASK>(mask, 0), g2 = table_fmt<MASK>(mask, 1);
    const Fmt g3 = table_fmt<MASK>(mask, 2), g4 = table_fmt<MASK>(mask, 3);
    const float y = g1.add(g1.mul(Ir, Ir), g1.mul(Ii, Ii));                  // Table 1 group 1
    const float z = g2.sqrt(y);                                              //         group 2
    w.s1 = g3.add(w.s1, z);                                                  //         group 3
    w.s2 = g4.add(w.s2, y);                                                  //         group 4
    const Fmt d1 = table_fmt<MASK>(mask, 7), d2 = table_fmt<MASK>(mask, 8);
    const Fmt d3 = table_fmt<MASK>(mask, 9), d4 = table_fmt<MASK>(mask, 10);
#pragma unroll
    for (int part = 0; part < 2; ++part) {                                   // real parts, imaginary parts
        const float a = d1.mul(Q[part], Q[part]);                            // Table 2 group 1
        const float b = d1.mul(U[part], U[part]);
        const float c = d1.mul(V[part], V[part]);
        const float p = d2.add(d2.sqrt(d2.add(d2.add(a, b), c)), d2.eps());  //         group 2
        w.qs[part] = d4.add(w.qs[part], d3.div(Q[part], p));                 //         groups 3, 4
        w.us[part] = d4.add(w.us[part], d3.div(U[part], p));
        w.vs[part] = d4.add(w.vs[part], d3.div(V[part], p));
    }
#pragma unroll
    for (int p = 0; p < 4; ++p) w.s[p] = add2(w.s[p], x[p]);
}

// Window tail: Table 1 groups 5-7, Table 2 groups 5-7, decision.
template <int MASK>
__device__ __forceinline__ bool tables_tail(const TabWin& w, const KParams& p, int cls, float& tau, float& r_re, float& r_im) {
    const uint32_t mask = p.arith_mask;
    const float d = cls ? p.d1 : p.d, s_low = cls ? p.s_low1 : p.s_low, s_high = cls ? p.s_high1 : p.s_high;
    const float gamma = cls ? p.thr1.gamma : p.thr0.gamma;
    const Fmt g5 = table_fmt<MASK>(mask, 4), g6 = table_fmt<MASK>(mask, 5), g7 = table_fmt<MASK>(mask, 6);
    const float Wf = (float)p.M;
    tau = g5.div(g5.add(g5.mul(Wf, d), 1.0f), g5.sub(Wf, 1.0f));           // group 5
    const float s12 = g6.mul(w.s1, w.s1);                                    // group 6
    const float ratio = g7.div(g7.mul(Wf, w.s2), g7.add(s12, g7.eps()));     // group 7
    tau = g7.mul(tau, g7.sub(ratio, 1.0f));
    bool keep = (g7.cv(tau) >= g7.cv(s_low)) && (g7.cv(tau) <= g7.cv(s_high));
    const Fmt d5 = table_fmt<MASK>(mask, 11), d6 = table_fmt<MASK>(mask, 12), d7 = table_fmt<MASK>(mask, 13);
    float r[2];
#pragma unroll
    for (int part = 0; part < 2; ++part) {
        const float q2 = d5.mul(w.qs[part], w.qs[part]);                     // group 5
        const float u2 = d5.mul(w.us[part], w.us[part]);
        const float v2 = d5.mul(w.vs[part], w.vs[part]);
        r[part] = d6.div(d6.sqrt(d6.add(d6.add(q2, u2), v2)), Wf);           // group 6
        keep = keep && (d7.cv(r[part]) <= d7.cv(gamma));              // group 7
    }
    r_re = r[0];
    r_im = r[1];
    return !keep;
}

template <int R, int SMASK, int TMASK = SMASK>
__global__ void __launch_bounds__(128, R == 1 ? 8 : (R == 2 ? 6 : 4)) rfi_tables_kernel(const KParams p) {
    const int lane = threadIdx.x & 31;
    const int n_tiles = (p.n_cells + 31) >> 5;
    const int unit = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (unit >= n_tiles * p.n_out_slab) return;
    const int o_local = unit / n_tiles;
    const int tile = unit - o_local * n_tiles;
    const LaneGeom g = lane_geom(p, tile, lane);
    const size_t row_stride = (size_t)p.n_cells * 32;
    const size_t blk_stride = row_stride * R;
    const uint8_t* ptr = static_cast<const uint8_t*>(p.vis) + (size_t)o_local * p.n_int * row_stride + (size_t)g.cell * 32;
    const int o_global = p.o_first + o_local;
    const int bpw = p.M / R;
    const int total = p.n_int / R;
    int w_global = o_global * p.wpo;

    f2 acc[4] = {0ull, 0ull, 0ull, 0ull};
    uint32_t wt = 0;
    TabWin w;
    w.reset();
    int blk = 0, b_in_win = 0;
    Raw<false> A[R], B[R];
    load_block<R, false, false>(ptr, row_stride, A);
    ptr += blk_stride;
    auto step = [&](Raw<false> (&cur)[R], Raw<false> (&nxt)[R]) {
        if (blk + 1 < total) {
            load_block<R, false, false>(ptr, row_stride, nxt);
            ptr += blk_stride;
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            f2 x[4];
            widen(cur[r], x);
            tables_sample<SMASK>(w, x, p.arith_mask);
        }
        ++blk;
        if (++b_in_win == bpw) {
            float tau, r_re, r_im;
            const bool flag = tables_tail<TMASK>(w, p, g.cls, tau, r_re, r_im);
            store_flags(p, g, p.k_first, w_global, flag);
            store_stats(p, g, w_global, tau, r_re, r_im);
            if (!flag) {
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[q] = add2(acc[q], w.s[q]);
                wt += (uint32_t)p.M;
            }
            ++w_global;
            b_in_win = 0;
            w.reset();
        }
    };
    while (blk + 2 <= total) {
        step(A, B);
        step(B, A);
    }
    if (blk < total) step(A, B);
    store_output(p, g, p.k_first, o_global, acc, wt);
}

}  // namespace rfi
