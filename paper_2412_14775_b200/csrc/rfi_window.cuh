// rfi_window.cuh -- per-window state of one cell, the per-block update, the window tail (Eq.(4), Eq.(9),
// decision) and the output stores.  One thread = one cell.  See rfi_common.cuh for the conventions.
#pragma once

#include "rfi_common.cuh"

namespace rfi {

struct Win {
    float mean, m2;            // running mean and centred second moment of z = |I|        (Eq.(3))
    f2 q, u, v;                // sums of unit vectors; lo = real-part triple, hi = imaginary-part triple (Eq.(8))
    f2 s[4];                   // plain sum of the window's samples (for the average)
    __device__ __forceinline__ void reset() {
        mean = m2 = 0.f;
        q = u = v = 0ull;
#pragma unroll
        for (int p = 0; p < 4; ++p) s[p] = 0ull;
    }
};

// One sample: Stokes (Eq.(2)), |I| (Table 1 groups 1-2), unit vectors and their sums (Eq.(6)-(8)), window sum.
// Returns z = |I|.
__device__ __forceinline__ float accumulate_sample(Win& w, const f2 (&x)[4]) {
    // Eq.(2): I = xx+yy, Q = xx-yy, U = xy+yx, V = j(xy-yx).  With D = xy-yx: Re V = -Im D, Im V = Re D.
    // The sign of V cannot change r (it enters through v^2 and (sum v)^2), so the real-part triple is taken
    // as (Re Q, Re U, Im D) and the imaginary-part triple as (Im Q, Im U, Re D): dsw = (Im D, Re D).
    const f2 I = add2(x[0], x[3]);
    const f2 Q = sub2(x[0], x[3]);
    const f2 U = add2(x[1], x[2]);
    float xyr, xyi, yxr, yxi;
    unpack2(x[1], xyr, xyi);
    unpack2(x[2], yxr, yxi);
    const f2 dsw = pack2(xyi - yxi, xyr - yxr);
    float Ir, Ii;
    unpack2(I, Ir, Ii);
    const float y = fmaf(Ir, Ir, Ii * Ii);                    // |I|^2
    const float z = sqrt_approx(y);                           // |I|
    // p^2 for both triples at once: lo = Qr^2+Ur^2+Di^2, hi = Qi^2+Ui^2+Dr^2            (Eq.(6))
    const f2 p2 = fma2(dsw, dsw, fma2(U, U, mul2(Q, Q)));
    float p2r, p2i;
    unpack2(p2, p2r, p2i);
    // exact-zero guard: p = 0 means q = u = v = 0, and 0 * rsqrt(FLT_MIN) = 0
    const f2 inv = pack2(rsqrt_approx(fmaxf(p2r, 1.17549435e-38f)), rsqrt_approx(fmaxf(p2i, 1.17549435e-38f)));
    w.q = fma2(Q, inv, w.q);                                  // Eq.(7)-(8)
    w.u = fma2(U, inv, w.u);
    w.v = fma2(dsw, inv, w.v);
#pragma unroll
    for (int p = 0; p < 4; ++p) w.s[p] = add2(w.s[p], x[p]);
    return z;
}

// R samples (one block) of the window; `blk` = index of the block inside the window (0-based).
// Merge of (n_a = blk*R, mean, m2) with the block's (R, mb, m2b):
//   delta = mb - mean;  mean += delta/(blk+1);  m2 += m2b + delta^2 * R*blk/(blk+1)
// The two halves are separate functions because the split kernel (rfi_split.cuh) computes the block statistics on one
// warp and merges them, in block order, on another: same operations in the same order, hence the same bits.
template <int R>
__device__ __forceinline__ void block_stats(const float (&z)[R], float& mb, float& m2b) {
    float zs = z[0];
#pragma unroll
    for (int r = 1; r < R; ++r) zs += z[r];
    mb = zs * (1.0f / R);
    m2b = 0.f;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const float dz = z[r] - mb;
        m2b = fmaf(dz, dz, m2b);
    }
}
template <int R>
__device__ __forceinline__ void merge_stats(Win& w, float mb, float m2b, int blk) {
    const float fb = (float)blk;
    const float wgt = rcp_approx(fb + 1.0f);                  // 1/(blk+1); blk = 0 -> exactly 1
    const float delta = mb - w.mean;
    w.mean = fmaf(delta, wgt, w.mean);
    w.m2 += fmaf(delta * delta, (float)R * fb * wgt, m2b);
}
template <int R>
__device__ __forceinline__ void merge_block(Win& w, const float (&z)[R], int blk) {
    float mb, m2b;
    block_stats<R>(z, mb, m2b);
    merge_stats<R>(w, mb, m2b, blk);
}

template <int R, bool FP16>
__device__ __forceinline__ void accumulate_block(Win& w, const Raw<FP16> (&raw)[R], int blk) {
    float z[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        f2 x[4];
        widen(raw[r], x);
        z[r] = accumulate_sample(w, x);
    }
    merge_block<R>(w, z, blk);
}

// sqrt(s) for s >= 0 from the hardware rsqrt plus one Newton step on the residual s - r^2 (an fma, exact):
// correctly rounded in practice and exact whenever sqrt(s) is representable (ties of Eq.(10) at r = k/W).
__device__ __forceinline__ float sqrt_refined(float s) {
    const float y0 = rsqrt_approx(fmaxf(s, 1.17549435e-38f));
    const float r0 = s * y0;
    return fmaf(fmaf(-r0, r0, s), 0.5f * y0, r0);
}

// T x F footprints (W = T * F): the F channels of a window are F adjacent lanes (F a power of two,
// groups lane-aligned because n_chan % F == 0 and F | 32).  Each lane arrives with the moments of its own T
// samples; a butterfly over the group merges them (equal counts: mean = (a+b)/2, m2 = m2a + m2b + delta^2 n/2)
// and adds the unit-vector sums.  Every operation is symmetric in the two partners, so all lanes of a group end
// with bit-identical statistics and hence the same flag.  The per-channel sample sums w.s stay per lane.
__device__ __forceinline__ f2 shfl_xor_f2(f2 v, int m) {
    return (f2)__shfl_xor_sync(0xffffffffu, (unsigned long long)v, m);
}
__device__ __forceinline__ void combine_group(Win& w, int F, int T) {
    float n = (float)T;                                       // samples behind each partner's moments
    for (int m = 1; m < F; m <<= 1, n += n) {
        const float mean_o = __shfl_xor_sync(0xffffffffu, w.mean, m);
        const float m2_o = __shfl_xor_sync(0xffffffffu, w.m2, m);
        const float delta = mean_o - w.mean;
        w.m2 = fmaf(delta * delta, 0.5f * n, w.m2 + m2_o);
        w.mean = 0.5f * (w.mean + mean_o);
        w.q = add2(w.q, shfl_xor_f2(w.q, m));
        w.u = add2(w.u, shfl_xor_f2(w.u, m));
        w.v = add2(w.v, shfl_xor_f2(w.v, m));
    }
}

// Window tail: Eq.(4) in centred form and Eq.(9).  x = W*S2/S1^2 - 1 = m2/(W mean^2); tau = c * x.
__device__ __forceinline__ void window_stats(const Win& w, float inv_M, float& x, float& r_re, float& r_im) {
    // all-zero window: S1 = 0 -> x = -1 (the eps -> 0 limit of Table 1 row 7).  (m2/mean)/(W mean) keeps the
    // intermediate values in range for small amplitudes (no mean^2).
    const float t = rcp_approx(w.mean);
    x = (w.mean == 0.f) ? -1.f : (w.m2 * t) * (t * inv_M);
    float qr, qi, ur, ui, vr, vi;
    unpack2(w.q, qr, qi);
    unpack2(w.u, ur, ui);
    unpack2(w.v, vr, vi);
    r_re = sqrt_refined(fmaf(qr, qr, fmaf(ur, ur, vr * vr))) * inv_M;
    r_im = sqrt_refined(fmaf(qi, qi, fmaf(ui, ui, vi * vi))) * inv_M;
}

// Eq.(5), Eq.(10), OR-combined; negated so that NaN flags.  tau = c x with c > 0, so
// tau < s_low <=> x < s_low / c: the thresholds arrive divided by c (one division on the host per set), and
// r_re > gamma OR r_im > gamma <=> max(r_re, r_im) > gamma (NaN-propagating max).  Every kernel decides here.
__device__ __forceinline__ bool decide(float x, float r_max, const Thr& t) {
    return !(x >= t.x_low && x <= t.x_high && r_max <= t.gamma);
}

// Per-unit lane geometry: which cell, which flag word / bit.
struct LaneGeom {
    int cell;          // clamped to a valid cell for loads
    bool valid;
    int word;          // b * wpb + c/32
    int bit;           // c % 32
    unsigned group;    // lanes of this warp that share `word`
    int cls;           // threshold class of the lane's baseline (0/1)
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
    g.cls = p.cls ? (int)p.cls[p.b_first + b] : 0;
    g.group = __match_any_sync(0xffffffffu, g.word);
    g.leader = g.valid && ((__ffs(g.group) - 1) == lane);
    return g;
}

// Pack the warp's flag bits into the mask (layout in include/rfi.h).  k = global set index.
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
                                             const f2 (&acc)[4], uint32_t wt) {
    if (!g.valid) return;
    const size_t oi = ((size_t)k * p.n_out_total + o_global) * p.n_cells + g.cell;
    float a[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) unpack2(acc[i], a[2 * i], a[2 * i + 1]);
    float4 lo, hi;
    if (wt) {
        const float iw = 1.0f / (float)wt;                      // one IEEE division, then 8 multiplies (<= 1.5 ulp)
        lo = make_float4(a[0] * iw, a[1] * iw, a[2] * iw, a[3] * iw);
        hi = make_float4(a[4] * iw, a[5] * iw, a[6] * iw, a[7] * iw);
    } else {
        lo = hi = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float4* dst = reinterpret_cast<float4*>(p.avg + oi * 8);
    // Outputs are written once and not read again by this pass: no L1 allocation, evict-first in L2 (measured with a
    // zero-compute probe of the K = 64 traffic mix: 2.90 -> 2.81 ms).  Aligned rows leave as one 256-bit store, i.e. the
    // cell's 32-byte sector whole.
    if ((reinterpret_cast<uintptr_t>(dst) & 31u) == 0) {
        asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(dst), "f"(lo.x),
                     "f"(lo.y), "f"(lo.z), "f"(lo.w), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w) : "memory");
    } else {
        dst[0] = lo;
        dst[1] = hi;
    }
    asm volatile("st.global.cs.u32 [%0], %1;" ::"l"(p.weight + oi), "r"(wt) : "memory");
}

// Single-set window tail shared by the streaming kernels: statistics, decision, flag word, statistics planes,
// masked accumulation into the output integration.  ADAPT: the thresholds come from device memory
// (`thr`: the lane's class, ADAPT = 1, or the lane's baseline stream, ADAPT = 2, 3) and, for ADAPT = 1, 2, the window's tau
// and max(r_re, r_im) are counted in a shared-memory histogram (the CTA's per-class pair, or the warp's own for its stream).
// ADAPT = 3: static per-stream thresholds (rfi_plan_set_stream_thresholds), nothing counted.
template <int ADAPT = 0>
__device__ __forceinline__ void finish_window(const KParams& p, const LaneGeom& g, Win& w, float inv_W,
                                              int w_global, f2 (&acc)[4], uint32_t& wt,
                                              const Thr* thr = nullptr, uint32_t* sh_hist = nullptr) {
    float x, r_re, r_im;
    if (p.F > 1) combine_group(w, p.F, p.M);
    window_stats(w, inv_W, x, r_re, r_im);
    const Thr& t = ADAPT ? *thr : (g.cls ? p.thr1 : p.thr0);  // per-baseline-class thresholds (cross / auto)
    const float r_max = max_nan(r_re, r_im);
    const bool flag = decide(x, r_max, t);
    const float tau = t.c * x;
    store_flags(p, g, p.k_first, w_global, flag);
    store_stats(p, g, w_global, tau, r_re, r_im);
    if constexpr (ADAPT == 1 || ADAPT == 2) {
        if (g.valid && fabsf(tau) <= 3.402823466e38f && fabsf(r_max) <= 3.402823466e38f) {   // finite statistics only
            uint32_t* h = sh_hist + (ADAPT == 1 ? g.cls * kAdaptBins : 0);   // per class: the CTA's; per stream: the warp's own
            atomicAdd(h + adapt_bin(tau, kAdaptTauLoExp, kAdaptTauBins), 1u);
            atomicAdd(h + kAdaptTauBins + adapt_bin(r_max, kAdaptRLoExp, kAdaptRBins), 1u);
        }
    }
    if (!flag) {
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[q] = add2(acc[q], w.s[q]);
        wt += (uint32_t)p.M;
    }
}

}  // namespace rfi
