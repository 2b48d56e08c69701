// rfi_rl.cu -- the reinforcement-learning ENVIRONMENT of the paper's section 3 as one kernel
// launch: B windows x one 14-bit precision mask -> per window the 45-value state (10 data features, 14 precision
// bits, 21 per-group errors against double precision), the operation + conversion cost, the overflow / underflow
// events, the agreement of the three flags with the double-precision flags and the reward (rfi_rl_evaluate,
// include/rfi.h).  An external SAC loop (host side, out of scope) calls this once per step for its whole batch.
//
// One thread = one window: the tables' sums run sequentially in sample order (reading T4), every operation is an
// IEEE round-to-nearest operation of its group's format (never contracted), the ground truth runs the same tables
// with every operation in double.  Readings T10-T15: include/rfi.h and DESIGN.md section 11.  Not bandwidth-critical
// (a window is 32 W bytes and costs ~40 W double-precision operations): one pass, everything in registers/local memory.
#include "rfi_internal.h"

#include <cuda_fp16.h>

namespace rfi {

constexpr int kRlRec = RFI_RL_RECORD_DOUBLES;

struct RlEvents { double over, under; };

// One format (single or half, run-time) with overflow / underflow detection (T13): `exact` is the operation carried
// out in double on the already converted operands.
struct RlFmt {
    bool half;
    RlEvents* ev;
    __device__ __forceinline__ double min_normal() const { return half ? 6.103515625e-05 : 1.17549435082228750797e-38; }
    __device__ __forceinline__ float to_half(float x) const { return __half2float(__float2half_rn(x)); }
    __device__ __forceinline__ float round(double exact, float r) const {
        if (isfinite(exact) && !isfinite(r)) ev->over += 1.0;
        else if (exact != 0.0 && fabs((double)r) < min_normal()) ev->under += 1.0;
        return r;
    }
    __device__ __forceinline__ float cv(float x) const {
        if (!half) return x;
        const float r = to_half(x);
        if (r != x && !(isnan(r) && isnan(x))) {
            if (isfinite(x) && !isfinite(r)) ev->over += 1.0;
            else if (x != 0.0f && fabs((double)r) < min_normal()) ev->under += 1.0;
        }
        return r;
    }
    __device__ __forceinline__ float fin(float native) const { return half ? to_half(native) : native; }
    __device__ __forceinline__ float add(float a, float b) const { a = cv(a); b = cv(b); return round((double)a + (double)b, fin(__fadd_rn(a, b))); }
    __device__ __forceinline__ float sub(float a, float b) const { a = cv(a); b = cv(b); return round((double)a - (double)b, fin(__fsub_rn(a, b))); }
    __device__ __forceinline__ float mul(float a, float b) const { a = cv(a); b = cv(b); return round((double)a * (double)b, fin(__fmul_rn(a, b))); }
    __device__ __forceinline__ float div(float a, float b) const { a = cv(a); b = cv(b); return round((double)a / (double)b, fin(__fdiv_rn(a, b))); }
    __device__ __forceinline__ float sqrt(float a) const { a = cv(a); return round(::sqrt((double)a), fin(__fsqrt_rn(a))); }
    __device__ __forceinline__ float eps() const { return half ? 9.765625e-4f : 1.1920928955078125e-7f; }
};

// running mean-absolute-error of one group's outputs; +inf once a non-finite value was seen (T11)
struct RlErr {
    double sum; bool bad;
    __device__ __forceinline__ void reset() { sum = 0.0; bad = false; }
    __device__ __forceinline__ void add(float mixed, double truth) {
        if (!isfinite(mixed) || !isfinite(truth)) bad = true;
        else sum += fabs((double)mixed - truth);
    }
    __device__ __forceinline__ double mean(int n) const { return bad ? __longlong_as_double(0x7ff0000000000000ll) : sum / n; }
};

__device__ __forceinline__ void rl_cost(uint32_t mask, int W, double& op_cost, double& conv) {
    auto C = [&](int bit) { return ((mask >> bit) & 1u) ? 0.6 : 1.0; };
    auto h = [&](int bit) { return (int)((mask >> bit) & 1u); };
    const double w = W;
    const double t1 = 3 * w * C(0) + w * C(1) + w * C(2) + w * C(3) + 1 * C(4) + 1 * C(5) + 3 * C(6);            // T10
    const double t2 = 3 * w * C(7) + w * C(8) + 3 * w * C(9) + 3 * w * C(10) + 3 * C(11) + 4 * C(12) + 1 * C(13);
    op_cost = t1 + 2 * t2;
    double c1 = 0, c2 = 0;                                                                                        // T12
    c1 += h(0) ? 2 * w : 0;  c1 += (h(0) != h(1)) ? w : 0;  c1 += (h(0) != h(3)) ? w : 0;  c1 += (h(1) != h(2)) ? w : 0;
    c1 += (h(2) != h(5)) ? 1 : 0;  c1 += (h(3) != h(6)) ? 1 : 0;  c1 += (h(4) != h(6)) ? 1 : 0;  c1 += (h(5) != h(6)) ? 1 : 0;
    c2 += h(7) ? 3 * w : 0;  c2 += (h(7) != h(8)) ? 3 * w : 0;  c2 += h(9) ? 3 * w : 0;  c2 += (h(8) != h(9)) ? w : 0;
    c2 += (h(9) != h(10)) ? 3 * w : 0;  c2 += (h(10) != h(11)) ? 3 : 0;  c2 += (h(11) != h(12)) ? 3 : 0;  c2 += (h(12) != h(13)) ? 1 : 0;
    conv = c1 + 2 * c2;
}

__global__ void __launch_bounds__(128) rfi_rl_kernel(const float* __restrict__ win, long long n_windows, int W, uint32_t mask_all,
                                                     const uint16_t* __restrict__ masks,
                                                     float d, float s_low, float s_high, float gamma, double rho,
                                                     double* __restrict__ out) {
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_windows) return;
    const uint32_t mask = masks ? (uint32_t)masks[n] & 0x3FFFu : mask_all;      // one action per window, or one for the batch
    const float4* x = reinterpret_cast<const float4*>(win + n * W * 8);
    double* o = out + n * kRlRec;
    RlEvents ev{0.0, 0.0};
    auto F = [&](int bit) { return RlFmt{((mask >> bit) & 1u) != 0, &ev}; };
    const float Wf = (float)W;
    const double Wd = W;
    const double eps_d = 2.220446049250313e-16;                                // machine epsilon of double (T2, T15)

    // ---- features (T15) and Table 1, one pass over the samples ----
    double m[2][5] = {{0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};
    int flags_mixed = 0, flags_dbl = 0;
    {
        const RlFmt g1 = F(0), g2 = F(1), g3 = F(2), g4 = F(3), g5 = F(4), g6 = F(5), g7 = F(6);
        RlErr e1, e2; e1.reset(); e2.reset();
        float s1 = 0.f, s2 = 0.f; double s1d = 0.0, s2d = 0.0;
        for (int i = 0; i < W; ++i) {
            const float4 lo = x[2 * i], hi = x[2 * i + 1];                     // xx, xy | yx, yy as (re, im)
            const float S[2][4] = {{__fadd_rn(lo.x, hi.z), __fsub_rn(lo.x, hi.z), __fadd_rn(lo.z, hi.x), -__fsub_rn(lo.w, hi.y)},
                                   {__fadd_rn(lo.y, hi.w), __fsub_rn(lo.y, hi.w), __fadd_rn(lo.w, hi.y), __fsub_rn(lo.z, hi.x)}};
#pragma unroll
            for (int part = 0; part < 2; ++part) {
                const double I = S[part][0], Q = S[part][1], U = S[part][2], V = S[part][3];
                m[part][0] += I * I; m[part][1] += I * I * I * I; m[part][2] += Q * Q; m[part][3] += U * U; m[part][4] += V * V;
            }
            const float xr = S[0][0], xi = S[1][0];
            const float y = g1.add(g1.mul(xr, xr), g1.mul(xi, xi));            // Table 1 group 1
            const float z = g2.sqrt(y);                                        //         group 2
            s1 = g3.add(s1, z);                                                //         group 3
            s2 = g4.add(s2, y);                                                //         group 4
            const double yd = (double)xr * xr + (double)xi * xi, zd = ::sqrt(yd);
            s1d += zd; s2d += yd;
            e1.add(y, yd); e2.add(z, zd);
        }
        const float pre = g5.div(g5.add(g5.mul(Wf, d), 1.0f), g5.sub(Wf, 1.0f));     // group 5
        const float s12 = g6.mul(s1, s1);                                            // group 6
        const float ratio = g7.div(g7.mul(Wf, s2), g7.add(s12, g7.eps()));           // group 7
        const float tau = g7.mul(pre, g7.sub(ratio, 1.0f));
        const bool ok = (g7.cv(tau) >= g7.cv(s_low)) && (g7.cv(tau) <= g7.cv(s_high));
        const double pred = (Wd * (double)d + 1.0) / (Wd - 1.0);
        const double s12d = s1d * s1d;
        const double taud = pred * (Wd * s2d / (s12d + eps_d) - 1.0);
        const bool okd = (taud >= (double)s_low) && (taud <= (double)s_high);
        flags_mixed |= ok ? 0 : 1; flags_dbl |= okd ? 0 : 1;
        RlErr e;
        o[24] = e1.mean(W); o[25] = e2.mean(W);
        e.reset(); e.add(s1, s1d); o[26] = e.mean(1);
        e.reset(); e.add(s2, s2d); o[27] = e.mean(1);
        e.reset(); e.add(pre, pred); o[28] = e.mean(1);
        e.reset(); e.add(s12, s12d); o[29] = e.mean(1);
        e.reset(); e.add(tau, taud); o[30] = e.mean(1);
    }
#pragma unroll
    for (int part = 0; part < 2; ++part)
#pragma unroll
        for (int k = 0; k < 5; ++k) o[part * 5 + k] = log(m[part][k]) / Wd;
    for (int b = 0; b < 14; ++b) o[10 + b] = (double)((mask >> b) & 1u);

    // ---- Table 2: real parts, then imaginary parts ----
    for (int part = 0; part < 2; ++part) {
        const RlFmt g1 = F(7), g2 = F(8), g3 = F(9), g4 = F(10), g5 = F(11), g6 = F(12), g7 = F(13);
        RlErr e1, e2, e3; e1.reset(); e2.reset(); e3.reset();
        float sum[3] = {0.f, 0.f, 0.f}; double sumd[3] = {0.0, 0.0, 0.0};
        for (int i = 0; i < W; ++i) {
            const float4 lo = x[2 * i], hi = x[2 * i + 1];
            float q, u, v;
            if (part == 0) { q = __fsub_rn(lo.x, hi.z); u = __fadd_rn(lo.z, hi.x); v = -__fsub_rn(lo.w, hi.y); }
            else           { q = __fsub_rn(lo.y, hi.w); u = __fadd_rn(lo.w, hi.y); v = __fsub_rn(lo.z, hi.x); }
            const float a = g1.mul(q, q), b = g1.mul(u, u), c = g1.mul(v, v);              // group 1
            const float p = g2.add(g2.sqrt(g2.add(g2.add(a, b), c)), g2.eps());            // group 2
            const float qh = g3.div(q, p), uh = g3.div(u, p), vh = g3.div(v, p);           // group 3
            sum[0] = g4.add(sum[0], qh); sum[1] = g4.add(sum[1], uh); sum[2] = g4.add(sum[2], vh);   // group 4
            const double ad = (double)q * q, bd = (double)u * u, cd = (double)v * v;
            const double pd = ::sqrt(ad + bd + cd) + eps_d;
            const double qd = q / pd, ud = u / pd, vd = v / pd;
            sumd[0] += qd; sumd[1] += ud; sumd[2] += vd;
            e1.add(a, ad); e1.add(b, bd); e1.add(c, cd);
            e2.add(p, pd);
            e3.add(qh, qd); e3.add(uh, ud); e3.add(vh, vd);
        }
        float sq[3]; double sqd[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) { sq[k] = g5.mul(sum[k], sum[k]); sqd[k] = sumd[k] * sumd[k]; }      // group 5
        const float r = g6.div(g6.sqrt(g6.add(g6.add(sq[0], sq[1]), sq[2])), Wf);                        // group 6
        const double rd = ::sqrt(sqd[0] + sqd[1] + sqd[2]) / Wd;
        const bool ok = g7.cv(r) <= g7.cv(gamma);                                                        // group 7
        const bool okd = rd <= (double)gamma;
        flags_mixed |= ok ? 0 : (2 << part); flags_dbl |= okd ? 0 : (2 << part);
        double* e = o + 31 + 7 * part;
        RlErr t;
        e[0] = e1.mean(3 * W); e[1] = e2.mean(W); e[2] = e3.mean(3 * W);
        t.reset(); for (int k = 0; k < 3; ++k) t.add(sum[k], sumd[k]); e[3] = t.mean(3);
        t.reset(); for (int k = 0; k < 3; ++k) t.add(sq[k], sqd[k]); e[4] = t.mean(3);
        t.reset(); t.add(r, rd); e[5] = t.mean(1);
        e[6] = (ok == okd) ? 0.0 : 1.0;
    }
    int match = 0;
#pragma unroll
    for (int b = 0; b < 3; ++b) match += (((flags_mixed >> b) & 1) == ((flags_dbl >> b) & 1)) ? 1 : 0;
    double op_cost, conv;
    rl_cost(mask, W, op_cost, conv);
    o[45] = op_cost; o[46] = conv; o[47] = ev.over; o[48] = ev.under; o[49] = (double)match;
    o[50] = rho * match - op_cost - 0.3 * conv - ((ev.over + ev.under) > 0.0 ? 20.0 : 0.0);              // T14
    o[51] = (double)(flags_mixed + 8 * flags_dbl);
}

}  // namespace rfi

namespace {
int rl_launch(const float* d_windows, int64_t n_windows, int W, uint32_t mask14, const uint16_t* d_masks,
              const rfi_thresholds* h_thr, double reward_per_match, double* d_out, void* cuda_stream, const char* who) {
    using namespace rfi_host;
    g_cuda_err[0] = 0;
    if (!d_windows || !d_out || !h_thr || n_windows < 0 || W < 2 || (mask14 >> 14) != 0 ||
        reinterpret_cast<uintptr_t>(d_windows) % 16 || reinterpret_cast<uintptr_t>(d_out) % 8 ||
        reinterpret_cast<uintptr_t>(d_masks) % 2) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: NULL / misaligned pointer, W < 2 or mask bits above 13", who);
        return RFI_EINVAL;
    }
    if (!(h_thr->d > 0.f)) return RFI_EINVAL;
    if (n_windows == 0) return RFI_OK;
    const unsigned grid = (unsigned)((n_windows + 127) / 128);
    rfi::rfi_rl_kernel<<<grid, 128, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        d_windows, (long long)n_windows, W, mask14, d_masks, h_thr->d, h_thr->s_low, h_thr->s_high, h_thr->gamma,
        reward_per_match, d_out);
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}
}  // namespace

extern "C" int rfi_rl_evaluate(const float* d_windows, int64_t n_windows, int W, uint32_t mask14,
                               const rfi_thresholds* h_thr, double reward_per_match, double* d_out, void* cuda_stream) {
    return rl_launch(d_windows, n_windows, W, mask14, nullptr, h_thr, reward_per_match, d_out, cuda_stream, "rfi_rl_evaluate");
}

extern "C" int rfi_rl_evaluate_masks(const float* d_windows, int64_t n_windows, int W, const uint16_t* d_masks,
                                     const rfi_thresholds* h_thr, double reward_per_match, double* d_out, void* cuda_stream) {
    if (!d_masks) return RFI_EINVAL;
    return rl_launch(d_windows, n_windows, W, 0u, d_masks, h_thr, reward_per_match, d_out, cuda_stream, "rfi_rl_evaluate_masks");
}
