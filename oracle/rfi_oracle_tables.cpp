// rfi_oracle_tables.cpp -- CPU ORACLE for the paper-literal mixed-precision arithmetic mode:
// Tables 1 and 2 of arxiv 2412.14775 executed group by group, each group in
// single (32 bit) or half (16 bit) precision as a 14-bit mask says.
//
// THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as rfi_oracle.cpp: only tests/, smoke() and
// bench.py's oracle legs may use it; it shares nothing with the CUDA path).
//
// Here the paper FIXES the precision (that is the whole point of its section 3), so this oracle is not fp64:
// it follows the tables step by step, in the paper's order and variable names, every operation an IEEE-754
// round-to-nearest-even operation of the group's format.  A half-precision operation is carried out as
//     round_to_half( float_op( operands converted to half ) )
// which IS the correctly rounded half operation for + - * / sqrt (the float result of two half operands
// carries >= 2*11+2 significand bits, so the second rounding is innocuous).  Values are held in `float`
// variables; a value produced by a half group is exactly representable in half.  "Type conversion"
// = the rounding of an operand into the precision of the group that consumes it.
//
// Mask: bit g-1 (g = 1..7) = Table 1 group g in half precision; bit 7+g-1 = Table 2 group g in half precision
// (the same seven bits serve the real-part and the imaginary-part pass of Table 2: 7+7+7 values
// but 14 precision choices).
//
// Readings:
//   T1  Table 1 row 7 is Eq.(4) with brackets restored: tau <- tau * (W s2/(s12+eps) - 1)   (G3)
//   T2  eps = machine epsilon of the group's format where it is used: 2^-23 (single), 2^-10 (half)
//   T3  Table 2 group 2 as printed in Table 2: p <- sqrt(a+b+c) + eps  (Table 4 prints sqrt(.+eps); Table 2 wins)
//   T4  sums run sequentially in sample order, the accumulator in the group's format
//   T5  the inputs xr, xi, q, u, v are the single-precision Stokes parameters, formed in single
//   T6  W, d, 1, the thresholds are constants converted into the consuming group's format
//   T7  comparisons are the strict ones of Eq.(5),(10), written negated so that NaN flags (G5, G6)
//
// Pins (tests/test_oracle_tables.py): with mask = 0 and inputs chosen so that every single-precision operation
// is exact, the tables reproduce the closed forms of the fp64 oracle up to the eps guards; half-precision
// operations against numpy.float16 arithmetic; overflow of y = x^2 in half above |x| = 255.9; mask bit order.

#include <cmath>
#include <cstdint>
#include <limits>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

inline float to_half(float x) { return static_cast<float>(static_cast<_Float16>(x)); }

// One arithmetic format: single or half.  Every method converts its operands into the format first.
struct Fmt {
    bool half;
    float cv(float x) const { return half ? to_half(x) : x; }                    // type conversion
    float add(float a, float b) const { return cv(cv(a) + cv(b)); }
    float sub(float a, float b) const { return cv(cv(a) - cv(b)); }
    float mul(float a, float b) const { return cv(cv(a) * cv(b)); }
    float div(float a, float b) const { return cv(cv(a) / cv(b)); }
    float sqrt(float a) const { return cv(std::sqrt(cv(a))); }
    float eps() const { return half ? 9.765625e-4f : 1.1920928955078125e-7f; }   // 2^-10, 2^-23   (T2)
};

inline Fmt fmt(uint32_t mask, int bit) { return Fmt{((mask >> bit) & 1u) != 0}; }

}  // namespace

extern "C" {

// Table 1 on one window.  xr[i], xi[i]: real and imaginary part of I_i (single).  Returns the flag; *tau_out = tau.
int oracle_tables_sk(const float* xr, const float* xi, int W, float d, float s_low, float s_high,
                     uint32_t mask, float* tau_out) {
    const Fmt g1 = fmt(mask, 0), g2 = fmt(mask, 1), g3 = fmt(mask, 2), g4 = fmt(mask, 3);
    const Fmt g5 = fmt(mask, 4), g6 = fmt(mask, 5), g7 = fmt(mask, 6);
    float s1 = 0.0f, s2 = 0.0f;
    for (int i = 0; i < W; ++i) {
        const float y = g1.add(g1.mul(xr[i], xr[i]), g1.mul(xi[i], xi[i]));      // group 1: y_i <- xr_i^2 + xi_i^2
        const float z = g2.sqrt(y);                                              // group 2: z_i <- sqrt(y_i)
        s1 = g3.add(s1, z);                                                      // group 3: s1 <- sum z_i
        s2 = g4.add(s2, y);                                                      // group 4: s2 <- sum y_i
    }
    const float Wf = static_cast<float>(W);
    float tau = g5.div(g5.add(g5.mul(Wf, d), 1.0f), g5.sub(Wf, 1.0f));           // group 5: tau <- (W d + 1)/(W - 1)
    const float s12 = g6.mul(s1, s1);                                            // group 6: s12 <- s1^2
    const float ratio = g7.div(g7.mul(Wf, s2), g7.add(s12, g7.eps()));           // group 7: W s2 / (s12 + eps)
    tau = g7.mul(tau, g7.sub(ratio, 1.0f));                                      //          tau <- tau (ratio - 1)   (T1)
    *tau_out = tau;
    const bool ok = (g7.cv(tau) >= g7.cv(s_low)) && (g7.cv(tau) <= g7.cv(s_high));   // group 7: tau < s_low OR tau > s_high
    return ok ? 0 : 1;
}

// Table 2 on one window, one part.  q,u,v: real parts (or imaginary parts) of Q_i, U_i, V_i (single).
int oracle_tables_ds(const float* q, const float* u, const float* v, int W, float gamma, uint32_t mask, float* r_out) {
    const Fmt g1 = fmt(mask, 7), g2 = fmt(mask, 8), g3 = fmt(mask, 9), g4 = fmt(mask, 10);
    const Fmt g5 = fmt(mask, 11), g6 = fmt(mask, 12), g7 = fmt(mask, 13);
    float qs = 0.0f, us = 0.0f, vs = 0.0f;
    for (int i = 0; i < W; ++i) {
        const float a = g1.mul(q[i], q[i]);                                      // group 1: a_i, b_i, c_i
        const float b = g1.mul(u[i], u[i]);
        const float c = g1.mul(v[i], v[i]);
        const float p = g2.add(g2.sqrt(g2.add(g2.add(a, b), c)), g2.eps());      // group 2: p_i <- sqrt(a+b+c) + eps   (T3)
        const float qh = g3.div(q[i], p);                                        // group 3: normalise
        const float uh = g3.div(u[i], p);
        const float vh = g3.div(v[i], p);
        qs = g4.add(qs, qh);                                                     // group 4: sums
        us = g4.add(us, uh);
        vs = g4.add(vs, vh);
    }
    const float q2 = g5.mul(qs, qs), u2 = g5.mul(us, us), v2 = g5.mul(vs, vs);   // group 5: squares
    const float r = g6.div(g6.sqrt(g6.add(g6.add(q2, u2), v2)), static_cast<float>(W));   // group 6: r <- sqrt(q+u+v)/W
    *r_out = r;
    return (g7.cv(r) <= g7.cv(gamma)) ? 0 : 1;                                   // group 7: r > gamma
}

// The whole path on one chunk in the tables' arithmetic (per-channel windows, one threshold set).
//   vis      [n_time][n_cells][4 pols][re,im] float32, time slowest (the stream is single precision).
//   thr      d, s_low, s_high, gamma (single).
// Outputs (any may be NULL): tau, r_re, r_im [n_win][n_cells] float; flags [n_win][n_cells] u8;
//   avg [n_out][n_cells][8] double (mean of the unflagged samples); weight [n_out][n_cells].
// The flag is SK OR DS(real parts) OR DS(imaginary parts).  Returns 0, or -1 on invalid arguments.
int oracle_tables_process(const float* vis, int64_t n_time, int64_t n_cells, int M, int64_t n_int,
                          float d, float s_low, float s_high, float gamma, uint32_t mask,
                          float* tau, float* r_re, float* r_im, uint8_t* flags,
                          double* avg, int64_t* weight, int n_threads) {
    if (!vis || M < 2 || n_int <= 0 || n_time <= 0 || n_cells < 0 || (mask >> 14) != 0) return -1;
    if (n_time % n_int != 0 || n_int % M != 0) return -1;
    const int64_t n_out = n_time / n_int;
    const int64_t win_per_out = n_int / M;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif

#pragma omp parallel for schedule(static)
    for (int64_t cell = 0; cell < n_cells; ++cell) {
        float* s = new float[static_cast<size_t>(M) * 8];       // Stokes of the window: [8][M]
        for (int64_t o = 0; o < n_out; ++o) {
            double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            int64_t cnt = 0;
            for (int64_t wl = 0; wl < win_per_out; ++wl) {
                const int64_t w = o * win_per_out + wl;
                for (int i = 0; i < M; ++i) {
                    const float* x = vis + ((w * M + i) * n_cells + cell) * 8;   // xx, xy, yx, yy as (re, im)
                    s[0 * M + i] = x[0] + x[6];            // I = xx + yy                    Eq.(2), in single (T5)
                    s[1 * M + i] = x[1] + x[7];
                    s[2 * M + i] = x[0] - x[6];            // Q = xx - yy
                    s[3 * M + i] = x[1] - x[7];
                    s[4 * M + i] = x[2] + x[4];            // U = xy + yx
                    s[5 * M + i] = x[3] + x[5];
                    s[6 * M + i] = -(x[3] - x[5]);         // V = j (xy - yx): Re V = -Im(xy - yx)
                    s[7 * M + i] = x[2] - x[4];            //                  Im V =  Re(xy - yx)
                }
                float t, rr, ri;
                const int f_sk = oracle_tables_sk(s + 0 * M, s + 1 * M, M, d, s_low, s_high, mask, &t);
                const int f_re = oracle_tables_ds(s + 2 * M, s + 4 * M, s + 6 * M, M, gamma, mask, &rr);
                const int f_im = oracle_tables_ds(s + 3 * M, s + 5 * M, s + 7 * M, M, gamma, mask, &ri);
                const int f = (f_sk || f_re || f_im) ? 1 : 0;
                if (tau)   tau[w * n_cells + cell] = t;
                if (r_re)  r_re[w * n_cells + cell] = rr;
                if (r_im)  r_im[w * n_cells + cell] = ri;
                if (flags) flags[w * n_cells + cell] = static_cast<uint8_t>(f);
                if (!f) {
                    for (int i = 0; i < M; ++i) {
                        const float* x = vis + ((w * M + i) * n_cells + cell) * 8;
                        for (int p = 0; p < 8; ++p) acc[p] += static_cast<double>(x[p]);
                    }
                    cnt += M;
                }
            }
            const int64_t oi = o * n_cells + cell;
            if (weight) weight[oi] = cnt;
            if (avg) for (int p = 0; p < 8; ++p) avg[oi * 8 + p] = cnt ? acc[p] / static_cast<double>(cnt) : 0.0;
        }
        delete[] s;
    }
    return 0;
}

// One rounding to half and back, exposed so that the tests can pin it against numpy.float16.
float oracle_tables_to_half(float x) { return to_half(x); }

}  // extern "C"

// =====================================================================================================================
// The reinforcement-learning ENVIRONMENT of section 3, evaluated window by window: state (45
// values), cost, penalty, flag agreement with the double-precision flags, reward.  Plain and slow; test infrastructure.
//
// Readings where the paper is garbled or silent (T10-T15):
//   T10  cost columns: Table 1 as printed (3W, W, W, W, 1, 1, 1+2); Table 2 one W per per-sample row and 1,1,1 / 4 / 1
//        for the tail, i.e. groups 1-7 = 3W, W, 3W, 3W, 3, 4, 1 (its cost column prints 12 entries for 14 rows,
//        PAPER.md:169); each multiplied by C = 1 (single) or 0.6 (half); Table 2 runs twice.
//   T11  the 21 error values ("7 + 7 + 7"): per group, the mean over the group's outputs of
//        |value in the chosen precisions - value with every operation in double|, +inf if either is not finite.
//        Outputs: Table 1 g1 y_i, g2 z_i, g3 s1, g4 s2, g5 tau prefactor, g6 s12, g7 tau; Table 2 g1 a_i,b_i,c_i,
//        g2 p_i, g3 qhat,uhat,vhat, g4 the three sums, g5 the three squares, g6 r, g7 the flag (0/1).
//   T12  type conversions (0.3 each): one per element carried over a data-flow edge whose two ends have
//        different formats; the inputs (xr, xi, q, u, v) are single; constants are pre-converted.
//        Table 1 edges: in->g1 (2W), g1->g2 (W), g1->g4 (W), g2->g3 (W), g3->g6, g4->g7, g5->g7, g6->g7 (1 each).
//        Table 2 edges (per part): in->g1 (3W), g1->g2 (3W), in->g3 (3W), g2->g3 (W), g3->g4 (3W), g4->g5 (3),
//        g5->g6 (3), g6->g7 (1).
//   T13  overflow / underflow (penalty 20 if any occurs in the window): an operation or conversion whose
//        exact result is finite but whose rounded result is not (overflow), or whose exact result is non-zero but whose
//        rounded result is below the smallest normal number of the format (underflow).  Events are also counted.
//   T14  reward = rho * (number of the three flags -- SK, DS real parts, DS imaginary parts -- equal to the
//        double-precision flags) - cost - 0.3 * conversions - 20 * [any overflow/underflow]; rho is an argument (the
//        printed constant is garbled).
//   T15  the 10 data features: log(sum_i real(X_i)^p) / W for (I,2), (I,4), (Q,2), (U,2), (V,2), then
//        the same for the imaginary parts; natural logarithm, in double, on the single-precision Stokes parameters.
//        eps of the double-precision ground truth = 2^-52 (T2: machine epsilon of the format).
// Record per window: RL_REC = 52 doubles: [0..9] features, [10..23] precision bits, [24..44] errors (Table 1 g1..g7,
// Table 2 real g1..g7, Table 2 imaginary g1..g7), [45] operation cost, [46] conversions, [47] overflow events,
// [48] underflow events, [49] matching flags (0..3), [50] reward, [51] flags: mixed (bit0 SK, bit1 DS re, bit2 DS im)
// + 8 * double-precision flags.
// =====================================================================================================================
namespace {

constexpr int RL_REC = 52;

struct Events { double over = 0, under = 0; };

struct FmtE {                                              // one format with event detection (T13)
    bool half;
    Events* ev;
    double min_normal() const { return half ? 6.103515625e-05 : 1.17549435082228750797e-38; }
    float round(double exact, float r) const {             // r = the correctly rounded result computed natively
        if (std::isfinite(exact) && !std::isfinite(r)) ev->over += 1;
        else if (exact != 0.0 && std::fabs(static_cast<double>(r)) < min_normal()) ev->under += 1;
        return r;
    }
    float cv(float x) const {                              // conversion into this format
        if (!half) return x;
        const float r = to_half(x);
        if (r != x && !(std::isnan(r) && std::isnan(x))) {
            if (std::isfinite(x) && !std::isfinite(r)) ev->over += 1;
            else if (x != 0.0f && std::fabs(static_cast<double>(r)) < min_normal()) ev->under += 1;
        }
        return r;
    }
    float fin(float native) const { return half ? to_half(native) : native; }
    float add(float a, float b) const { a = cv(a); b = cv(b); return round((double)a + (double)b, fin(a + b)); }
    float sub(float a, float b) const { a = cv(a); b = cv(b); return round((double)a - (double)b, fin(a - b)); }
    float mul(float a, float b) const { a = cv(a); b = cv(b); return round((double)a * (double)b, fin(a * b)); }
    float div(float a, float b) const { a = cv(a); b = cv(b); return round((double)a / (double)b, fin(a / b)); }
    float sqrt(float a) const { a = cv(a); return round(std::sqrt((double)a), fin(std::sqrt(a))); }
    float eps() const { return half ? 9.765625e-4f : 1.1920928955078125e-7f; }
};

inline double mean_abs_err(const float* a, const double* b, int n) {
    double s = 0;
    for (int i = 0; i < n; ++i) {
        if (!std::isfinite(a[i]) || !std::isfinite(b[i])) return std::numeric_limits<double>::infinity();
        s += std::fabs(static_cast<double>(a[i]) - b[i]);
    }
    return s / n;
}

}  // namespace

extern "C" {

int oracle_rl_record_doubles(void) { return RL_REC; }

// Operation cost (T10) and conversion count (T12) of a mask for window size W.
void oracle_rl_cost(uint32_t mask, int W, double* op_cost, double* conversions) {
    auto C = [&](int bit) { return ((mask >> bit) & 1u) ? 0.6 : 1.0; };
    auto h = [&](int bit) { return (int)((mask >> bit) & 1u); };
    const double w = W;
    const double t1 = 3 * w * C(0) + w * C(1) + w * C(2) + w * C(3) + 1 * C(4) + 1 * C(5) + 3 * C(6);
    const double t2 = 3 * w * C(7) + w * C(8) + 3 * w * C(9) + 3 * w * C(10) + 3 * C(11) + 4 * C(12) + 1 * C(13);
    *op_cost = t1 + 2 * t2;
    double c1 = 0, c2 = 0;
    c1 += h(0) ? 2 * w : 0;                                  // in -> g1
    c1 += (h(0) != h(1)) ? w : 0;                            // g1 -> g2
    c1 += (h(0) != h(3)) ? w : 0;                            // g1 -> g4
    c1 += (h(1) != h(2)) ? w : 0;                            // g2 -> g3
    c1 += (h(2) != h(5)) ? 1 : 0;                            // g3 -> g6
    c1 += (h(3) != h(6)) ? 1 : 0;                            // g4 -> g7
    c1 += (h(4) != h(6)) ? 1 : 0;                            // g5 -> g7
    c1 += (h(5) != h(6)) ? 1 : 0;                            // g6 -> g7
    c2 += h(7) ? 3 * w : 0;                                  // in -> g1
    c2 += (h(7) != h(8)) ? 3 * w : 0;                        // g1 -> g2
    c2 += h(9) ? 3 * w : 0;                                  // in -> g3
    c2 += (h(8) != h(9)) ? w : 0;                            // g2 -> g3
    c2 += (h(9) != h(10)) ? 3 * w : 0;                       // g3 -> g4
    c2 += (h(10) != h(11)) ? 3 : 0;                          // g4 -> g5
    c2 += (h(11) != h(12)) ? 3 : 0;                          // g5 -> g6
    c2 += (h(12) != h(13)) ? 1 : 0;                          // g6 -> g7
    *conversions = c1 + 2 * c2;
}

// windows [n_windows][W][4 pols][re,im] float32 (each window's W samples contiguous); out [n_windows][RL_REC] double.
int oracle_rl_evaluate(const float* windows, int64_t n_windows, int W, uint32_t mask, float d, float s_low, float s_high,
                       float gamma, double rho, double* out, int n_threads) {
    if (!windows || !out || W < 2 || n_windows < 0 || (mask >> 14) != 0) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    double op_cost, conv;
    oracle_rl_cost(mask, W, &op_cost, &conv);
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < n_windows; ++n) {
        const float* x = windows + n * W * 8;
        double* o = out + n * RL_REC;
        // single-precision Stokes parameters (T5): [part][which][i], which = I, Q, U, V
        float* S = new float[static_cast<size_t>(8) * W];
        auto st = [&](int part, int which, int i) -> float& { return S[(static_cast<size_t>(part) * 4 + which) * W + i]; };
        for (int i = 0; i < W; ++i) {
            const float* v = x + i * 8;
            st(0, 0, i) = v[0] + v[6];  st(1, 0, i) = v[1] + v[7];             // I = xx + yy
            st(0, 1, i) = v[0] - v[6];  st(1, 1, i) = v[1] - v[7];             // Q = xx - yy
            st(0, 2, i) = v[2] + v[4];  st(1, 2, i) = v[3] + v[5];             // U = xy + yx
            st(0, 3, i) = -(v[3] - v[5]); st(1, 3, i) = v[2] - v[4];           // V = j (xy - yx)
        }
        // ---- features (T15) ----
        for (int part = 0; part < 2; ++part) {
            double m[5] = {0, 0, 0, 0, 0};
            for (int i = 0; i < W; ++i) {
                const double I = st(part, 0, i), Q = st(part, 1, i), U = st(part, 2, i), V = st(part, 3, i);
                m[0] += I * I; m[1] += I * I * I * I; m[2] += Q * Q; m[3] += U * U; m[4] += V * V;
            }
            for (int k = 0; k < 5; ++k) o[part * 5 + k] = std::log(m[k]) / W;
        }
        for (int b = 0; b < 14; ++b) o[10 + b] = (mask >> b) & 1u;
        // ---- Table 1: chosen precisions and double, side by side ----
        Events ev;
        const float Wf = static_cast<float>(W);
        const double Wd = W;
        int flags_mixed = 0, flags_dbl = 0;
        {
            const FmtE g1{fmt(mask, 0).half, &ev}, g2{fmt(mask, 1).half, &ev}, g3{fmt(mask, 2).half, &ev}, g4{fmt(mask, 3).half, &ev};
            const FmtE g5{fmt(mask, 4).half, &ev}, g6{fmt(mask, 5).half, &ev}, g7{fmt(mask, 6).half, &ev};
            float* y = new float[W]; float* z = new float[W];
            double* yd = new double[W]; double* zd = new double[W];
            float s1 = 0, s2 = 0; double s1d = 0, s2d = 0;
            for (int i = 0; i < W; ++i) {
                const float xr = st(0, 0, i), xi = st(1, 0, i);
                y[i] = g1.add(g1.mul(xr, xr), g1.mul(xi, xi));
                z[i] = g2.sqrt(y[i]);
                s1 = g3.add(s1, z[i]);
                s2 = g4.add(s2, y[i]);
                yd[i] = (double)xr * xr + (double)xi * xi;
                zd[i] = std::sqrt(yd[i]);
                s1d += zd[i]; s2d += yd[i];
            }
            const float pre = g5.div(g5.add(g5.mul(Wf, d), 1.0f), g5.sub(Wf, 1.0f));
            const float s12 = g6.mul(s1, s1);
            const float ratio = g7.div(g7.mul(Wf, s2), g7.add(s12, g7.eps()));
            const float tau = g7.mul(pre, g7.sub(ratio, 1.0f));
            const bool ok = (g7.cv(tau) >= g7.cv(s_low)) && (g7.cv(tau) <= g7.cv(s_high));
            const double pred = (Wd * (double)d + 1.0) / (Wd - 1.0);
            const double s12d = s1d * s1d;
            const double taud = pred * (Wd * s2d / (s12d + 2.220446049250313e-16) - 1.0);
            const bool okd = (taud >= (double)s_low) && (taud <= (double)s_high);
            flags_mixed |= ok ? 0 : 1; flags_dbl |= okd ? 0 : 1;
            o[24] = mean_abs_err(y, yd, W); o[25] = mean_abs_err(z, zd, W);
            o[26] = mean_abs_err(&s1, &s1d, 1); o[27] = mean_abs_err(&s2, &s2d, 1);
            o[28] = mean_abs_err(&pre, &pred, 1); o[29] = mean_abs_err(&s12, &s12d, 1); o[30] = mean_abs_err(&tau, &taud, 1);
            delete[] y; delete[] z; delete[] yd; delete[] zd;
        }
        // ---- Table 2, real parts then imaginary parts ----
        for (int part = 0; part < 2; ++part) {
            const FmtE g1{fmt(mask, 7).half, &ev}, g2{fmt(mask, 8).half, &ev}, g3{fmt(mask, 9).half, &ev}, g4{fmt(mask, 10).half, &ev};
            const FmtE g5{fmt(mask, 11).half, &ev}, g6{fmt(mask, 12).half, &ev}, g7{fmt(mask, 13).half, &ev};
            float* abc = new float[3 * W]; float* p = new float[W]; float* hat = new float[3 * W];
            double* abcd = new double[3 * W]; double* pd = new double[W]; double* hatd = new double[3 * W];
            float sum[3] = {0, 0, 0}; double sumd[3] = {0, 0, 0};
            for (int i = 0; i < W; ++i) {
                const float q = st(part, 1, i), u = st(part, 2, i), v = st(part, 3, i);
                abc[3 * i] = g1.mul(q, q); abc[3 * i + 1] = g1.mul(u, u); abc[3 * i + 2] = g1.mul(v, v);
                p[i] = g2.add(g2.sqrt(g2.add(g2.add(abc[3 * i], abc[3 * i + 1]), abc[3 * i + 2])), g2.eps());
                hat[3 * i] = g3.div(q, p[i]); hat[3 * i + 1] = g3.div(u, p[i]); hat[3 * i + 2] = g3.div(v, p[i]);
                for (int k = 0; k < 3; ++k) sum[k] = g4.add(sum[k], hat[3 * i + k]);
                abcd[3 * i] = (double)q * q; abcd[3 * i + 1] = (double)u * u; abcd[3 * i + 2] = (double)v * v;
                pd[i] = std::sqrt(abcd[3 * i] + abcd[3 * i + 1] + abcd[3 * i + 2]) + 2.220446049250313e-16;
                hatd[3 * i] = q / pd[i]; hatd[3 * i + 1] = u / pd[i]; hatd[3 * i + 2] = v / pd[i];
                for (int k = 0; k < 3; ++k) sumd[k] += hatd[3 * i + k];
            }
            float sq[3]; double sqd[3];
            for (int k = 0; k < 3; ++k) { sq[k] = g5.mul(sum[k], sum[k]); sqd[k] = sumd[k] * sumd[k]; }
            const float r = g6.div(g6.sqrt(g6.add(g6.add(sq[0], sq[1]), sq[2])), Wf);
            const double rd = std::sqrt(sqd[0] + sqd[1] + sqd[2]) / Wd;
            const bool ok = g7.cv(r) <= g7.cv(gamma);
            const bool okd = rd <= (double)gamma;
            flags_mixed |= ok ? 0 : (2 << part); flags_dbl |= okd ? 0 : (2 << part);
            const float f = ok ? 0.f : 1.f; const double fd = okd ? 0.0 : 1.0;
            double* e = o + 31 + 7 * part;
            e[0] = mean_abs_err(abc, abcd, 3 * W); e[1] = mean_abs_err(p, pd, W); e[2] = mean_abs_err(hat, hatd, 3 * W);
            e[3] = mean_abs_err(sum, sumd, 3); e[4] = mean_abs_err(sq, sqd, 3); e[5] = mean_abs_err(&r, &rd, 1);
            e[6] = mean_abs_err(&f, &fd, 1);
            delete[] abc; delete[] p; delete[] hat; delete[] abcd; delete[] pd; delete[] hatd;
        }
        int match = 0;
        for (int b = 0; b < 3; ++b) match += (((flags_mixed >> b) & 1) == ((flags_dbl >> b) & 1)) ? 1 : 0;
        o[45] = op_cost; o[46] = conv; o[47] = ev.over; o[48] = ev.under; o[49] = match;
        o[50] = rho * match - op_cost - 0.3 * conv - ((ev.over + ev.under) > 0 ? 20.0 : 0.0);
        o[51] = flags_mixed + 8 * flags_dbl;
        delete[] S;
    }
    return 0;
}

}  // extern "C"
