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
