// rfi_oracle.cpp -- fp64 CPU ORACLE for the flag-and-average hot path of
// "Energy and polarization based online interference mitigation in radio
// interferometry" (arxiv 2412.14775; text in /root/reference/PAPER.md).
//
// THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call it.  It shares no code, header, table or helper with
// the CUDA path under paper_2412_14775_b200/csrc/, and neither includes the other.
//
// It is the paper's definitions written out, one statement per equation, in
// double precision, in the paper's order and notation.  No blocking, fusion or
// reordering: three nested loops (cell, window, sample).  OpenMP over cells is
// used for wall-clock only (cells are independent) and changes no
// arithmetic.
//
// Pins (tests/test_oracle_pins.py): closed forms and invariants listed in
// DESIGN.md section "Oracle pins".  Every exported function is pinned; none is
// "parity unpinned".
//
// Readings of the paper (DESIGN.md section "Readings"):
//   G1  Stokes V = j (xy - yx), j the imaginary unit      PAPER.md:54 (glyph garbled)
//   G3  tau follows Eq.(4) (parenthesised), not Table 1 row 7   PAPER.md:68 vs :142
//   G4  epsilon guards replaced by exact-zero guards (the eps->0 limit) PAPER.md:131,142,169
//   G5  strict comparisons: tau==s_low, tau==s_high, r==gamma are not flagged PAPER.md:72,103
//   G6  NaN statistics flag the window (negated comparisons)
//   G9  weight = number of unflagged samples; avg = sum of unflagged / weight

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// IEEE binary16 -> double, exact.  (Written out here; the CUDA path uses the
// hardware conversion.  They share nothing.)
double half_bits_to_double(uint16_t h) {
    const int sign = (h >> 15) & 1;
    const int expo = (h >> 10) & 0x1f;
    const int frac = h & 0x3ff;
    double v;
    if (expo == 0) {
        v = std::ldexp(static_cast<double>(frac), -24);           // subnormal or zero
    } else if (expo == 31) {
        v = frac ? std::numeric_limits<double>::quiet_NaN()
                 : std::numeric_limits<double>::infinity();
    } else {
        v = std::ldexp(static_cast<double>(frac + 1024), expo - 25);
    }
    return sign ? -v : v;
}

// One real number of the visibility array, widened exactly to double.
// storage: 0 = float32, 1 = float16 (IEEE binary16), 2 = float64.
double load_real(const void* base, int storage, int64_t idx) {
    switch (storage) {
        case 0:  return static_cast<double>(static_cast<const float*>(base)[idx]);
        case 1:  return half_bits_to_double(static_cast<const uint16_t*>(base)[idx]);
        default: return static_cast<const double*>(base)[idx];
    }
}

}  // namespace

extern "C" {

// Complex Stokes parameters of one sample, Eq.(2).
//   v[8] = {xx.re, xx.im, xy.re, xy.im, yx.re, yx.im, yy.re, yy.im}   (row-major Eq.(1))
//   s[8] = {I.re, I.im, Q.re, Q.im, U.re, U.im, V.re, V.im}
// No factor 1/2 (the paper has none).  V = j*(xy - yx): for D = xy - yx,
// j*D = (-D.im) + j*(D.re).
void oracle_rfi_stokes(const double* v, double* s) {
    const double xx_re = v[0], xx_im = v[1];
    const double xy_re = v[2], xy_im = v[3];
    const double yx_re = v[4], yx_im = v[5];
    const double yy_re = v[6], yy_im = v[7];
    s[0] = xx_re + yy_re;           // I = xx + yy
    s[1] = xx_im + yy_im;
    s[2] = xx_re - yy_re;           // Q = xx - yy
    s[3] = xx_im - yy_im;
    s[4] = xy_re + yx_re;           // U = xy + yx
    s[5] = xy_im + yx_im;
    const double d_re = xy_re - yx_re;
    const double d_im = xy_im - yx_im;
    s[6] = -d_im;                   // V = j (xy - yx)
    s[7] = d_re;
}

// Statistics of one window of W = M samples (win[i*8 + 0..7], layout as above).
//   tau  : Eq.(3)-(4).
//   r_re : Eq.(6)-(9) on the real parts of (Q,U,V).
//   r_im : the same on the imaginary parts.
// Returns 0.
int oracle_rfi_window_stats(const double* win, int M, double d,
                            double* tau, double* r_re, double* r_im) {
    const double W = static_cast<double>(M);

    // --- spectral kurtosis, section 2.1 ---
    double S1 = 0.0, S2 = 0.0;
    for (int i = 0; i < M; ++i) {
        double s[8];
        oracle_rfi_stokes(win + 8 * i, s);
        const double y = s[0] * s[0] + s[1] * s[1];   // |I_i|^2   (Table 1 group 1)
        const double z = std::sqrt(y);                // |I_i|     (Table 1 group 2)
        S1 += z;                                      // Eq.(3)
        S2 += y;
    }
    const double c = (W * d + 1.0) / (W - 1.0);       // Table 1 group 5
    if (S1 == 0.0) {
        // Reading G4: the eps-guard's limit for an all-zero window: W*S2/(S1^2+eps) -> 0.
        *tau = -c;
    } else {
        *tau = c * (W * S2 / (S1 * S1) - 1.0);        // Eq.(4)
    }

    // --- directional statistics of polarization, section 2.2, once per part ---
    for (int part = 0; part < 2; ++part) {            // 0: real parts, 1: imaginary parts
        double q = 0.0, u = 0.0, v = 0.0;
        for (int i = 0; i < M; ++i) {
            double s[8];
            oracle_rfi_stokes(win + 8 * i, s);
            const double qi = s[2 + part];
            const double ui = s[4 + part];
            const double vi = s[6 + part];
            const double p = std::sqrt(qi * qi + ui * ui + vi * vi);   // Eq.(6)
            if (p == 0.0) continue;                   // reading G4: zero vector contributes nothing
            q += qi / p;                              // Eq.(7), Eq.(8)
            u += ui / p;
            v += vi / p;
        }
        const double r = std::sqrt(q * q + u * u + v * v) / W;         // Eq.(9)
        if (part == 0) *r_re = r; else *r_im = r;
    }
    return 0;
}

// Decision for one window and one threshold set, Eq.(5), Eq.(10).
// Strict inequalities (G5); written in negated form so that a NaN statistic flags (G6).
int oracle_rfi_decide(double tau, double r_re, double r_im,
                      double s_low, double s_high, double gamma) {
    const bool sk_ok  = (tau >= s_low) && (tau <= s_high);   // not (tau < s_low OR tau > s_high)
    const bool dsr_ok = (r_re <= gamma);                     // not (r > gamma)
    const bool dsi_ok = (r_im <= gamma);
    return (!sk_ok || !dsr_ok || !dsi_ok) ? 1 : 0;
}

// The whole path on one chunk.
//
//   vis      [n_time][n_cells][4 pols][re,im], storage 0/1/2 (f32/f16/f64), time slowest.
//            A "cell" is one (baseline, channel) stream; baselines are independent,
//            so any subset of cells (whole groups of F adjacent channels) may be passed.
//   M, F     window footprint: T = M time samples x F frequency samples, W = T x F (
//            typical W = 20 as 10 x 2 or 5 x 4).  The F channels of a window are
//            F consecutive cells (n_cells % F == 0).  F = 1 is the per-channel window (reading G7).
//            The statistics of Eq.(3)-(4) and Eq.(6)-(9) run over all W samples of the footprint;
//            the flag applies to all of them.  M * F >= 2.
//   n_int    samples per output integration; n_time % n_int == 0, n_int % M == 0 (reading G8).
//   thr      [K][4] = d, s_low, s_high, gamma for each threshold set.
// Outputs (any may be NULL), all per cell (the F cells of a window carry the same statistics and flag):
//   tau      [K][n_win][n_cells]       n_win = n_time / M, window index w counts from chunk start
//   r_re,r_im[n_win][n_cells]
//   flags    [K][n_win][n_cells]       1 = flagged
//   avg      [K][n_out][n_cells][8]    mean of the unflagged samples of the cell, 0 if none;
//                                      no averaging across frequency (reading G9)
//   weight   [K][n_out][n_cells]       number of unflagged samples of the cell
// Returns 0, or -1 on invalid arguments.
int oracle_rfi_process_tf(const void* vis, int storage,
                          int64_t n_time, int64_t n_cells, int M, int F, int64_t n_int,
                          int K, const double* thr,
                          double* tau, double* r_re, double* r_im, uint8_t* flags,
                          double* avg, int64_t* weight, int n_threads) {
    if (!vis || !thr || M < 1 || F < 1 || M * F < 2 || n_int <= 0 || n_time <= 0 || n_cells < 0 || K < 1) return -1;
    if (n_time % n_int != 0 || n_int % M != 0 || n_cells % F != 0) return -1;
    if (storage < 0 || storage > 2) return -1;
    const int64_t n_win = n_time / M;
    const int64_t n_out = n_time / n_int;
    const int64_t win_per_out = n_int / M;
    const int64_t n_groups = n_cells / F;
    const int W = M * F;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif

#pragma omp parallel for schedule(static)
    for (int64_t grp = 0; grp < n_groups; ++grp) {
        const int64_t cell0 = grp * F;
        double* win = new double[static_cast<size_t>(W) * 8];      // sample (i, f) at index i * F + f
        double* acc = new double[static_cast<size_t>(K) * F * 8];
        int64_t* cnt = new int64_t[static_cast<size_t>(K) * F];
        for (int64_t o = 0; o < n_out; ++o) {
            // per-set, per-channel running sums for this output
            for (int64_t j = 0; j < static_cast<int64_t>(K) * F; ++j) { cnt[j] = 0; for (int p = 0; p < 8; ++p) acc[j * 8 + p] = 0.0; }

            for (int64_t wl = 0; wl < win_per_out; ++wl) {
                const int64_t w = o * win_per_out + wl;
                for (int i = 0; i < M; ++i) {
                    const int64_t t = w * M + i;
                    for (int f = 0; f < F; ++f)
                        for (int p = 0; p < 8; ++p)
                            win[(i * F + f) * 8 + p] = load_real(vis, storage, (t * n_cells + cell0 + f) * 8 + p);
                }
                for (int k = 0; k < K; ++k) {
                    const double d = thr[k * 4 + 0], s_low = thr[k * 4 + 1];
                    const double s_high = thr[k * 4 + 2], gamma = thr[k * 4 + 3];
                    double t_k, rr, ri;
                    oracle_rfi_window_stats(win, W, d, &t_k, &rr, &ri);
                    const int fl = oracle_rfi_decide(t_k, rr, ri, s_low, s_high, gamma);
                    for (int f = 0; f < F; ++f) {
                        const int64_t cell = cell0 + f;
                        if (tau)   tau[(static_cast<int64_t>(k) * n_win + w) * n_cells + cell] = t_k;
                        if (flags) flags[(static_cast<int64_t>(k) * n_win + w) * n_cells + cell] = static_cast<uint8_t>(fl);
                        if (k == 0) {
                            if (r_re) r_re[w * n_cells + cell] = rr;
                            if (r_im) r_im[w * n_cells + cell] = ri;
                        }
                        if (!fl) {                              // flagged windows are excluded
                            for (int i = 0; i < M; ++i)
                                for (int p = 0; p < 8; ++p) acc[(k * F + f) * 8 + p] += win[(i * F + f) * 8 + p];
                            cnt[k * F + f] += M;
                        }
                    }
                }
            }
            for (int k = 0; k < K; ++k)
                for (int f = 0; f < F; ++f) {
                    const int64_t oi = (static_cast<int64_t>(k) * n_out + o) * n_cells + cell0 + f;
                    const int64_t n = cnt[k * F + f];
                    if (weight) weight[oi] = n;
                    if (avg)
                        for (int p = 0; p < 8; ++p)
                            avg[oi * 8 + p] = n ? acc[(k * F + f) * 8 + p] / static_cast<double>(n) : 0.0;
                }
        }
        delete[] acc;
        delete[] cnt;
        delete[] win;
    }
    return 0;
}

// The per-channel window (F = 1, M >= 2): the main path of the build (reading G7).
int oracle_rfi_process(const void* vis, int storage,
                       int64_t n_time, int64_t n_cells, int M, int64_t n_int,
                       int K, const double* thr,
                       double* tau, double* r_re, double* r_im, uint8_t* flags,
                       double* avg, int64_t* weight, int n_threads) {
    if (M < 2) return -1;
    return oracle_rfi_process_tf(vis, storage, n_time, n_cells, M, 1, n_int, K, thr,
                                 tau, r_re, r_im, flags, avg, weight, n_threads);
}

// Bit-packed flag mask in the boundary's layout (include/rfi.h):
//   out[row][b][c / 32] bit (c % 32), 1 = flagged, rows = K * n_win, words per
//   baseline = ceil(n_chan / 32), unused high bits of the last word are 0.
//   flags[row][b * n_chan + c] is the byte array written by oracle_rfi_process.
int oracle_rfi_pack_flags(const uint8_t* flags, int64_t rows, int64_t n_baselines, int64_t n_chan,
                          uint32_t* out) {
    if (!flags || !out || rows < 0 || n_baselines < 0 || n_chan <= 0) return -1;
    const int64_t wpb = (n_chan + 31) / 32;
    for (int64_t r = 0; r < rows; ++r)
        for (int64_t b = 0; b < n_baselines; ++b)
            for (int64_t j = 0; j < wpb; ++j) {
                uint32_t word = 0;
                for (int bit = 0; bit < 32; ++bit) {
                    const int64_t c = j * 32 + bit;
                    if (c < n_chan && flags[(r * n_baselines + b) * n_chan + c]) word |= (1u << bit);
                }
                out[(r * n_baselines + b) * wpb + j] = word;
            }
    return 0;
}

int oracle_rfi_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
