// rfi_adapt.cu -- on-line threshold adaptation: the update step that
// runs on the device between chunks.  The streaming kernel (rfi_direct_kernel<..., ADAPT>) has counted tau and
// max(r_re, r_im) of every window with finite statistics into per-class histograms; this kernel folds them into the
// running histograms (exponential forgetting), reads the quantiles that hold the requested false-alarm rate and
// writes the thresholds the NEXT chunk's kernel will load.  Everything stays on the device and on the caller's
// stream: rfi_process_chunk remains free of host synchronisation and can be captured in a CUDA graph.
//
// Readings A1-A6: constant false-alarm rate by rank -- s_low = Q_tau(beta/2),
// s_high = Q_tau(1 - beta/2), gamma = Q_r(1 - beta), beta = 1 - sqrt(1 - alpha) (two OR-ed detectors);
// a class with fewer than n_min counted windows keeps its thresholds.  Reading A8 (rfi_plan_set_adaptive_limit): with
// a bound lam >= 0 a threshold moves at most lam * |its a-priori value| in the loosening direction, because the
// histograms hold the contaminated windows too and their quantiles drift into the RFI once its occupancy exceeds alpha.
#include "rfi_internal.h"

namespace rfi {

__device__ double adapt_edge(int i, int lo_exp) {             // lower edge of bin i: 2^e (1 + m/64)
    return ldexp(1.0 + (double)(i & 63) / 64.0, lo_exp + (i >> 6));
}

// Quantile of a histogram in shared memory by one warp (A4): the bin where the cumulative count first reaches q N,
// linear interpolation between the bin's edges.  Lane l owns n_bins/32 consecutive bins; segment sums, a warp prefix
// and one short scan in the lane that holds the crossing.  (Counts are integers scaled by powers of `forget`: for the
// usual dyadic values every partial sum is exact, so the association of the sums does not matter.)
__device__ double adapt_quantile_warp(const double* h, int n_bins, int lo_exp, double total, double q) {
    const int lane = threadIdx.x & 31, seg = n_bins >> 5;
    const double* mine = h + lane * seg;
    double s = 0.0;
    for (int k = 0; k < seg; ++k) s += mine[k];
    double incl = s;
    for (int d = 1; d < 32; d <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    const double target = q * total;
    const unsigned crossed = __ballot_sync(0xffffffffu, incl >= target && s > 0.0);
    double result = adapt_edge(n_bins, lo_exp);
    if (crossed) {
        const int src = __ffs(crossed) - 1;
        if (lane == src) {
            double cum = incl - s;
            for (int k = 0; k < seg; ++k) {
                const double c = mine[k];
                if (c > 0.0 && cum + c >= target) {
                    const int i = lane * seg + k;
                    const double lo = adapt_edge(i, lo_exp), hi = adapt_edge(i + 1, lo_exp);
                    result = lo + (hi - lo) * ((target - cum) / c);
                    break;
                }
                cum += c;
            }
        }
        result = __shfl_sync(0xffffffffu, result, src);
    }
    return result;
}

// hist: this chunk's counts [2][kAdaptBins] (zeroed here for the next chunk); acc: running histograms (double);
// thr: the device thresholds the streaming kernel reads; raw: the same as (d, s_low, s_high, gamma) for inspection.
// prior: the a-priori sets (never written); lam < 0: no loosening bound.
__global__ void __launch_bounds__(256) rfi_adapt_update_kernel(uint32_t* hist, double* acc, Thr* thr, rfi_thresholds* raw,
                                                               const rfi_thresholds* __restrict__ prior, double lam,
                                                               int n_classes, double beta, double forget, double n_min) {
    __shared__ double sh[2 * kAdaptBins];
    __shared__ double tot[4];
    // one CTA per pair of histograms: the two classes, or baseline streams 2 b, 2 b + 1 (n_classes = streams in all)
    hist += (size_t)blockIdx.x * 2 * kAdaptBins;
    acc += (size_t)blockIdx.x * 2 * kAdaptBins;
    thr += blockIdx.x * 2;
    raw += blockIdx.x * 2;
    prior += blockIdx.x * 2;
    n_classes = min(2, n_classes - 2 * (int)blockIdx.x);
    for (int i = threadIdx.x; i < n_classes * kAdaptBins; i += blockDim.x) {
        const double v = forget * acc[i] + (double)hist[i];   // A3
        acc[i] = v;
        sh[i] = v;
        hist[i] = 0u;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp < 2 * n_classes) {                               // totals: warp w sums histogram (class w/2, tau or r)
        const int cls = warp >> 1, is_r = warp & 1;
        const double* h = sh + cls * kAdaptBins + (is_r ? kAdaptTauBins : 0);
        const int seg = (is_r ? kAdaptRBins : kAdaptTauBins) >> 5;
        double v = 0.0;
        for (int k = 0; k < seg; ++k) v += h[lane * seg + k];
        for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
        if (lane == 0) tot[warp] = v;
    }
    __syncthreads();
    // warp 3 cls + j computes quantile j of class cls (A5); a class with fewer than n_min counted windows keeps its
    // thresholds (A6)
    if (warp < 3 * n_classes) {
        const int cls = warp / 3, j = warp % 3;
        const double* ht = sh + cls * kAdaptBins;
        if (tot[2 * cls] >= n_min) {
            if (j == 0) {
                double q = adapt_quantile_warp(ht, kAdaptTauBins, kAdaptTauLoExp, tot[2 * cls], 0.5 * beta);
                if (lam >= 0.0) q = fmax(q, (double)prior[cls].s_low - lam * fabs((double)prior[cls].s_low));        // A8
                const float s_low = (float)q;
                if (lane == 0) { thr[cls].x_low = (float)((double)s_low / (double)thr[cls].c); raw[cls].s_low = s_low; }   // x = tau / c
            } else if (j == 1) {
                double q = adapt_quantile_warp(ht, kAdaptTauBins, kAdaptTauLoExp, tot[2 * cls], 1.0 - 0.5 * beta);
                if (lam >= 0.0) q = fmin(q, (double)prior[cls].s_high + lam * fabs((double)prior[cls].s_high));
                const float s_high = (float)q;
                if (lane == 0) { thr[cls].x_high = (float)((double)s_high / (double)thr[cls].c); raw[cls].s_high = s_high; }
            } else {
                double q = adapt_quantile_warp(ht + kAdaptTauBins, kAdaptRBins, kAdaptRLoExp, tot[2 * cls + 1], 1.0 - beta);
                if (lam >= 0.0) q = fmin(q, (double)prior[cls].gamma + lam * fabs((double)prior[cls].gamma));
                const float gamma = (float)q;
                if (lane == 0) { thr[cls].gamma = gamma; raw[cls].gamma = gamma; }
            }
        }
    }
}

}  // namespace rfi

namespace rfi_host {

int launch_adapt_update(uint32_t* d_hist, double* d_acc, rfi::Thr* d_thr, rfi_thresholds* d_raw, const rfi_thresholds* d_prior,
                        double max_loosen, int n_classes, double alpha, double forget, cudaStream_t st) {
    const double beta = 1.0 - sqrt(1.0 - alpha);
    rfi::rfi_adapt_update_kernel<<<(unsigned)((n_classes + 1) / 2), 256, 0, st>>>(d_hist, d_acc, d_thr, d_raw, d_prior, max_loosen,
                                                                                  n_classes, beta, forget, 1000.0);
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

}  // namespace rfi_host
