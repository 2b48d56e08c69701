// rfi_sim42.cu -- the paper's section-4.2 simulator as a device generator: rfi_sim42_generate
// (include/rfi.h).  One realisation = one simulated baseline = a block of n_time x n_chan time-frequency samples of
// the four correlations; realisations sit on the baseline axis of the layout of include/rfi.h, vis[t][r][c][pol],
// so a batch feeds rfi_process_chunk directly (the 400-run FA/MD-vs-INR sweep of PAPER.md:235-237 is one chunk).
//
// Recipe and readings: DESIGN.md section 2 (S1-S9); restated here where it is implemented.  Random numbers come from
// a counter-based generator (Philox-4x32, 10 rounds; Salmon et al., SC'11) keyed by the seed with the counter
// (index, 0, stream, realisation), so every value is a pure function of its coordinates: no generator state, any
// launch shape, and a CPU restatement draws the identical integers (tests compare the fields element by element).
//
//   stream 0  per-realisation parameters (call index in the draw table below)
//   stream 1  noise: sample (t, c), call q = 0..3: index (t n_chan + c) 4 + q
//
// Kernels: parameters (one thread per realisation, fp64) -> source coherence per (realisation, channel) (fp64) ->
// celestial signal = a e_p e_q^H + sky + sources (fp32, writes vis once, reduces its total power) -> RFI power ->
// vis += g * rfi on the RFI support only, g^2 = INR P_cel / P_rfi -> window-level ground truth, bit-packed.
#include "rfi_internal.h"

#include <cmath>
#include <mutex>

namespace rfi {

constexpr int kSimMaxComp = RFI_SIM42_MAX_COMPONENTS;
constexpr int kSimMaxTries = 16;
constexpr int kSimCallsPerComp = 1 + 2 * kSimMaxTries;
constexpr double kCLight = 299792458.0;

struct SimCfg {
    int n_time, n_chan, n_real, n_sources, n_bb, n_nb, n_nd, polarized, wT, wF;
    uint32_t k0, k1;
    double inr;
};

// ---- Philox-4x32-10 ----
struct U4 { uint32_t x, y, z, w; };
__device__ __forceinline__ U4 philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return {c0, c1, c2, c3};
}
__device__ __forceinline__ double uniform01(uint32_t x) { return ((double)x + 0.5) * 0x1p-32; }
// normal pair, fp64 (parameters) and fp32 (noise): u = (2 (xa >> 9) + 1) 2^-24 and the angle (xb >> 8) 2^-24 turns are
// exact in both formats
__device__ __forceinline__ void normal_pair(uint32_t xa, uint32_t xb, double& z0, double& z1) {
    const double u = (2.0 * (double)(xa >> 9) + 1.0) * 0x1p-24;
    const double r = sqrt(-2.0 * log(u));
    double s, c;
    sincospi(2.0 * ((double)(xb >> 8) * 0x1p-24), &s, &c);
    z0 = r * c; z1 = r * s;
}
__device__ __forceinline__ void normal_pair(uint32_t xa, uint32_t xb, float& z0, float& z1) {
    const float u = (float)(2u * (xa >> 9) + 1u) * 0x1p-24f;
    const float r = sqrtf(-2.0f * logf(u));
    float s, c;
    sincospif(2.0f * ((float)(xb >> 8) * 0x1p-24f), &s, &c);
    z0 = r * c; z1 = r * s;
}

// ---- kernel 1: the per-realisation parameter table (draw table of the header comment in include/rfi.h) ----
__global__ void sim42_params_kernel(const SimCfg cfg, rfi_sim42_realisation* __restrict__ tab) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= cfg.n_real) return;
    rfi_sim42_realisation& o = tab[r];
    U4 x = philox(0, 0, 0, r, cfg.k0, cfg.k1);
    o.a = 100.0 * uniform01(x.x);                              // receiver-noise scale, constant over the block
    x = philox(1, 0, 0, r, cfg.k0, cfg.k1);
    double z0, z1, z2, z3;
    normal_pair(x.x, x.y, z0, z1);
    normal_pair(x.z, x.w, z2, z3);
    o.u = 300.0 * z0; o.v = 300.0 * z1; o.w = 300.0 * z2;
    o.p_cel = 0.0; o.p_rfi = 0.0; o.gain = 0.0;
    const int n_comp = cfg.n_bb + cfg.n_nb + cfg.n_nd;
    o.n_comp = n_comp;
    for (int i = 0; i < n_comp; ++i) {
        rfi_sim42_component& c = o.comp[i];
        const uint32_t base = 2u + (uint32_t)cfg.n_sources + (uint32_t)i * kSimCallsPerComp;
        x = philox(base, 0, 0, r, cfg.k0, cfg.k1);
        const double u0 = uniform01(x.x), u1 = uniform01(x.y), u2 = uniform01(x.z), u3 = uniform01(x.w);
        if (i < cfg.n_bb) {
            int e0 = (int)floor(u0 * (cfg.n_time + 1)), e1 = (int)floor(u1 * (cfg.n_time + 1));
            int f0 = (int)floor(u2 * (cfg.n_chan + 1)), f1 = (int)floor(u3 * (cfg.n_chan + 1));
            if (e0 > e1) { const int t = e0; e0 = e1; e1 = t; }
            if (f0 > f1) { const int t = f0; f0 = f1; f1 = t; }
            if (e0 == e1) { if (e0 == cfg.n_time) --e0; else ++e1; }
            if (f0 == f1) { if (f0 == cfg.n_chan) --f0; else ++f1; }
            c.kind = 0; c.t0 = e0; c.t1 = e1; c.c0 = f0; c.c1 = f1; c.period = 0.0;
        } else if (i < cfg.n_bb + cfg.n_nb) {
            const int ch = min((int)floor(u0 * cfg.n_chan), cfg.n_chan - 1);
            c.kind = 1; c.t0 = 0; c.t1 = cfg.n_time; c.c0 = ch; c.c1 = ch + 1; c.period = fmax(120.0 * u1, 2.0);
        } else {
            const int tt = min((int)floor(u0 * cfg.n_time), cfg.n_time - 1);
            c.kind = 2; c.t0 = tt; c.t1 = tt + 1; c.c0 = 0; c.c1 = cfg.n_chan; c.period = fmax(1024.0 * u1, 2.0);
        }
        double J[8];
        int tries = 0;
        if (cfg.polarized) {
            for (int k = 0; k < kSimMaxTries; ++k) {
                const U4 xa = philox(base + 1 + 2 * k, 0, 0, r, cfg.k0, cfg.k1);
                const U4 xb = philox(base + 2 + 2 * k, 0, 0, r, cfg.k0, cfg.k1);
                normal_pair(xa.x, xa.y, J[0], J[1]);
                normal_pair(xa.z, xa.w, J[2], J[3]);
                normal_pair(xb.x, xb.y, J[4], J[5]);
                normal_pair(xb.z, xb.w, J[6], J[7]);
                for (int q = 0; q < 8; ++q) J[q] *= 0.70710678118654752440;
                tries = k + 1;
                // polarised fraction of the coherency C = J J^H of J = [[J0,J1],[J2,J3]]  (the 90 % cut)
                const double c00 = J[0] * J[0] + J[1] * J[1] + J[2] * J[2] + J[3] * J[3];
                const double c11 = J[4] * J[4] + J[5] * J[5] + J[6] * J[6] + J[7] * J[7];
                // C01 = J0 conj(J2) + J1 conj(J3)
                const double c01r = J[0] * J[4] + J[1] * J[5] + J[2] * J[6] + J[3] * J[7];
                const double c01i = J[1] * J[4] - J[0] * J[5] + J[3] * J[6] - J[2] * J[7];
                const double I = c00 + c11, Q = c00 - c11, U = 2.0 * c01r, V = -2.0 * c01i;
                if (sqrt(Q * Q + U * U + V * V) / I <= 0.9) break;
            }
        } else {
            for (int q = 0; q < 8; ++q) J[q] = 0.0;
            J[0] = 1.0; J[6] = 1.0;                            // (1, 0, 0, 1): Q = U = V = 0
        }
        double nrm = 0.0;
        for (int q = 0; q < 8; ++q) nrm += J[q] * J[q];
        nrm = sqrt(nrm);
        for (int q = 0; q < 8; ++q) c.J[q] = J[q] / nrm;       // J / ||J||
        c.tries = tries;
    }
}

// ---- kernel 2: source coherence per (realisation, channel): sum_s S_s exp(j 2 pi f_c kappa_s) ----
__global__ void __launch_bounds__(256) sim42_sources_kernel(const SimCfg cfg, const rfi_sim42_realisation* __restrict__ tab,
                                                            double2* __restrict__ src) {
    extern __shared__ double sh[];                             // [n_sources] kappa, [n_sources] S
    const int r = blockIdx.x;
    double* kappa = sh;
    double* flux = sh + cfg.n_sources;
    const double u = tab[r].u, v = tab[r].v, w = tab[r].w;
    for (int s = threadIdx.x; s < cfg.n_sources; s += blockDim.x) {
        const U4 x = philox(2u + s, 0, 0, r, cfg.k0, cfg.k1);
        const double l = uniform01(x.x) - 0.5, m = uniform01(x.y) - 0.5;
        const double n = sqrt(1.0 - l * l - m * m);
        kappa[s] = (u * l + v * m + w * (n - 1.0)) / kCLight;
        flux[s] = 1.0 + 9.0 * uniform01(x.z);
    }
    __syncthreads();
    for (int c = threadIdx.x; c < cfg.n_chan; c += blockDim.x) {
        const double f = 120.0e6 + (double)c * (200.0e3 / (double)cfg.n_chan);
        double re = 0.0, im = 0.0;
        for (int s = 0; s < cfg.n_sources; ++s) {
            double sn, cs;
            sincospi(2.0 * (f * kappa[s]), &sn, &cs);
            re += flux[s] * cs; im += flux[s] * sn;
        }
        src[(size_t)r * cfg.n_chan + c] = make_double2(re, im);
    }
}

// One noise sample in fp32: a e_p e_q^H + sky.  out = xx, xy, yx, yy as (re, im).
__device__ __forceinline__ void noise_sample(const SimCfg& cfg, int t, int c, int r, float a, float (&o)[8]) {
    const unsigned long long base = ((unsigned long long)t * cfg.n_chan + c) * 4ull;
    float e[8], s[8];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const unsigned long long j = base + q;
        const U4 x = philox((uint32_t)j, (uint32_t)(j >> 32), 1u, (uint32_t)r, cfg.k0, cfg.k1);
        float z0, z1, z2, z3;
        normal_pair(x.x, x.y, z0, z1);
        normal_pair(x.z, x.w, z2, z3);
        float* dst = q < 2 ? e + 4 * q : s + 4 * (q - 2);
        dst[0] = z0 * 0.70710678f; dst[1] = z1 * 0.70710678f; dst[2] = z2 * 0.70710678f; dst[3] = z3 * 0.70710678f;
    }
    // e = (e_px, e_py, e_qx, e_qy); receiver = e_p e_q^H: (px qx*, px qy*, py qx*, py qy*)
    const float pxr = e[0], pxi = e[1], pyr = e[2], pyi = e[3], qxr = e[4], qxi = e[5], qyr = e[6], qyi = e[7];
    o[0] = a * (pxr * qxr + pxi * qxi) + s[0]; o[1] = a * (pxi * qxr - pxr * qxi) + s[1];
    o[2] = a * (pxr * qyr + pxi * qyi) + s[2]; o[3] = a * (pxi * qyr - pxr * qyi) + s[3];
    o[4] = a * (pyr * qxr + pyi * qxi) + s[4]; o[5] = a * (pyi * qxr - pyr * qxi) + s[5];
    o[6] = a * (pyr * qyr + pyi * qyi) + s[6]; o[7] = a * (pyi * qyr - pyr * qyi) + s[7];
}

constexpr int kSimTT = 16;                                     // time steps per block (one power atomic per block)

__device__ __forceinline__ double block_sum(double v, double* sh) {
    for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x < 32) {
        t = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        for (int m = 16; m > 0; m >>= 1) t += __shfl_xor_sync(0xffffffffu, t, m);
    }
    return t;                                                  // valid in thread 0
}

// ---- kernel 3: celestial signal = noise + sources, written once; total power per realisation ----
__global__ void __launch_bounds__(256) sim42_celestial_kernel(const SimCfg cfg, rfi_sim42_realisation* __restrict__ tab,
                                                              const double2* __restrict__ src, float* __restrict__ vis) {
    __shared__ double sh[8];
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = blockIdx.y;
    const int t_begin = blockIdx.z * kSimTT, t_end = min(t_begin + kSimTT, cfg.n_time);
    double pw = 0.0;
    if (c < cfg.n_chan) {
        const float a = (float)tab[r].a;
        const double2 sv = src[(size_t)r * cfg.n_chan + c];
        const float hr = (float)(0.5 * sv.x), hi = (float)(0.5 * sv.y);   // unpolarised source: xx = yy = S/2 * phase
        for (int t = t_begin; t < t_end; ++t) {
            float o[8];
            noise_sample(cfg, t, c, r, a, o);
            o[0] += hr; o[1] += hi; o[6] += hr; o[7] += hi;
            float p = 0.f;
#pragma unroll
            for (int q = 0; q < 8; ++q) p = fmaf(o[q], o[q], p);
            pw += (double)p;
            float4* dst = reinterpret_cast<float4*>(vis + (((size_t)t * cfg.n_real + r) * cfg.n_chan + c) * 8);
            dst[0] = make_float4(o[0], o[1], o[2], o[3]);
            dst[1] = make_float4(o[4], o[5], o[6], o[7]);
        }
    }
    const double tot = block_sum(pw, sh);
    if (threadIdx.x == 0) atomicAdd(&tab[r].p_cel, tot);
}

// The unscaled RFI field at (t, c): sum over components of amplitude * J/||J||.  Returns whether any
// component covers the point.
__device__ __forceinline__ bool rfi_field(const rfi_sim42_realisation& R, int t, int c, double (&f)[8]) {
    bool any = false;
#pragma unroll
    for (int q = 0; q < 8; ++q) f[q] = 0.0;
    for (int i = 0; i < R.n_comp; ++i) {
        const rfi_sim42_component& k = R.comp[i];
        if (t < k.t0 || t >= k.t1 || c < k.c0 || c >= k.c1) continue;
        any = true;
        double ar = 1.0, ai = 0.0;
        if (k.kind != 0) sincospi(2.0 * ((double)(k.kind == 1 ? t : c) / k.period), &ai, &ar);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            f[2 * q] += ar * k.J[2 * q] - ai * k.J[2 * q + 1];
            f[2 * q + 1] += ar * k.J[2 * q + 1] + ai * k.J[2 * q];
        }
    }
    return any;
}

// ---- kernel 4 (ADD = false): total power of the RFI field; kernel 5 (ADD = true): vis += g * field ----
template <bool ADD>
__global__ void __launch_bounds__(256) sim42_rfi_kernel(const SimCfg cfg, rfi_sim42_realisation* __restrict__ tab,
                                                        float* __restrict__ vis) {
    __shared__ double sh[8];
    __shared__ rfi_sim42_realisation R;
    const int r = blockIdx.y;
    for (int i = threadIdx.x; i < (int)(sizeof(R) / 4); i += blockDim.x)
        reinterpret_cast<uint32_t*>(&R)[i] = reinterpret_cast<const uint32_t*>(&tab[r])[i];
    __syncthreads();
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int t_begin = blockIdx.z * kSimTT, t_end = min(t_begin + kSimTT, cfg.n_time);
    double g = 0.0;
    if (ADD) {
        g = (cfg.inr > 0.0 && R.p_rfi > 0.0) ? sqrt(cfg.inr * R.p_cel / R.p_rfi) : 0.0;
        if (c == 0 && blockIdx.z == 0) tab[r].gain = g;
        if (g == 0.0) return;
    }
    double pw = 0.0;
    if (c < cfg.n_chan) {
        for (int t = t_begin; t < t_end; ++t) {
            double f[8];
            if (!rfi_field(R, t, c, f)) continue;
            if (ADD) {
                float4* dst = reinterpret_cast<float4*>(vis + (((size_t)t * cfg.n_real + r) * cfg.n_chan + c) * 8);
                float4 lo = dst[0], hi = dst[1];
                lo.x += (float)(g * f[0]); lo.y += (float)(g * f[1]); lo.z += (float)(g * f[2]); lo.w += (float)(g * f[3]);
                hi.x += (float)(g * f[4]); hi.y += (float)(g * f[5]); hi.z += (float)(g * f[6]); hi.w += (float)(g * f[7]);
                dst[0] = lo; dst[1] = hi;
            } else {
#pragma unroll
                for (int q = 0; q < 8; ++q) pw += f[q] * f[q];
            }
        }
    }
    if (!ADD) {
        const double tot = block_sum(pw, sh);
        if (threadIdx.x == 0 && tot != 0.0) atomicAdd(&tab[r].p_rfi, tot);
    }
}

// ---- kernel 6: window-level ground truth, bit-packed like one set of the flag mask: [n_win][n_real][ceil(n_chan/32)] ----
__global__ void sim42_truth_kernel(const SimCfg cfg, const rfi_sim42_realisation* __restrict__ tab, uint32_t* __restrict__ truth) {
    const int wpb = (cfg.n_chan + 31) / 32;
    const size_t n = (size_t)(cfg.n_time / cfg.wT) * cfg.n_real * wpb;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int j = (int)(i % wpb);
    const int r = (int)((i / wpb) % cfg.n_real);
    const int w = (int)(i / ((size_t)wpb * cfg.n_real));
    const rfi_sim42_realisation& R = tab[r];
    uint32_t word = 0;
    if (R.gain > 0.0) {
        const int ta = w * cfg.wT, tb = ta + cfg.wT;
        for (int b = 0; b < 32; ++b) {
            const int c = j * 32 + b;
            if (c >= cfg.n_chan) break;
            const int ca = c - c % cfg.wF, cb = ca + cfg.wF;   // the footprint this channel belongs to
            for (int k = 0; k < R.n_comp; ++k)
                if (R.comp[k].t0 < tb && R.comp[k].t1 > ta && R.comp[k].c0 < cb && R.comp[k].c1 > ca) { word |= 1u << b; break; }
        }
    }
    truth[i] = word;
}

}  // namespace rfi

extern "C" {

size_t rfi_sim42_vis_bytes(const rfi_sim42_config* c) {
    return c ? (size_t)c->n_time * c->n_real * c->n_chan * 32 : 0;
}
size_t rfi_sim42_truth_bytes(const rfi_sim42_config* c) {
    return (c && c->window_T > 0) ? (size_t)(c->n_time / c->window_T) * c->n_real * ((c->n_chan + 31) / 32) * 4 : 0;
}

int rfi_sim42_generate(const rfi_sim42_config* c, void* d_vis, uint32_t* d_truth, rfi_sim42_realisation* d_table,
                       double* d_sources, void* cuda_stream) {
    using namespace rfi_host;
    g_cuda_err[0] = 0;
    if (!c || !d_vis) return RFI_EINVAL;
    const int n_comp = c->n_broadband + c->n_narrowband + c->n_narrowdur;
    if (c->n_time < 1 || c->n_chan < 1 || c->n_real < 1 || c->n_real > 65535 || c->n_sources < 0 || c->n_sources > 4096 ||
        c->n_broadband < 0 || c->n_narrowband < 0 || c->n_narrowdur < 0 || n_comp > rfi::kSimMaxComp ||
        !(c->inr >= 0.f) || std::isinf(c->inr) || reinterpret_cast<uintptr_t>(d_vis) % 16) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_sim42_generate: bad configuration (sizes >= 1, n_real <= 65535, "
                 "n_sources <= 4096, at most %d RFI components, finite inr >= 0, 16-byte aligned d_vis)", rfi::kSimMaxComp);
        return RFI_EINVAL;
    }
    if (d_truth && (c->window_T < 1 || c->window_F < 1 || c->n_time % c->window_T || c->n_chan % c->window_F)) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_sim42_generate: the truth mask needs window_T | n_time and window_F | n_chan");
        return RFI_EINVAL;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    rfi::SimCfg k{c->n_time, c->n_chan, c->n_real, c->n_sources, c->n_broadband, c->n_narrowband, c->n_narrowdur,
                  c->polarized ? 1 : 0, c->window_T, c->window_F, (uint32_t)(c->seed & 0xffffffffull), (uint32_t)(c->seed >> 32),
                  (double)c->inr};
    rfi_sim42_realisation* tab = d_table;
    double2* src = reinterpret_cast<double2*>(d_sources);
    bool own_tab = false, own_src = false;
    int rc = RFI_OK;
    auto body = [&]() -> int {
        if (!tab) {
            if (cudaMalloc(&tab, sizeof(rfi_sim42_realisation) * (size_t)c->n_real) != cudaSuccess) { cudaGetLastError(); tab = nullptr; return RFI_ENOMEM; }
            own_tab = true;
        }
        if (!src) {
            if (cudaMalloc(&src, sizeof(double2) * (size_t)c->n_real * c->n_chan) != cudaSuccess) { cudaGetLastError(); src = nullptr; return RFI_ENOMEM; }
            own_src = true;
        }
        rfi::sim42_params_kernel<<<(c->n_real + 127) / 128, 128, 0, st>>>(k, tab);
        RFI_CUDA(cudaGetLastError());
        rfi::sim42_sources_kernel<<<c->n_real, 256, 2 * sizeof(double) * (size_t)(c->n_sources > 0 ? c->n_sources : 1), st>>>(k, tab, src);
        RFI_CUDA(cudaGetLastError());
        const dim3 grid((c->n_chan + 255) / 256, c->n_real, (c->n_time + rfi::kSimTT - 1) / rfi::kSimTT);
        if (grid.z > 65535) { snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_sim42_generate: n_time too large"); return RFI_EINVAL; }
        rfi::sim42_celestial_kernel<<<grid, 256, 0, st>>>(k, tab, src, static_cast<float*>(d_vis));
        RFI_CUDA(cudaGetLastError());
        if (c->inr > 0.f && n_comp > 0) {
            rfi::sim42_rfi_kernel<false><<<grid, 256, 0, st>>>(k, tab, nullptr);
            RFI_CUDA(cudaGetLastError());
            rfi::sim42_rfi_kernel<true><<<grid, 256, 0, st>>>(k, tab, static_cast<float*>(d_vis));
            RFI_CUDA(cudaGetLastError());
        }
        if (d_truth) {
            const size_t n = rfi_sim42_truth_bytes(c) / 4;
            rfi::sim42_truth_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(k, tab, d_truth);
            RFI_CUDA(cudaGetLastError());
        }
        return RFI_OK;
    };
    rc = body();
    if (own_tab || own_src) {
        // internal work buffers: wait for the kernels that use them, then release (the call is then synchronous)
        const cudaError_t e = cudaStreamSynchronize(st);
        if (own_tab && tab) cudaFree(tab);
        if (own_src && src) cudaFree(src);
        if (rc == RFI_OK && e != cudaSuccess) { cuda_ok(e, "cudaStreamSynchronize"); rc = RFI_ECUDA; }
    }
    return rc;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// rfi_sim42_generate_static: the same generator for callers that have no way to obtain device work memory.
//
// Who that is: code that runs inside somebody else's memory budget.  A correlator or beam-former process typically
// carves up the whole GPU at start-up (ring buffers for the ingest, a pool for everything else) and hands a plug-in
// only the input and output buffers of each call; a tuning loop that wants fresh section-4.2 blocks next to the live
// flagging streams must not call cudaMalloc / cudaFree either, because both serialise with every stream of the device
// and would stall the ingest for the duration.  rfi_sim42_generate needs two work arrays between its kernels (the
// parameter table and the source coherence) and either allocates them itself or takes them from the caller -- neither
// works for such a caller.  Here they live in one array that is part of the library image: the driver places it in
// device memory when the module is loaded on a GPU, so this entry point performs no allocation of any kind.
//
// The price: every GPU that loads librfi.so carries the array (kSim42StaticBytes, about 4.8 MiB) until the process
// exits, sizes are capped (RFI_SIM42_STATIC_MAX_REAL realisations, RFI_SIM42_STATIC_MAX_CELLS realisation x channel
// cells), and all calls on one device share the one array -- see the notes at the entry point.
constexpr size_t kSim42StaticTabBytes =
    (sizeof(rfi_sim42_realisation) * (size_t)RFI_SIM42_STATIC_MAX_REAL + 255) / 256 * 256;   // region 0: parameter table
constexpr size_t kSim42StaticSrcBytes = sizeof(double2) * (size_t)RFI_SIM42_STATIC_MAX_CELLS;  // region 1: source coherence
constexpr size_t kSim42StaticBytes = kSim42StaticTabBytes + kSim42StaticSrcBytes;
static_assert(sizeof(rfi_sim42_realisation) % 8 == 0 && kSim42StaticTabBytes % 256 == 0, "regions keep their alignment");
static_assert(kSim42StaticBytes <= (8u << 20), "the built-in work area is meant to stay small");

// One instance per device.  In host code this name is only a handle for the runtime's symbol calls, never a device
// address: the kernels get the pointer cudaGetSymbolAddress returns (sim42_static_scratch below).
static __device__ __align__(256) unsigned char g_sim42_static_scratch[kSim42StaticBytes];

namespace {

constexpr int kSim42StaticMaxDevices = 64;
std::mutex g_sim42_static_mu;
unsigned char* g_sim42_static_addr[kSim42StaticMaxDevices] = {};   // device address of the array, per device ordinal

// Device address of the work area on the CURRENT device; resolved once per device (the first call on a device makes
// the runtime load this module there, which is why that call should not happen inside a stream capture).
int sim42_static_scratch(int* dev_out, unsigned char** base_out) {
    using namespace rfi_host;
    int dev = -1;
    RFI_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kSim42StaticMaxDevices) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_sim42_generate_static: device ordinal %d is outside 0..%d", dev,
                 kSim42StaticMaxDevices - 1);
        return RFI_EINVAL;
    }
    std::lock_guard<std::mutex> lock(g_sim42_static_mu);
    if (!g_sim42_static_addr[dev]) {
        void* p = nullptr;
        RFI_CUDA(cudaGetSymbolAddress(&p, g_sim42_static_scratch));
        if (!p || reinterpret_cast<uintptr_t>(p) % 256) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_sim42_generate_static: the runtime returned an unusable address for the work area");
            return RFI_ECUDA;
        }
        g_sim42_static_addr[dev] = static_cast<unsigned char*>(p);
    }
    *dev_out = dev;
    *base_out = g_sim42_static_addr[dev];
    return RFI_OK;
}

}  // namespace

extern "C" {

size_t rfi_sim42_static_bytes(void) { return kSim42StaticBytes; }

int rfi_sim42_generate_static(const rfi_sim42_config* c, void* d_vis, uint32_t* d_truth, void* cuda_stream) {
    using namespace rfi_host;
    g_cuda_err[0] = 0;
    if (!c || !d_vis) return RFI_EINVAL;
    // the cap first, with its own message; every other rule of the configuration is checked by rfi_sim42_generate
    if (c->n_real >= 1 && c->n_chan >= 1 &&
        (c->n_real > RFI_SIM42_STATIC_MAX_REAL || (size_t)c->n_real * (size_t)c->n_chan > (size_t)RFI_SIM42_STATIC_MAX_CELLS)) {
        snprintf(g_cuda_err, sizeof(g_cuda_err),
                 "rfi_sim42_generate_static: n_real = %d, n_real * n_chan = %zu do not fit the built-in work area (at most %d "
                 "realisations and %d realisation-channel cells per call); split the batch, or use rfi_sim42_generate with "
                 "your own d_table / d_sources", c->n_real, (size_t)c->n_real * (size_t)c->n_chan,
                 RFI_SIM42_STATIC_MAX_REAL, RFI_SIM42_STATIC_MAX_CELLS);
        return RFI_EINVAL;
    }
    int dev = -1;
    unsigned char* base = nullptr;
    const int rc = sim42_static_scratch(&dev, &base);
    if (rc != RFI_OK) return rc;
    // the work area belongs to the current device: output buffers that live on another GPU would be written by
    // kernels running here through peer access at best, and not at all otherwise
    cudaPointerAttributes attr{};
    if (cudaPointerGetAttributes(&attr, d_vis) == cudaSuccess) {
        if (attr.type == cudaMemoryTypeDevice && attr.device != dev) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_sim42_generate_static: d_vis lives on device %d, the current device is %d",
                     attr.device, dev);
            return RFI_EINVAL;
        }
    } else {
        cudaGetLastError();
    }
    // With both work arrays given, rfi_sim42_generate only enqueues its kernels: no allocation, no synchronisation.
    // Nothing in the area has to be cleared here -- kernel 1 rewrites every field of the table rows it uses, the three
    // accumulators (p_cel, p_rfi, gain) to zero, and kernel 2 writes every source cell before kernel 3 reads it.
    return rfi_sim42_generate(c, d_vis, d_truth, reinterpret_cast<rfi_sim42_realisation*>(base),
                              reinterpret_cast<double*>(base + kSim42StaticTabBytes), cuda_stream);
}

}  // extern "C"
