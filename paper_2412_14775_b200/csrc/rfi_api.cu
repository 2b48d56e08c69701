// rfi_api.cu -- host side of librfi.so: plan object, argument validation, kernel selection and the
// C ABI declared in include/rfi.h.  No CPU implementation of the method lives here: without a CUDA
// device every process call fails with RFI_ENODEV / RFI_ECUDA.
#include "rfi_internal.h"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace rfi_host {
thread_local char g_cuda_err[512] = "";
}

using namespace rfi_host;

namespace {

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    // function-local static: initialised exactly once, thread-safe (plans of different threads are independent)
    static const EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            return reinterpret_cast<EncodeTiledFn>(p);
        cudaGetLastError();
        return nullptr;
    }();
    return fn;
}

struct MapEntry {
    const void* ptr;
    int rows;
    int R;                     // rows per box; -1: cell-major transposing map
    CUtensorMap map;
};

}  // namespace

struct rfi_plan {
    int n_stations, n_baselines, n_chan, n_time, M, precision, n_int;
    int layout = RFI_LAYOUT_TIME_MAJOR;       // input layout
    int arith = RFI_ARITH_FAST;               // arithmetic mode
    uint32_t arith_mask = 0;                  // 14-bit precision mask of the tables mode
    int F = 1;                                // window extent in frequency (channels), W = M * F
    int n_classes = 1;                        // baseline threshold classes (1 or 2); thr holds K * n_classes sets, [k][class]
    std::vector<uint8_t> h_cls;               // class of every baseline of the whole array (n_classes == 2)
    uint8_t* d_cls = nullptr;
    bool cls_uploaded = false;
    const uint32_t* d_truth = nullptr;        // rfi_plan_set_truth: ground-truth mask and [K][4] counters of every device-path call
    uint64_t* d_counts = nullptr;
    bool truth_fused = false;                 // the last enqueue counted in its own kernel
    bool count_now = false;                   // inside rfi_process_chunk with a truth mask set
    int truth_K = 0;                          // K at rfi_plan_set_truth time: d_counts was sized for it
    int n_baselines_total = 0, b_first = 0;   // n_baselines is the shard this plan processes (default: all)
    int K = 0;
    std::vector<rfi_thresholds> thr;
    int variant = RFI_VARIANT_AUTO;
    int last_variant = 0;
    uint64_t launches = 0;
    // device state (created lazily)
    int device = -1;
    int sm_count = 0;
    int smem_optin = 0;
    bool dev_ready = false;
    uint32_t* d_flags = nullptr;
    size_t flags_words_cap = 0;
    bool have_result = false;
    std::vector<MapEntry> maps;
    // on-line threshold adaptation (rfi_plan_set_adaptive): device-resident thresholds, chunk and running histograms
    double adapt_alpha = 0.0, adapt_forget = 0.0;
    double adapt_loosen = -1.0;                // rfi_plan_set_adaptive_limit: < 0 = no bound (reading A8)
    int adapt_ns = 0;                          // streams of the state last uploaded (offset of the a-priori copy in d_thr_raw)
    rfi::Thr* d_thr = nullptr;                 // [2] thresholds the ADAPT kernel loads
    rfi_thresholds* d_thr_raw = nullptr;       // [2] the same as (d, s_low, s_high, gamma), then [2] the a-priori sets (kept)
    uint32_t* d_hist = nullptr;                // [2][kAdaptBins] this chunk's counts
    double* d_hist_acc = nullptr;              // [2][kAdaptBins] running histograms
    std::vector<rfi::Thr> adapt_stage_thr;     // host staging of the a-priori thresholds (per class or per stream)
    std::vector<rfi_thresholds> adapt_stage_raw;
    bool adapt_uploaded = false;               // d_thr holds the a-priori thresholds / the state was reset
    int adapt_scope = RFI_ADAPT_PER_CLASS;     // thresholds and histograms per class ([2]) or per baseline stream
    int adapt_cap = 0;                         // streams the adaptation buffers were allocated for
    std::vector<rfi_thresholds> stream_thr;    // rfi_plan_set_stream_thresholds: one set per baseline of the shard (empty: off)
    bool per_stream() const { return adapt_scope == RFI_ADAPT_PER_BASELINE || (!stream_thr.empty() && adapt_alpha <= 0.0); }
    int adapt_streams() const { return per_stream() ? n_baselines : 2; }
    // host path
    void* d_stage[2] = {nullptr, nullptr};
    size_t d_stage_cap[2] = {0, 0};
    cudaStream_t streams[2] = {nullptr, nullptr};
    cudaEvent_t ev_copied[2] = {nullptr, nullptr};
    cudaEvent_t ev_done[2] = {nullptr, nullptr};
    float* d_avg = nullptr;
    uint32_t* d_weight = nullptr;
    float* d_stats = nullptr;
    size_t d_avg_cap = 0, d_weight_cap = 0, d_stats_cap = 0;

    size_t n_cells() const { return (size_t)n_baselines * n_chan; }
    int wpb() const { return (n_chan + 31) / 32; }
    int n_win() const { return n_time / M; }
    int n_out() const { return n_time / n_int; }
    size_t sample_bytes() const { return precision == RFI_FP16 ? 16 : 32; }
    size_t flags_words() const { return (size_t)(K > 0 ? K : 1) * n_win() * n_baselines * wpb(); }
};

namespace {

int ensure_device(rfi_plan* p) {
    if (p->dev_ready) {
        // a plan is bound to the device that was current at its first process call (its flag buffer, class table and
        // staging buffers live there): refuse to run with another device current instead of faulting later
        int cur = -1;
        RFI_CUDA(cudaGetDevice(&cur));
        if (cur != p->device) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "plan is bound to CUDA device %d but device %d is current", p->device, cur);
            return RFI_EINVAL;
        }
        return RFI_OK;
    }
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count == 0) {
        cudaGetLastError();
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return RFI_ENODEV;
    }
    RFI_CUDA(cudaGetDevice(&p->device));
    cudaDeviceProp prop;
    RFI_CUDA(cudaGetDeviceProperties(&prop, p->device));
    if (prop.major != 10) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "device %s is sm_%d%d; this library is built for sm_100a only",
                 prop.name, prop.major, prop.minor);
        return RFI_ENODEV;
    }
    p->sm_count = prop.multiProcessorCount;
    p->smem_optin = (int)prop.sharedMemPerBlockOptin;
    p->dev_ready = true;
    return RFI_OK;
}

rfi::Thr to_device_thr(const rfi_thresholds& t, int W) {
    rfi::Thr r;
    r.c = (float)(((double)W * (double)t.d + 1.0) / ((double)W - 1.0));
    // Eq.(5) on x = tau / c (c > 0): +-inf stay +-inf, 0 stays 0
    r.x_low = (float)((double)t.s_low / (double)r.c);
    r.x_high = (float)((double)t.s_high / (double)r.c);
    r.gamma = t.gamma;
    return r;
}

// The map is returned BY VALUE (it is consumed as a __grid_constant__ kernel parameter): no pointer into the cache
// outlives an eviction.  Key: everything the encoding depends on that can change during a plan's life (the shard and
// the layout clear the cache).
int get_tensor_map(rfi_plan* p, const void* vis, int rows, int R, CUtensorMap* out) {
    for (auto& e : p->maps)
        if (e.ptr == vis && e.rows == rows && e.R == R) { *out = e.map; return RFI_OK; }
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled entry point not found");
        return RFI_ECUDA;
    }
    MapEntry e;
    e.ptr = vis; e.rows = rows; e.R = R;
    CUresult rc;
    const size_t ncell = p->n_cells();
    if (R < 0) {
        // cell-major vis[cell][t][sample]: {32 words = one 128-byte line = 4 (fp32) / 8 (fp16) samples of a cell,
        // rows / samples-per-line, n_cells}; box {32, 1, 32 cells}; 128-byte swizzle
        const size_t sb = p->sample_bytes();
        cuuint64_t dims[3] = {32, (cuuint64_t)((size_t)rows * sb / 128), (cuuint64_t)ncell};
        cuuint64_t strides[2] = {128, (cuuint64_t)rows * sb};
        cuuint32_t box[3] = {32, 1, 32};
        cuuint32_t estr[3] = {1, 1, 1};
        rc = enc(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, const_cast<void*>(vis), dims, strides, box, estr,
                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else if (p->precision == RFI_FP32) {
        // {32 floats = 4 cells, n_cells/4 groups, rows}; box {32, 8, R}; 128-byte swizzle
        cuuint64_t dims[3] = {32, (cuuint64_t)(ncell / 4), (cuuint64_t)rows};
        cuuint64_t strides[2] = {128, (cuuint64_t)ncell * 32};
        cuuint32_t box[3] = {32, 8, (cuuint32_t)R};
        cuuint32_t estr[3] = {1, 1, 1};
        rc = enc(&e.map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(vis), dims, strides, box, estr,
                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else {
        // {n_cells*4 32-bit words, rows}; box {128 words = 32 cells, R}
        cuuint64_t dims[2] = {(cuuint64_t)ncell * 4, (cuuint64_t)rows};
        cuuint64_t strides[1] = {(cuuint64_t)ncell * 16};
        cuuint32_t box[2] = {128, (cuuint32_t)R};
        cuuint32_t estr[2] = {1, 1};
        rc = enc(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(vis), dims, strides, box, estr,
                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (rc != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)rc);
        return RFI_ECUDA;
    }
    if (p->maps.size() >= 16) p->maps.erase(p->maps.begin());
    p->maps.push_back(e);
    *out = e.map;
    return RFI_OK;
}

bool tma_allowed(const rfi_plan* p) {
    if (p->precision == RFI_FP32) return p->n_cells() % 4 == 0;      // 128-byte inner box = 4 cells
    return true;
}

int ensure_flags(rfi_plan* p) {
    const size_t need = p->flags_words();
    if (need > p->flags_words_cap) {
        if (p->d_flags) cudaFree(p->d_flags);
        p->d_flags = nullptr;
        p->flags_words_cap = 0;
        if (cudaMalloc(&p->d_flags, need * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            return RFI_ENOMEM;
        }
        p->flags_words_cap = need;
    }
    return RFI_OK;
}

// Enqueue the kernel(s) for one slab of `n_out_slab` whole integrations starting at output o_first.
int enqueue_slab(rfi_plan* p, const void* d_vis_slab, int o_first, int n_out_slab, float* d_avg, uint32_t* d_weight,
                 float* d_stats, cudaStream_t st) {
    rfi::KParams kp;
    memset(&kp, 0, sizeof(kp));
    kp.vis = d_vis_slab;
    kp.avg = d_avg;
    kp.weight = d_weight;
    kp.stats = d_stats;
    kp.flags = p->d_flags;
    const int nc = p->n_classes;
    kp.thr0 = to_device_thr(p->thr[0], p->M * p->F);
    kp.thr1 = to_device_thr(p->thr[nc - 1], p->M * p->F);
    kp.cls = nc > 1 ? p->d_cls : nullptr;
    kp.b_first = p->b_first;
    kp.n_cells = (int)p->n_cells();
    kp.n_chan = p->n_chan;
    kp.n_baselines = p->n_baselines;
    kp.wpb = p->wpb();
    kp.M = p->M;
    kp.F = p->F;
    kp.inv_W = (float)(1.0 / ((double)p->M * p->F));
    kp.n_int = p->n_int;
    kp.wpo = p->n_int / p->M;
    kp.n_out_slab = n_out_slab;
    kp.o_first = o_first;
    kp.n_out_total = p->n_out();
    kp.n_win_total = p->n_win();
    kp.K = p->K;
    kp.k_first = 0;
    kp.flags_atomic = (p->n_chan % 32 != 0 && 32 % p->n_chan != 0) ? 1 : 0;
    if (p->adapt_alpha > 0.0) { kp.d_thr = p->d_thr; kp.hist = p->d_hist; kp.adapt_streams = p->adapt_scope == RFI_ADAPT_PER_BASELINE; }
    else if (!p->stream_thr.empty()) { kp.d_thr = p->d_thr; kp.adapt_streams = 2; }
    p->truth_fused = false;

    const bool fp16 = p->precision == RFI_FP16;
    if (p->arith == RFI_ARITH_TABLES) {
        // paper-literal Tables 1-2: single-precision stream, per-channel windows, one threshold set
        if (fp16 || p->F != 1 || p->K != 1 || p->layout != RFI_LAYOUT_TIME_MAJOR) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "tables arithmetic needs RFI_FP32 storage, F = 1, K = 1 and the time-major layout");
            return RFI_EINVAL;
        }
        kp.d = p->thr[0].d;
        kp.s_low = p->thr[0].s_low;
        kp.s_high = p->thr[0].s_high;
        kp.thr0.gamma = p->thr[0].gamma;
        kp.d1 = p->thr[nc - 1].d;
        kp.s_low1 = p->thr[nc - 1].s_low;
        kp.s_high1 = p->thr[nc - 1].s_high;
        kp.thr1.gamma = p->thr[nc - 1].gamma;
        kp.arith_mask = p->arith_mask;
        p->last_variant = RFI_VARIANT_TABLES;
        const int rc = launch_tables(kp, st);
        if (rc == RFI_OK) p->launches++;
        return rc;
    }
    if (p->layout == RFI_LAYOUT_CELL_MAJOR) {
        const int R = fp16 ? 8 : 4;                       // samples per 128-byte line
        if (p->M % R != 0 || n_out_slab != p->n_out()) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "cell-major layout needs window_M %% %d == 0 and device buffers", R);
            return RFI_EINVAL;
        }
        CUtensorMap map_v;
        const CUtensorMap* map = &map_v;
        int rc = get_tensor_map(p, kp.vis, p->n_time, -1, &map_v);
        if (rc != RFI_OK) return rc;
        if (p->K == 1) {
            p->last_variant = RFI_VARIANT_TMA;
            rc = launch_tma_cellmajor(fp16, kp, map, p->sm_count, p->smem_optin, st);
            if (rc == RFI_OK) p->launches++;
            return rc;
        }
        p->last_variant = RFI_VARIANT_BATCHED;
        for (int k0 = 0; k0 < p->K; k0 += rfi::kMaxBatch) {
            rfi::BatchThr bt;
            memset(&bt, 0, sizeof(bt));
            kp.k_first = k0;
            kp.K = p->K - k0 < rfi::kMaxBatch ? p->K - k0 : rfi::kMaxBatch;
            for (int k = 0; k < kp.K; ++k) {
                bt.t[k] = to_device_thr(p->thr[(size_t)(k0 + k) * nc], p->M * p->F);
                bt.t1[k] = to_device_thr(p->thr[(size_t)(k0 + k) * nc + nc - 1], p->M * p->F);
            }
            if (batched_mask_supported(kp) && p->count_now) {
                kp.truth = p->d_truth;
                kp.counts = reinterpret_cast<unsigned long long*>(p->d_counts);
                p->truth_fused = true;
            }
            if (batched_mask_supported(kp))
                rc = fp16 ? launch_batched_mask_f16(kp, bt, map, R, true, p->sm_count, p->smem_optin, st)
                          : launch_batched_mask_f32(kp, bt, map, R, true, p->sm_count, p->smem_optin, st);
            else
                rc = launch_batched_tma_cellmajor(fp16, kp, bt, map, p->sm_count, p->smem_optin, st);
            if (rc != RFI_OK) return rc;
            p->launches++;
        }
        return RFI_OK;
    }
    if (p->K > 1) {
        // batched-threshold mode: all sets in one pass over the data, 64 sets per launch
        p->last_variant = RFI_VARIANT_BATCHED;
        // same block length as the single-set direct kernel whenever that one uses R <= 4 (fp32) / 8 (fp16): then
        // K sets equal K single-set runs bit for bit
        int R = pick_rows(p->M, fp16, fp16 ? 8 : 4);
        // the second-generation kernel also has R = 5 (the paper's T = 10 and T = 5, as the direct kernel takes them)
        const int R5 = pick_rows(p->M, fp16, fp16 ? 8 : 5);
        const bool mask_ok = batched_mask_supported(kp) && tma_allowed(p) && env_int("RFI_BATCHED_TMA", 1) != 0;
        if (mask_ok && batched_mask_rows(fp16, R5)) R = R5;
        CUtensorMap map_v;
        const CUtensorMap* map = &map_v;
        const bool use_mask = mask_ok && batched_mask_rows(fp16, R);
        const bool use_tma = use_mask || (batched_tma_supported(fp16, kp, R) && tma_allowed(p));
        if (use_tma) {
            const int rc = get_tensor_map(p, kp.vis, n_out_slab * p->n_int, R, &map_v);
            if (rc != RFI_OK) return rc;
        }
        for (int k0 = 0; k0 < p->K; k0 += rfi::kMaxBatch) {
            rfi::BatchThr bt;
            memset(&bt, 0, sizeof(bt));
            kp.k_first = k0;
            kp.K = p->K - k0 < rfi::kMaxBatch ? p->K - k0 : rfi::kMaxBatch;
            for (int k = 0; k < kp.K; ++k) {
                bt.t[k] = to_device_thr(p->thr[(size_t)(k0 + k) * nc], p->M * p->F);
                bt.t1[k] = to_device_thr(p->thr[(size_t)(k0 + k) * nc + nc - 1], p->M * p->F);
            }
            int rc;
            if (use_mask && p->count_now) {   // counters in the same kernel (device path)
                kp.truth = p->d_truth;
                kp.counts = reinterpret_cast<unsigned long long*>(p->d_counts);
                p->truth_fused = true;
            }
            if (use_mask)
                rc = fp16 ? launch_batched_mask_f16(kp, bt, map, R, false, p->sm_count, p->smem_optin, st)
                          : launch_batched_mask_f32(kp, bt, map, R, false, p->sm_count, p->smem_optin, st);
            else
                rc = use_tma ? launch_batched_tma(fp16, kp, bt, map, R, p->sm_count, p->smem_optin, st)
                             : launch_batched(fp16, kp, bt, st);
            if (rc != RFI_OK) return rc;
            p->launches++;
        }
        return RFI_OK;
    }
    int variant = p->variant;
    // measured on B200 (profiles/): the register-staged direct kernel is the faster one for both storage types
    if (variant == RFI_VARIANT_AUTO) variant = RFI_VARIANT_DIRECT;
    if (variant == RFI_VARIANT_TMA && !tma_allowed(p)) {
        snprintf(g_cuda_err, sizeof(g_cuda_err),
                 "RFI_VARIANT_TMA with RFI_FP32 storage needs n_baselines * n_chan %% 4 == 0 (128-byte tensor-map rows); "
                 "use RFI_VARIANT_AUTO or RFI_VARIANT_DIRECT for %zu cells", p->n_cells());
        return RFI_EINVAL;
    }
    p->last_variant = variant;
    int rc;
    if (variant == RFI_VARIANT_SPLIT) {
        rc = launch_split(fp16, kp, p->smem_optin, st);
    } else if (variant == RFI_VARIANT_TMA) {
        const int rows = n_out_slab * p->n_int;
        const int R = tma_rows(p->M);
        CUtensorMap map_v;
        rc = get_tensor_map(p, kp.vis, rows, R, &map_v);
        if (rc != RFI_OK) return rc;
        rc = launch_tma(fp16, kp, &map_v, R, p->sm_count, p->smem_optin, st);
    } else {
        rc = launch_direct(fp16, kp, st);
    }
    if (rc == RFI_OK) p->launches++;
    return rc;
}

int prepare(rfi_plan* p, cudaStream_t st) {
    if (!p) return RFI_EINVAL;
    if (p->K < 1) return RFI_ESTATE;
    int rc = ensure_device(p);
    if (rc != RFI_OK) return rc;
    rc = ensure_flags(p);
    if (rc != RFI_OK) return rc;
    if (p->n_classes > 1 && !p->cls_uploaded) {
        if (!p->d_cls && cudaMalloc(&p->d_cls, p->h_cls.size()) != cudaSuccess) { cudaGetLastError(); return RFI_ENOMEM; }
        RFI_CUDA(cudaMemcpy(p->d_cls, p->h_cls.data(), p->h_cls.size(), cudaMemcpyHostToDevice));
        p->cls_uploaded = true;
    }
    if (p->variant == RFI_VARIANT_SPLIT && (p->K != 1 || p->arith != RFI_ARITH_FAST || p->layout != RFI_LAYOUT_TIME_MAJOR)) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "RFI_VARIANT_SPLIT needs K = 1, RFI_ARITH_FAST and the time-major layout "
                 "(the plan has K = %d%s%s); use RFI_VARIANT_AUTO", p->K, p->arith != RFI_ARITH_FAST ? ", tables arithmetic" : "",
                 p->layout != RFI_LAYOUT_TIME_MAJOR ? ", cell-major layout" : "");
        return RFI_EINVAL;
    }
    const bool flags_atomic = (p->n_chan % 32 != 0 && 32 % p->n_chan != 0);
    if (flags_atomic) RFI_CUDA(cudaMemsetAsync(p->d_flags, 0, p->flags_words() * sizeof(uint32_t), st));
    const bool stream_table = !p->stream_thr.empty();
    if (stream_table && (int)p->stream_thr.size() != p->n_baselines) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_plan_set_stream_thresholds was given %zu sets, the plan now processes %d baselines",
                 p->stream_thr.size(), p->n_baselines);
        return RFI_ESTATE;
    }
    if (p->adapt_alpha > 0.0 || stream_table) {
        if (p->K != 1 || p->arith != RFI_ARITH_FAST || p->layout != RFI_LAYOUT_TIME_MAJOR || p->variant == RFI_VARIANT_TMA ||
            p->variant == RFI_VARIANT_SPLIT) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "adaptive and per-stream thresholds need K = 1, RFI_ARITH_FAST, the time-major layout "
                     "and the direct kernel (RFI_VARIANT_AUTO or RFI_VARIANT_DIRECT)");
            return RFI_EINVAL;
        }
        if (p->per_stream() && p->n_chan % 32 != 0) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "thresholds / adaptation per baseline stream need n_chan %% 32 == 0 (a 32-cell tile must lie in one baseline)");
            return RFI_EINVAL;
        }
        const int ns = p->adapt_streams();
        const size_t hb = (size_t)ns * rfi::kAdaptBins;
        if (!p->d_thr || ns > p->adapt_cap) {
            cudaFree(p->d_thr); cudaFree(p->d_thr_raw); cudaFree(p->d_hist); cudaFree(p->d_hist_acc);
            p->d_thr = nullptr; p->d_thr_raw = nullptr; p->d_hist = nullptr; p->d_hist_acc = nullptr; p->adapt_cap = 0;
            if (cudaMalloc(&p->d_thr, ns * sizeof(rfi::Thr)) != cudaSuccess || cudaMalloc(&p->d_thr_raw, 2 * ns * sizeof(rfi_thresholds)) != cudaSuccess ||
                cudaMalloc(&p->d_hist, hb * sizeof(uint32_t)) != cudaSuccess || cudaMalloc(&p->d_hist_acc, hb * sizeof(double)) != cudaSuccess) {
                cudaGetLastError();
                return RFI_ENOMEM;
            }
            p->adapt_cap = ns;
            p->adapt_uploaded = false;
        }
        if (!p->adapt_uploaded) {
            // (re)start from the thresholds given a priori: every stream begins with its class's set.  The host
            // staging vectors live in the plan, so the asynchronous copies may complete after this call returns.
            const int nc = p->n_classes;
            p->adapt_stage_thr.resize(ns);
            p->adapt_stage_raw.resize(2 * (size_t)ns);     // [ns] current (updated on the device), [ns] a priori (kept: A8)
            for (int i = 0; i < ns; ++i) {
                int cls = i == 0 ? 0 : nc - 1;                // per class: [0] = class 0, [1] = class 1 (or 0 again)
                if (p->per_stream()) cls = nc > 1 ? (int)p->h_cls[p->b_first + i] : 0;
                // a stream table given by the caller is the a-priori state of its streams (and all there is without adaptation)
                const rfi_thresholds& src = (stream_table && p->per_stream()) ? p->stream_thr[i] : p->thr[cls];
                p->adapt_stage_thr[i] = to_device_thr(src, p->M * p->F);
                p->adapt_stage_raw[i] = src;
                p->adapt_stage_raw[ns + i] = src;
            }
            p->adapt_ns = ns;
            RFI_CUDA(cudaMemcpyAsync(p->d_thr, p->adapt_stage_thr.data(), ns * sizeof(rfi::Thr), cudaMemcpyHostToDevice, st));
            RFI_CUDA(cudaMemcpyAsync(p->d_thr_raw, p->adapt_stage_raw.data(), 2 * ns * sizeof(rfi_thresholds), cudaMemcpyHostToDevice, st));
            RFI_CUDA(cudaMemsetAsync(p->d_hist, 0, hb * sizeof(uint32_t), st));
            RFI_CUDA(cudaMemsetAsync(p->d_hist_acc, 0, hb * sizeof(double), st));
            p->adapt_uploaded = true;
        }
    }
    return RFI_OK;
}

// After the chunk's kernels: fold the chunk's histograms into the running ones and set the next chunk's thresholds.
int finish_adaptive(rfi_plan* p, cudaStream_t st) {
    if (p->adapt_alpha <= 0.0) return RFI_OK;                 // (static per-stream thresholds: nothing to update)
    const int rc = launch_adapt_update(p->d_hist, p->d_hist_acc, p->d_thr, p->d_thr_raw, p->d_thr_raw + p->adapt_ns, p->adapt_loosen,
                                       p->adapt_scope == RFI_ADAPT_PER_BASELINE ? p->n_baselines : p->n_classes, p->adapt_alpha,
                                       p->adapt_forget, st);
    if (rc == RFI_OK) p->launches++;
    return rc;
}

}  // namespace

extern "C" {

int rfi_plan_create(rfi_plan** out, int n_stations, int n_baselines, int n_chan, int n_time, int window_M,
                    int precision) {
    if (!out) return RFI_EINVAL;
    *out = nullptr;
    if (n_stations < 1 || n_chan < 1 || n_time < 1 || window_M < 2) return RFI_EINVAL;
    const long N = n_stations;
    if (n_baselines < 1 || ((long)n_baselines != N * (N + 1) / 2 && (long)n_baselines != N * (N - 1) / 2))
        return RFI_EINVAL;
    if (n_time % window_M != 0) return RFI_EINVAL;
    if (precision != RFI_FP32 && precision != RFI_FP16) return RFI_EINVAL;
    if ((long)n_baselines * n_chan > (1L << 30)) return RFI_EINVAL;
    rfi_plan* p = new (std::nothrow) rfi_plan();
    if (!p) return RFI_ENOMEM;
    p->n_stations = n_stations;
    p->n_baselines = n_baselines;
    p->n_baselines_total = n_baselines;
    p->n_chan = n_chan;
    p->n_time = n_time;
    p->M = window_M;
    p->precision = precision;
    p->n_int = n_time;
    *out = p;
    return RFI_OK;
}

int rfi_plan_set_integration(rfi_plan* p, int n_int) {
    if (!p || n_int < 1) return RFI_EINVAL;
    if (p->n_time % n_int != 0 || n_int % p->M != 0) return RFI_EINVAL;
    p->n_int = n_int;
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_set_baseline_classes(rfi_plan* p, int n_classes, const uint8_t* h_class) {
    if (!p || n_classes < 1 || n_classes > 2) return RFI_EINVAL;
    if (n_classes == 2) {
        if (!h_class) return RFI_EINVAL;
        for (int b = 0; b < p->n_baselines_total; ++b)
            if (h_class[b] > 1) return RFI_EINVAL;
        p->h_cls.assign(h_class, h_class + p->n_baselines_total);
    } else {
        p->h_cls.clear();
    }
    p->n_classes = n_classes;
    p->cls_uploaded = false;
    p->K = 0;                                 // the threshold table changes shape: thresholds must be set again
    p->thr.clear();
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_set_layout(rfi_plan* p, int layout) {
    if (!p || (layout != RFI_LAYOUT_TIME_MAJOR && layout != RFI_LAYOUT_CELL_MAJOR)) return RFI_EINVAL;
    p->layout = layout;
    p->have_result = false;
    p->maps.clear();
    return RFI_OK;
}

int rfi_plan_set_window_freq(rfi_plan* p, int F) {
    if (!p || F < 1 || F > 32 || (F & (F - 1)) != 0 || p->n_chan % F != 0) return RFI_EINVAL;
    p->F = F;
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_set_arithmetic(rfi_plan* p, int mode, uint32_t mask14) {
    if (!p || (mode != RFI_ARITH_FAST && mode != RFI_ARITH_TABLES) || (mask14 >> 14) != 0) return RFI_EINVAL;
    if (mode == RFI_ARITH_FAST && mask14 != 0) return RFI_EINVAL;
    p->arith = mode;
    p->arith_mask = mask14;
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_set_baseline_shard(rfi_plan* p, int b_first, int b_count) {
    if (!p || b_first < 0 || b_count < 1 || (long)b_first + b_count > p->n_baselines_total) return RFI_EINVAL;
    p->b_first = b_first;
    p->n_baselines = b_count;
    p->have_result = false;
    p->adapt_uploaded = false;                // per-stream adaptation state belongs to the old baseline range
    p->maps.clear();
    return RFI_OK;
}

int rfi_set_thresholds(rfi_plan* p, int K, const rfi_thresholds* h_sets) {
    if (!p || K < 1 || !h_sets || K > 4096) return RFI_EINVAL;
    const int n_sets = K * p->n_classes;                      // [k][class]
    for (int k = 0; k < n_sets; ++k) {
        const rfi_thresholds& t = h_sets[k];
        if (!(t.d > 0.f) || std::isinf(t.d)) return RFI_EINVAL;
        if (std::isnan(t.s_low) || std::isnan(t.s_high) || std::isnan(t.gamma)) return RFI_EINVAL;
    }
    p->thr.assign(h_sets, h_sets + n_sets);
    p->K = K;
    p->have_result = false;
    p->adapt_uploaded = false;                // adaptation restarts from the new a-priori thresholds
    return RFI_OK;
}

int rfi_plan_set_truth(rfi_plan* p, const uint32_t* d_truth, uint64_t* d_counts) {
    if (!p || (d_truth == nullptr) != (d_counts == nullptr)) return RFI_EINVAL;
    if (reinterpret_cast<uintptr_t>(d_truth) % 4 || reinterpret_cast<uintptr_t>(d_counts) % 8) return RFI_EINVAL;
    p->d_truth = d_truth;
    p->d_counts = d_counts;
    p->truth_K = p->K;
    return RFI_OK;
}

int rfi_plan_set_adaptive(rfi_plan* p, float false_alarm, float forget) {
    if (!p || !(false_alarm >= 0.f) || !(false_alarm < 0.5f) || !(forget >= 0.f) || !(forget < 1.f)) return RFI_EINVAL;
    p->adapt_alpha = false_alarm;
    p->adapt_forget = forget;
    p->adapt_uploaded = false;
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_set_adaptive_limit(rfi_plan* p, float max_loosen) {
    if (!p || std::isnan(max_loosen)) return RFI_EINVAL;
    p->adapt_loosen = max_loosen < 0.f ? -1.0 : (double)max_loosen;     // applies from the next update on; no restart
    return RFI_OK;
}

int rfi_plan_set_stream_thresholds(rfi_plan* p, const rfi_thresholds* h_sets) {
    if (!p) return RFI_EINVAL;
    if (h_sets) {
        for (int b = 0; b < p->n_baselines; ++b) {
            const rfi_thresholds& t = h_sets[b];
            if (!(t.d > 0.f) || std::isinf(t.d) || std::isnan(t.s_low) || std::isnan(t.s_high) || std::isnan(t.gamma)) return RFI_EINVAL;
        }
        p->stream_thr.assign(h_sets, h_sets + p->n_baselines);
    } else {
        p->stream_thr.clear();
    }
    p->adapt_uploaded = false;
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_set_adaptive_scope(rfi_plan* p, int scope) {
    if (!p || (scope != RFI_ADAPT_PER_CLASS && scope != RFI_ADAPT_PER_BASELINE)) return RFI_EINVAL;
    p->adapt_scope = scope;
    p->adapt_uploaded = false;
    p->have_result = false;
    return RFI_OK;
}

int rfi_plan_get_stream_thresholds(rfi_plan* p, rfi_thresholds* h_out) {
    if (!p || !h_out) return RFI_EINVAL;
    if (!p->per_stream() || !p->d_thr_raw || !p->adapt_uploaded) return RFI_ESTATE;
    RFI_CUDA(cudaMemcpy(h_out, p->d_thr_raw, (size_t)p->n_baselines * sizeof(rfi_thresholds), cudaMemcpyDeviceToHost));
    return RFI_OK;
}

int rfi_plan_get_stream_histograms(rfi_plan* p, double* h_out) {
    if (!p || !h_out) return RFI_EINVAL;
    if (p->adapt_scope != RFI_ADAPT_PER_BASELINE || p->adapt_alpha <= 0.0 || !p->d_hist_acc || !p->adapt_uploaded) return RFI_ESTATE;
    RFI_CUDA(cudaMemcpy(h_out, p->d_hist_acc, (size_t)p->n_baselines * rfi::kAdaptBins * sizeof(double), cudaMemcpyDeviceToHost));
    return RFI_OK;
}

int rfi_plan_get_adaptive_histogram(rfi_plan* p, double* h_out) {
    if (!p || !h_out) return RFI_EINVAL;
    if (p->adapt_scope != RFI_ADAPT_PER_CLASS || p->adapt_alpha <= 0.0 || !p->d_hist_acc || !p->adapt_uploaded) return RFI_ESTATE;
    RFI_CUDA(cudaMemcpy(h_out, p->d_hist_acc, 2 * (size_t)rfi::kAdaptBins * sizeof(double), cudaMemcpyDeviceToHost));
    return RFI_OK;
}

int rfi_plan_get_thresholds(rfi_plan* p, rfi_thresholds* h_out) {
    if (!p || !h_out) return RFI_EINVAL;
    if (p->K < 1) return RFI_ESTATE;
    const int nc = p->n_classes;
    if (p->adapt_alpha > 0.0 && p->d_thr_raw && p->adapt_uploaded && p->adapt_scope == RFI_ADAPT_PER_CLASS) {
        rfi_thresholds r[2];
        RFI_CUDA(cudaMemcpy(r, p->d_thr_raw, sizeof(r), cudaMemcpyDeviceToHost));    // waits for the device work so far
        for (int c = 0; c < nc; ++c) h_out[c] = r[c == 0 ? 0 : 1];
        return RFI_OK;
    }
    for (int c = 0; c < nc; ++c) h_out[c] = p->thr[c];
    return RFI_OK;
}

int rfi_plan_set_variant(rfi_plan* p, int variant) {
    if (!p || !(variant == RFI_VARIANT_AUTO || variant == RFI_VARIANT_DIRECT || variant == RFI_VARIANT_TMA ||
                variant == RFI_VARIANT_SPLIT)) return RFI_EINVAL;                             // BATCHED / TABLES are not selectable
    p->variant = variant;
    return RFI_OK;
}

int rfi_process_chunk(rfi_plan* p, const void* d_vis, void* d_avg, void* d_weight, void* d_stats, void* cuda_stream) {
    g_cuda_err[0] = 0;                        // rfi_last_cuda_error() describes THIS call if it fails
    if (!p) return RFI_EINVAL;
    if (p->K < 1) return RFI_ESTATE;
    if (!d_vis || !d_avg || !d_weight) return RFI_EINVAL;
    if (reinterpret_cast<uintptr_t>(d_vis) % 16 || reinterpret_cast<uintptr_t>(d_avg) % 16 ||
        reinterpret_cast<uintptr_t>(d_weight) % 4 || reinterpret_cast<uintptr_t>(d_stats) % 4)
        return RFI_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int rc = prepare(p, st);
    if (rc != RFI_OK) return rc;
    if (p->d_truth && p->truth_K != p->K) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_plan_set_truth was called with K = %d threshold sets, the plan now has %d: "
                 "set the truth mask (and a counter buffer of K x 4) again", p->truth_K, p->K);
        return RFI_ESTATE;
    }
    if (p->d_truth) RFI_CUDA(cudaMemsetAsync(p->d_counts, 0, (size_t)p->K * 4 * sizeof(uint64_t), st));
    p->count_now = p->d_truth != nullptr;
    rc = enqueue_slab(p, d_vis, 0, p->n_out(), static_cast<float*>(d_avg), static_cast<uint32_t*>(d_weight),
                      static_cast<float*>(d_stats), st);
    p->count_now = false;
    if (rc == RFI_OK && p->d_truth && !p->truth_fused) {     // kernels without in-kernel counters: a pass over the masks
        rc = launch_confusion(p->d_flags, p->d_truth, p->d_counts, p->K, (size_t)p->n_win() * p->n_baselines * p->wpb(),
                              p->wpb(), p->n_chan, p->sm_count, st);
        if (rc == RFI_OK) p->launches++;
    }
    if (rc == RFI_OK) rc = finish_adaptive(p, st);
    if (rc == RFI_OK) p->have_result = true;
    return rc;
}

int rfi_get_flags(rfi_plan* p, const uint32_t** d_flags, size_t* n_words) {
    if (!p || !d_flags || !n_words) return RFI_EINVAL;
    if (!p->have_result) return RFI_ESTATE;
    *d_flags = p->d_flags;
    *n_words = p->flags_words();
    return RFI_OK;
}

int rfi_confusion_counts(rfi_plan* p, const uint32_t* d_truth, uint64_t* d_counts, void* cuda_stream) {
    if (!p || !d_truth || !d_counts) return RFI_EINVAL;
    if (reinterpret_cast<uintptr_t>(d_truth) % 4 || reinterpret_cast<uintptr_t>(d_counts) % 8) return RFI_EINVAL;
    if (!p->have_result) return RFI_ESTATE;
    const size_t n_words = (size_t)p->n_win() * p->n_baselines * p->wpb();
    const int rc = launch_confusion(p->d_flags, d_truth, d_counts, p->K, n_words, p->wpb(), p->n_chan, p->sm_count,
                                    static_cast<cudaStream_t>(cuda_stream));
    if (rc == RFI_OK) p->launches++;
    return rc;
}

int rfi_process_chunk_host(rfi_plan* p, const void* h_vis, void* h_avg, void* h_weight, void* h_flags,
                           void* h_stats) {
    g_cuda_err[0] = 0;
    if (!p) return RFI_EINVAL;
    if (p->K < 1) return RFI_ESTATE;
    if (!h_vis || !h_avg || !h_weight || !h_flags) return RFI_EINVAL;
    if (p->layout != RFI_LAYOUT_TIME_MAJOR) return RFI_EINVAL;   // integrations are contiguous slabs only in time-major order
    int rc = ensure_device(p);
    if (rc != RFI_OK) return rc;
    const size_t slab_bytes = (size_t)p->n_int * p->n_cells() * p->sample_bytes();
    for (int i = 0; i < 2; ++i) {
        if (!p->streams[i]) RFI_CUDA(cudaStreamCreateWithFlags(&p->streams[i], cudaStreamNonBlocking));
        if (!p->ev_copied[i]) RFI_CUDA(cudaEventCreateWithFlags(&p->ev_copied[i], cudaEventDisableTiming));
        if (!p->ev_done[i]) RFI_CUDA(cudaEventCreateWithFlags(&p->ev_done[i], cudaEventDisableTiming));
    }
    auto grow = [](auto*& ptr, size_t& cap, size_t need) -> int {
        if (need <= cap) return RFI_OK;
        if (ptr) cudaFree(ptr);
        ptr = nullptr; cap = 0;
        void* q = nullptr;
        if (cudaMalloc(&q, need) != cudaSuccess) { cudaGetLastError(); return RFI_ENOMEM; }
        ptr = static_cast<std::remove_reference_t<decltype(ptr)>>(q);
        cap = need;
        return RFI_OK;
    };
    if ((rc = grow(p->d_avg, p->d_avg_cap, rfi_avg_bytes(p))) != RFI_OK) return rc;
    if ((rc = grow(p->d_weight, p->d_weight_cap, rfi_weight_bytes(p))) != RFI_OK) return rc;
    if (h_stats && (rc = grow(p->d_stats, p->d_stats_cap, rfi_stats_bytes(p))) != RFI_OK) return rc;
    // the staging slabs hold one integration of the CURRENT shape: rfi_plan_set_integration / _set_baseline_shard
    // can enlarge it between calls (no work of a previous call is in flight here: every host call synchronises)
    for (int i = 0; i < 2; ++i)
        if ((rc = grow(p->d_stage[i], p->d_stage_cap[i], slab_bytes)) != RFI_OK) return rc;

    cudaStream_t copy_st = p->streams[0], comp_st = p->streams[1];
    rc = prepare(p, comp_st);
    if (rc != RFI_OK) return rc;
    if (p->d_truth && p->truth_K != p->K) {                    // before any slab is enqueued: flags and adaptive state stay untouched
        snprintf(g_cuda_err, sizeof(g_cuda_err), "rfi_plan_set_truth was called with K = %d threshold sets, the plan now has %d: "
                 "set the truth mask (and a counter buffer of K x 4) again", p->truth_K, p->K);
        return RFI_ESTATE;
    }
    const int n_out = p->n_out();
    const uint8_t* src = static_cast<const uint8_t*>(h_vis);
    // Every exit path below drains both internal streams first: no copy from (or to) the caller's host buffers is
    // left in flight after the call returns, error or not.
    auto pipeline = [&]() -> int {
        for (int o = 0; o < n_out; ++o) {
            const int b = o & 1;
            // the staging buffer is free once the kernel that read it (slab o-2) has finished
            if (o >= 2) RFI_CUDA(cudaStreamWaitEvent(copy_st, p->ev_done[b], 0));
            RFI_CUDA(cudaMemcpyAsync(p->d_stage[b], src + (size_t)o * slab_bytes, slab_bytes, cudaMemcpyHostToDevice, copy_st));
            RFI_CUDA(cudaEventRecord(p->ev_copied[b], copy_st));
            RFI_CUDA(cudaStreamWaitEvent(comp_st, p->ev_copied[b], 0));
            const int rc2 = enqueue_slab(p, p->d_stage[b], o, 1, p->d_avg, p->d_weight, h_stats ? p->d_stats : nullptr, comp_st);
            if (rc2 != RFI_OK) return rc2;
            RFI_CUDA(cudaEventRecord(p->ev_done[b], comp_st));
        }
        const int rc3 = finish_adaptive(p, comp_st);
        if (rc3 != RFI_OK) return rc3;
        if (p->d_truth) {                                      // rfi_plan_set_truth: the mask pass over the completed flags
            const int rc4 = launch_confusion(p->d_flags, p->d_truth, p->d_counts, p->K,
                                             (size_t)p->n_win() * p->n_baselines * p->wpb(), p->wpb(), p->n_chan, p->sm_count, comp_st);
            if (rc4 != RFI_OK) return rc4;
            p->launches++;
        }
        RFI_CUDA(cudaMemcpyAsync(h_avg, p->d_avg, rfi_avg_bytes(p), cudaMemcpyDeviceToHost, comp_st));
        RFI_CUDA(cudaMemcpyAsync(h_weight, p->d_weight, rfi_weight_bytes(p), cudaMemcpyDeviceToHost, comp_st));
        RFI_CUDA(cudaMemcpyAsync(h_flags, p->d_flags, rfi_flags_bytes(p), cudaMemcpyDeviceToHost, comp_st));
        if (h_stats) RFI_CUDA(cudaMemcpyAsync(h_stats, p->d_stats, rfi_stats_bytes(p), cudaMemcpyDeviceToHost, comp_st));
        return RFI_OK;
    };
    rc = pipeline();
    const cudaError_t e1 = cudaStreamSynchronize(copy_st);
    const cudaError_t e2 = cudaStreamSynchronize(comp_st);
    if (rc != RFI_OK) return rc;
    RFI_CUDA(e1);
    RFI_CUDA(e2);
    p->have_result = true;
    return RFI_OK;
}

int rfi_plan_destroy(rfi_plan* p) {
    if (!p) return RFI_EINVAL;
    if (p->dev_ready) {
        if (p->d_flags) cudaFree(p->d_flags);
        if (p->d_cls) cudaFree(p->d_cls);
        if (p->d_thr) cudaFree(p->d_thr);
        if (p->d_thr_raw) cudaFree(p->d_thr_raw);
        if (p->d_hist) cudaFree(p->d_hist);
        if (p->d_hist_acc) cudaFree(p->d_hist_acc);
        if (p->d_avg) cudaFree(p->d_avg);
        if (p->d_weight) cudaFree(p->d_weight);
        if (p->d_stats) cudaFree(p->d_stats);
        for (int i = 0; i < 2; ++i) {
            if (p->d_stage[i]) cudaFree(p->d_stage[i]);
            if (p->ev_copied[i]) cudaEventDestroy(p->ev_copied[i]);
            if (p->ev_done[i]) cudaEventDestroy(p->ev_done[i]);
            if (p->streams[i]) cudaStreamDestroy(p->streams[i]);
        }
        cudaGetLastError();
    }
    delete p;
    return RFI_OK;
}

const char* rfi_strerror(int code) {
    switch (code) {
        case RFI_OK: return "ok";
        case RFI_EINVAL: return "invalid argument";
        case RFI_ECUDA: return "CUDA call failed (see rfi_last_cuda_error)";
        case RFI_ENOMEM: return "out of memory";
        case RFI_ESTATE: return "call order: thresholds not set or no chunk processed";
        case RFI_ENODEV: return "no usable sm_100 CUDA device";
        default: return "unknown error code";
    }
}

const char* rfi_last_cuda_error(void) { return g_cuda_err; }

size_t rfi_flags_bytes(const rfi_plan* p) { return p ? p->flags_words() * sizeof(uint32_t) : 0; }
size_t rfi_avg_bytes(const rfi_plan* p) {
    return p ? (size_t)(p->K > 0 ? p->K : 1) * p->n_out() * p->n_cells() * 8 * sizeof(float) : 0;
}
size_t rfi_weight_bytes(const rfi_plan* p) {
    return p ? (size_t)(p->K > 0 ? p->K : 1) * p->n_out() * p->n_cells() * sizeof(uint32_t) : 0;
}
size_t rfi_stats_bytes(const rfi_plan* p) { return p ? (size_t)3 * p->n_win() * p->n_cells() * sizeof(float) : 0; }
size_t rfi_vis_bytes(const rfi_plan* p) { return p ? (size_t)p->n_time * p->n_cells() * p->sample_bytes() : 0; }
uint64_t rfi_plan_launch_count(const rfi_plan* p) { return p ? p->launches : 0; }
int rfi_plan_last_variant(const rfi_plan* p) { return p ? p->last_variant : 0; }
const char* rfi_version(void) { return "rfi-b200 0.1 (sm_100a)"; }

}  // extern "C"
