// rfi_confusion.cu -- per-set confusion counters of a flag mask against a ground-truth mask
// (BASELINE.json configs[4]: "per-set flag fraction against injected-RFI ground truth"; false-alarm and
// missed-detection probabilities as the paper defines them).  Pure bit work: popcounts over the
// bit-packed masks (layout of include/rfi.h), exact integers.
#include "rfi_internal.h"

namespace rfi {

// flags [K][n_rows][wpb-words per baseline...] flattened as [K][n_words]; truth [n_words]; word j of a baseline
// row holds channels 32j..32j+31, the last word of a baseline only n_chan % 32 valid bits.
__global__ void __launch_bounds__(256) rfi_confusion_kernel(const uint32_t* __restrict__ flags,
                                                            const uint32_t* __restrict__ truth,
                                                            unsigned long long* __restrict__ counts,
                                                            size_t n_words, int wpb, uint32_t last_mask) {
    const int k = blockIdx.y;
    const uint32_t* f = flags + (size_t)k * n_words;
    unsigned long long fa = 0, clean = 0, md = 0, rfi_n = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t valid = ((int)(i % (size_t)wpb) == wpb - 1) ? last_mask : 0xffffffffu;
        const uint32_t fw = f[i] & valid, tw = truth[i] & valid;
        fa += __popc(fw & ~tw);
        clean += __popc(~tw & valid);
        md += __popc(~fw & tw);
        rfi_n += __popc(tw);
    }
    for (int m = 16; m > 0; m >>= 1) {
        fa += __shfl_xor_sync(0xffffffffu, fa, m);
        clean += __shfl_xor_sync(0xffffffffu, clean, m);
        md += __shfl_xor_sync(0xffffffffu, md, m);
        rfi_n += __shfl_xor_sync(0xffffffffu, rfi_n, m);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(counts + 4 * k + 0, fa);
        atomicAdd(counts + 4 * k + 1, clean);
        atomicAdd(counts + 4 * k + 2, md);
        atomicAdd(counts + 4 * k + 3, rfi_n);
    }
}

}  // namespace rfi

namespace rfi_host {

int launch_confusion(const uint32_t* d_flags, const uint32_t* d_truth, uint64_t* d_counts, int K, size_t n_words,
                     int wpb, int n_chan, int sm_count, cudaStream_t st) {
    RFI_CUDA(cudaMemsetAsync(d_counts, 0, (size_t)K * 4 * sizeof(uint64_t), st));
    const uint32_t last_mask = (n_chan % 32) ? ((1u << (n_chan % 32)) - 1u) : 0xffffffffu;
    size_t bx = (n_words + 255) / 256;
    const size_t cap = (size_t)sm_count * 8;
    if (bx > cap) bx = cap;
    if (bx < 1) bx = 1;
    dim3 grid((unsigned)bx, (unsigned)K);
    rfi::rfi_confusion_kernel<<<grid, 256, 0, st>>>(d_flags, d_truth, reinterpret_cast<unsigned long long*>(d_counts),
                                                    n_words, wpb, last_mask);
    RFI_CUDA(cudaGetLastError());
    return RFI_OK;
}

}  // namespace rfi_host
