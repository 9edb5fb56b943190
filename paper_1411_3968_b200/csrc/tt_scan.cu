// tt_scan.cu -- device-wide exclusive scan of uint32 (reduce / scan-of-sums / apply), used by the
// radix fallback and the ordered compactions.  Deterministic: no atomics, no look-back races.
#include "tt_common.cuh"

namespace tt {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;  // 2048

__global__ void __launch_bounds__(kScanThreads) scan_reduce_kernel(const uint32_t* __restrict__ in,
                                                                   uint32_t* __restrict__ sums, uint32_t n) {
    __shared__ uint32_t sm[33];
    const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    uint32_t v = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < n) v += in[base + k];
    uint32_t total;
    block_exclusive_scan(v, sm, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// exclusive scan in place of a short array by ONE block (loops with a running carry)
__global__ void __launch_bounds__(1024) scan_small_kernel(uint32_t* __restrict__ a, uint32_t n,
                                                          uint32_t* __restrict__ total_out) {
    __shared__ uint32_t sm[33];
    uint32_t carry = 0;
    for (uint32_t base = 0; base < n; base += 1024) {
        const uint32_t i = base + threadIdx.x;
        const uint32_t v = i < n ? a[i] : 0u;
        uint32_t total;
        const uint32_t ex = block_exclusive_scan(v, sm, &total);
        if (i < n) a[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(kScanThreads) scan_apply_kernel(const uint32_t* in,  // may alias out
                                                                  uint32_t* out,
                                                                  const uint32_t* __restrict__ sums, uint32_t n) {
    __shared__ uint32_t sm[33];
    const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    uint32_t x[kScanItems];
    uint32_t v = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        x[k] = base + k < n ? in[base + k] : 0u;
        v += x[k];
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(v, sm, &total) + sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) out[base + k] = ex;
        ex += x[k];
    }
}

size_t scan_ws_count(uint32_t n) {
    // level-1 sums, then level-2 sums (level 2 is always small enough for one block: n < 2^32)
    const size_t nb1 = div_up(n, kScanTile);
    const size_t nb2 = div_up(nb1, kScanTile);
    return nb1 + nb2 + 64;
}

int exclusive_scan_u32(const uint32_t* in, uint32_t* out, uint32_t n, uint32_t* scratch, uint32_t* total,
                       cudaStream_t s) {
    if (n == 0) {
        if (total) TT_CUDA_OK(cudaMemsetAsync(total, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    const uint32_t nb1 = div_up(n, kScanTile);
    uint32_t* sums1 = scratch;
    TT_K(scan_reduce_kernel)<<<nb1, kScanThreads, 0, s>>>(in, sums1, n);
    if (nb1 <= 8192) {
        TT_K(scan_small_kernel)<<<1, 1024, 0, s>>>(sums1, nb1, total);
    } else {
        const uint32_t nb2 = div_up(nb1, kScanTile);
        uint32_t* sums2 = scratch + nb1;
        TT_K(scan_reduce_kernel)<<<nb2, kScanThreads, 0, s>>>(sums1, sums2, nb1);
        TT_K(scan_small_kernel)<<<1, 1024, 0, s>>>(sums2, nb2, total);
        TT_K(scan_apply_kernel)<<<nb2, kScanThreads, 0, s>>>(sums1, sums1, sums2, nb1);
    }
    TT_K(scan_apply_kernel)<<<nb1, kScanThreads, 0, s>>>(in, out, sums1, n);
    TT_LAUNCH_OK();
    return TT_OK;
}

}  // namespace tt
