// tt_radix.cu -- general stable sort of arbitrary (unsorted) input: LSD radix sort of
// (order-preserving uint64 key, uint32 input index) pairs, 8 bits per pass, then one gather of the
// 16-byte records.  This is the path for d_run_offsets == NULL ("classical sorting
// methods" on arbitrary data) and the safety net of the run-merge path; the per-PMT runs of the
// paper's workload go through tt_merge.cu instead.
//
// Segments: after the 8 key passes, ceil(log256(n_seg)) more passes on the segment id of the input
// index make every segment contiguous again (LSD: the last digit dominates), sorted inside.
// Passes whose digit is the same for all elements are skipped (decided on the device).
#include "tt_radix.cuh"

namespace tt {

constexpr int kRThreads = 256;
constexpr int kRItems = 8;
constexpr int kRTile = kRThreads * kRItems;  // 2048
constexpr int kRChunks = kRItems * (kRThreads / 32);  // 64 warp-chunks of 32 elements per tile

__global__ void __launch_bounds__(256) radix_extract_kernel(const uint4* __restrict__ hits, uint64_t* __restrict__ keys,
                                                            uint32_t* __restrict__ idx, uint32_t n,
                                                            RadixState* st) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { st->cur = 0; st->skip = 0; }
    if (i < n) {
        keys[i] = key_of(hit_time(__ldg(hits + i)));
        idx[i] = i;
    }
}

__device__ __forceinline__ uint32_t digit_of(uint64_t key, uint32_t id, int pass, const uint32_t* __restrict__ seg_off,
                                             uint32_t n_seg) {
    if (pass < 8) return (uint32_t)(key >> (8 * pass)) & 255u;
    const uint32_t s = find_segment(seg_off, n_seg, id);
    return (s >> (8 * (pass - 8))) & 255u;
}

// per-tile digit histogram -> hist[d * nblocks + b]
__global__ void __launch_bounds__(kRThreads) radix_hist_kernel(const uint64_t* __restrict__ keys0,
                                                               const uint64_t* __restrict__ keys1,
                                                               const uint32_t* __restrict__ idx0,
                                                               const uint32_t* __restrict__ idx1, uint32_t n, int pass,
                                                               const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                               const RadixState* __restrict__ st,
                                                               uint32_t* __restrict__ hist, uint32_t nblocks) {
    __shared__ uint32_t h[256];
    const uint32_t cur = st->cur;
    const uint64_t* keys = cur ? keys1 : keys0;
    const uint32_t* idx = cur ? idx1 : idx0;
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * kRTile;
#pragma unroll
    for (int r = 0; r < kRItems; ++r) {
        const uint32_t i = base + r * kRThreads + threadIdx.x;
        if (i < n) atomicAdd(&h[digit_of(keys[i], idx[i], pass, seg_off, n_seg)], 1u);
    }
    __syncthreads();
    hist[threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// after the scan: a pass is trivial iff one digit owns all n elements.  One block of 256 threads:
// thread d looks at the total of digit d = (scan[d+1 first] - scan[d first]).
__global__ void __launch_bounds__(256) radix_decide_kernel(const uint32_t* __restrict__ scanned, uint32_t nblocks,
                                                           uint32_t n, RadixState* st) {
    const uint32_t d = threadIdx.x;
    const uint32_t lo = scanned[d * nblocks];
    const uint32_t hi = d == 255 ? n : scanned[(d + 1) * nblocks];
    const int trivial = __syncthreads_or(hi - lo == n);
    if (d == 0) st->skip = trivial ? 1u : 0u;
}

__global__ void __launch_bounds__(kRThreads) radix_scatter_kernel(uint64_t* __restrict__ keys0, uint64_t* __restrict__ keys1,
                                                                  uint32_t* __restrict__ idx0, uint32_t* __restrict__ idx1,
                                                                  uint32_t n, int pass,
                                                                  const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                                  const RadixState* __restrict__ st,
                                                                  const uint32_t* __restrict__ scanned, uint32_t nblocks) {
    if (st->skip) return;
    __shared__ uint16_t chunk[kRChunks][256];  // 32 KB: per warp-chunk digit counts -> exclusive prefixes
    __shared__ uint32_t dbase[256];
    const uint32_t cur = st->cur;
    const uint64_t* kin = cur ? keys1 : keys0;
    const uint32_t* iin = cur ? idx1 : idx0;
    uint64_t* kout = cur ? keys0 : keys1;
    uint32_t* iout = cur ? idx0 : idx1;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int c = warp; c < kRChunks; c += kRThreads / 32)
        for (int d = lane; d < 256; d += 32) chunk[c][d] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * kRTile;
    uint64_t key[kRItems];
    uint32_t id[kRItems], dig[kRItems], rk[kRItems];
#pragma unroll
    for (int r = 0; r < kRItems; ++r) {
        const uint32_t i = base + r * kRThreads + threadIdx.x;
        const bool valid = i < n;
        key[r] = valid ? kin[i] : 0;
        id[r] = valid ? iin[i] : 0;
        dig[r] = valid ? digit_of(key[r], id[r], pass, seg_off, n_seg) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, dig[r]);
        rk[r] = __popc(peers & lanemask_lt());
        if (valid && rk[r] == 0) chunk[r * (kRThreads / 32) + warp][dig[r]] = (uint16_t)__popc(peers);
    }
    __syncthreads();
    {
        const uint32_t d = threadIdx.x;
        uint32_t run = 0;
        for (int c = 0; c < kRChunks; ++c) {
            const uint32_t v = chunk[c][d];
            chunk[c][d] = (uint16_t)run;
            run += v;
        }
        dbase[d] = scanned[d * nblocks + blockIdx.x];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kRItems; ++r) {
        if (dig[r] < 256u) {
            const uint32_t pos = dbase[dig[r]] + chunk[r * (kRThreads / 32) + warp][dig[r]] + rk[r];
            kout[pos] = key[r];
            iout[pos] = id[r];
        }
    }
}

__global__ void radix_flip_kernel(RadixState* st) {
    if (!st->skip) st->cur ^= 1u;
    st->skip = 0;
}

__global__ void __launch_bounds__(256) radix_gather_kernel(const uint4* __restrict__ hits, uint4* __restrict__ out,
                                                           uint32_t* __restrict__ perm,
                                                           const uint32_t* __restrict__ idx0,
                                                           const uint32_t* __restrict__ idx1,
                                                           const RadixState* __restrict__ st, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t src = (st->cur ? idx1 : idx0)[i];
    out[i] = __ldg(hits + src);
    if (perm) perm[i] = src;
}

void radix_plan(Arena& a, uint32_t n, RadixPlan& p) {
    p.nblocks = div_up(n, kRTile);
    p.keys0 = a.take<uint64_t>(n);
    p.keys1 = a.take<uint64_t>(n);
    p.idx0 = a.take<uint32_t>(n);
    p.idx1 = a.take<uint32_t>(n);
    p.hist = a.take<uint32_t>((size_t)256 * p.nblocks);
    p.scan_scratch = a.take<uint32_t>(scan_ws_count(256u * p.nblocks));
    p.st = a.take<RadixState>(1);
}

// LSD passes [pass_begin, pass_end) over the (key, index) pairs of the plan; st->cur says where they end up
int radix_run_passes(const RadixPlan& p, uint32_t n, int pass_begin, int pass_end, const uint32_t* d_seg_offsets,
                     uint32_t n_seg, cudaStream_t s) {
    for (int pass = pass_begin; pass < pass_end; ++pass) {
        prof_mark(s, "sort.radix_hist");
        TT_K(radix_hist_kernel)<<<p.nblocks, kRThreads, 0, s>>>(p.keys0, p.keys1, p.idx0, p.idx1, n, pass, d_seg_offsets,
                                                          n_seg, p.st, p.hist, p.nblocks);
        prof_mark(s, "sort.radix_scan");
        int rc = exclusive_scan_u32(p.hist, p.hist, 256u * p.nblocks, p.scan_scratch, nullptr, s);
        if (rc != TT_OK) return rc;
        TT_K(radix_decide_kernel)<<<1, 256, 0, s>>>(p.hist, p.nblocks, n, p.st);
        prof_mark(s, "sort.radix_scatter");
        TT_K(radix_scatter_kernel)<<<p.nblocks, kRThreads, 0, s>>>(p.keys0, p.keys1, p.idx0, p.idx1, n, pass,
                                                             d_seg_offsets, n_seg, p.st, p.hist, p.nblocks);
        TT_K(radix_flip_kernel)<<<1, 1, 0, s>>>(p.st);
    }
    return TT_OK;
}

size_t radix_ws_bytes(uint32_t n) {
    Arena a(nullptr);
    RadixPlan p;
    radix_plan(a, n, p);
    return a.off;
}

int radix_sort(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
               uint32_t n_seg, void* d_ws, cudaStream_t s) {
    if (n == 0) return TT_OK;
    Arena a(d_ws);
    RadixPlan p;
    radix_plan(a, n, p);
    const uint32_t nb256 = div_up(n, 256);
    prof_mark(s, "sort.radix_extract");
    TT_K(radix_extract_kernel)<<<nb256, 256, 0, s>>>((const uint4*)d_in, p.keys0, p.idx0, n, p.st);
    int seg_passes = 0;
    for (uint32_t v = n_seg - 1; v; v >>= 8) ++seg_passes;
    const int rc = radix_run_passes(p, n, 0, 8 + seg_passes, d_seg_offsets, n_seg, s);
    if (rc != TT_OK) return rc;
    prof_mark(s, "sort.radix_gather");
    TT_K(radix_gather_kernel)<<<nb256, 256, 0, s>>>((const uint4*)d_in, (uint4*)d_out, d_perm, p.idx0, p.idx1, p.st, n);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

}  // namespace tt
