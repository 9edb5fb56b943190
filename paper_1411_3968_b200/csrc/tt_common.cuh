// tt_common.cuh -- shared device/host helpers of libtt (CUDA path only; the oracle shares nothing with this).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tt.h"

#define TT_CUDA_OK(expr)                          \
    do {                                          \
        cudaError_t e__ = (expr);                 \
        if (e__ != cudaSuccess) return TT_E_CUDA; \
    } while (0)
#define TT_LAUNCH_OK()                                       \
    do {                                                     \
        if (cudaPeekAtLastError() != cudaSuccess) {          \
            (void)cudaGetLastError();                        \
            return TT_E_CUDA;                                \
        }                                                    \
    } while (0)

namespace tt {

// Per-device one-time set-up (cudaFuncSetAttribute is per device): runs fn() once for (current device, slot), under a
// lock, so a second GPU or a second host thread never launches before the attributes are set (tt_api.cu).
enum { kSlotMerge = 0, kSlotTrigger = 1, kSlotPairs = 2 };
int once_per_device(int slot, int (*fn)());
int sm_count();  // SMs of the current device (cached per device)

// ---- launch counter and stage profiler (tt_prof.cu) ------------------------------------------------
void count_launch();                                // every kernel launch of the library goes through TT_K
void prof_mark(cudaStream_t s, const char* name);   // no-op unless tt_prof_enable(1): records an event that
                                                    // opens stage `name` (and closes the previous one)
void prof_end(cudaStream_t s);                      // closes the current stage
void prof_counter(cudaStream_t s, const char* name, const uint32_t* d_value);  // samples a device counter (profiling only)
#define TT_K(k) tt::count_launch(), k

struct tt_geometry_dev {  // device view of the causality table
    const int32_t* pair_block;  // [n_tower*n_tower]
    const int32_t* blocks;      // [n_blocks][ppt][ppt]
    uint32_t n_pmt, n_tower, ppt, n_blocks;
    int32_t max_dt;  // max entry over all connected blocks (-1: no edge anywhere)
};

// Bump allocator over the caller's workspace; 256-byte granules.  Used twice with identical call
// sequences: once with base = nullptr to size, once to carve.
struct Arena {
    char* base;
    size_t off;
    explicit Arena(void* b) : base((char*)b), off(0) {}
    template <typename T>
    T* take(size_t count) {
        size_t bytes = (count * sizeof(T) + 255) & ~size_t(255);
        T* p = base ? (T*)(base + off) : nullptr;
        off += bytes;
        return p;
    }
};

static inline uint32_t div_up(uint64_t a, uint64_t b) { return (uint32_t)((a + b - 1) / b); }

// ---- device helpers ------------------------------------------------------------------------------
struct HitView {
    int64_t t;
    uint32_t pmt, floor, charge, pad;
};
__device__ __forceinline__ HitView unpack(const uint4& v) {
    HitView h;
    h.t = (int64_t)(((uint64_t)v.y << 32) | (uint64_t)v.x);
    h.pmt = v.z & 0xFFFFu;
    h.floor = v.z >> 16;
    h.charge = v.w & 0xFFFFu;
    h.pad = v.w >> 16;
    return h;
}
__device__ __forceinline__ int64_t hit_time(const uint4& v) { return (int64_t)(((uint64_t)v.y << 32) | (uint64_t)v.x); }
// order-preserving map int64 -> uint64
__device__ __forceinline__ uint64_t key_of(int64_t t) { return (uint64_t)t ^ 0x8000000000000000ull; }
// |a-b| for a >= b as unsigned (exact for any int64 pair)
__device__ __forceinline__ uint64_t udiff(int64_t hi, int64_t lo) { return (uint64_t)hi - (uint64_t)lo; }

__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// segment s with off[s] <= i < off[s+1] (empty segments skipped): upper_bound(off, i) - 1
__device__ __forceinline__ uint32_t find_segment(const uint32_t* __restrict__ off, uint32_t n_seg, uint32_t i) {
    uint32_t lo = 0, hi = n_seg;  // invariant: off[lo] <= i, off[hi] > i (off[n_seg] = n > i)
    while (hi - lo > 1) {
        uint32_t mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// block-wide exclusive scan of one uint32 per thread (blockDim.x multiple of 32, <= 1024).
// sm must hold 33 uint32.  Returns the exclusive prefix; *total = block sum.
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* sm, uint32_t* total) {
    const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= (uint32_t)d) inc += o;
    }
    if (lane == 31) sm[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t s = lane < nw ? sm[lane] : 0u;
        uint32_t si = s;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t o = __shfl_up_sync(0xffffffffu, si, d);
            if (lane >= (uint32_t)d) si += o;
        }
        sm[lane] = si - s;  // exclusive warp offsets
        if (lane == 31) sm[32] = si;
    }
    __syncthreads();
    uint32_t r = sm[w] + inc - v;
    *total = sm[32];
    __syncthreads();  // sm reusable after return
    return r;
}

// ---- device-wide exclusive scan of a uint32 array of host-known length (tt_scan.cu) ----------------
size_t scan_ws_count(uint32_t n);  // number of uint32 of scratch needed
// out may alias in.  total (nullable) receives the sum.
int exclusive_scan_u32(const uint32_t* in, uint32_t* out, uint32_t n, uint32_t* scratch, uint32_t* total,
                       cudaStream_t s);

}  // namespace tt

// opaque handle of the C ABI
struct tt_geometry {
    tt::tt_geometry_dev dev;
    int32_t* d_pair_block;
    int32_t* d_blocks;
};
