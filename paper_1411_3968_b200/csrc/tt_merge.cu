// tt_merge.cu -- sort of P concatenated, individually time-ordered runs (the per-PMT streams,
// "our data ... is time-ordered for single PMT").
// v0: verifies the runs and falls through to the general radix path.
#include "tt_common.cuh"

namespace tt {
size_t radix_ws_bytes(uint32_t n);
int radix_sort(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
               uint32_t n_seg, void* d_ws, cudaStream_t s);

// run r with off[r] <= i < off[r+1]
__global__ void __launch_bounds__(256) run_check_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                        const uint32_t* __restrict__ run_off, uint32_t n_runs,
                                                        int32_t* __restrict__ status) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (i > 0 && i < n) {
        const uint32_t r = find_segment(run_off, n_runs, i);
        if (__ldg(run_off + r) != i) bad = hit_time(__ldg(hits + i)) < hit_time(__ldg(hits + i - 1));
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(status, TT_S_RUN_UNSORTED);
}

size_t merge_ws_bytes(uint32_t n, const uint32_t*, uint32_t, const uint32_t*, uint32_t) { return radix_ws_bytes(n); }

int merge_sort_runs(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
                    const uint32_t*, uint32_t n_seg, const uint32_t* d_run_offsets, const uint32_t*, uint32_t n_runs,
                    void* d_ws, int32_t* d_status, cudaStream_t s) {
    prof_mark(s, "sort.run_check");
    TT_K(run_check_kernel)<<<div_up(n, 256), 256, 0, s>>>((const uint4*)d_in, n, d_run_offsets, n_runs, d_status);
    return radix_sort(d_in, d_out, d_perm, n, d_seg_offsets, n_seg, d_ws, s);
}
}  // namespace tt
