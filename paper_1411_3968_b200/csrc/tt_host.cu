// tt_host.cu -- host-buffer convenience wrapper over the three hot calls (end-to-end path).
#include <cstdlib>

#include "tt_common.cuh"

struct tt_host_ctx {
    uint32_t max_n, max_seg, max_runs, seed_cap, event_cap;
    cudaStream_t stream;
    tt_hit *d_in, *d_sorted;
    uint8_t* d_flags;
    uint32_t *d_seg, *d_runs, *d_seeds, *d_counts;  // d_counts: n_seeds, n_events, status
    tt_event* d_events;
    void* d_ws;
    size_t ws_bytes;
};

static size_t max_sz(size_t a, size_t b) { return a > b ? a : b; }

extern "C" int tt_host_ctx_destroy(tt_host_ctx* c) {
    if (!c) return TT_OK;
    cudaFree(c->d_in); cudaFree(c->d_sorted); cudaFree(c->d_flags); cudaFree(c->d_seg); cudaFree(c->d_runs);
    cudaFree(c->d_seeds); cudaFree(c->d_counts); cudaFree(c->d_events); cudaFree(c->d_ws);
    if (c->stream) cudaStreamDestroy(c->stream);
    std::free(c);
    (void)cudaGetLastError();
    return TT_OK;
}

extern "C" int tt_host_ctx_create(tt_host_ctx** out, uint32_t max_n, uint32_t max_seg, uint32_t max_runs,
                                  uint32_t seed_cap, uint32_t event_cap) {
    if (!out || max_seg < 1 || max_n >= 0xFFF00000u) return TT_E_INVAL;
    tt_host_ctx* c = (tt_host_ctx*)std::calloc(1, sizeof(tt_host_ctx));
    if (!c) return TT_E_INVAL;
    c->max_n = max_n; c->max_seg = max_seg; c->max_runs = max_runs; c->seed_cap = seed_cap; c->event_cap = event_cap;
    // worst-case workspace: the radix path bounds the merge path; sized by querying with trivial offsets
    uint32_t seg1[2] = {0, max_n};
    size_t ws_sort = 0, ws_trig = 0, ws_ev = 0;
    tt_params p = {20000, 3000000, 3000000, 5, 0, 300, 0};
    tt_geometry dummy = {};
    int rc = tt_sort_slice(nullptr, nullptr, nullptr, max_n, nullptr, seg1, 1, nullptr, nullptr, 0, nullptr, &ws_sort,
                           nullptr, nullptr);
    if (rc == TT_OK)
        rc = tt_trigger_slice(nullptr, max_n, nullptr, seg1, 1, &dummy, &p, nullptr, nullptr, seed_cap, nullptr, nullptr,
                              &ws_trig, nullptr, nullptr);
    if (rc == TT_OK)
        rc = tt_extract_events(nullptr, max_n, nullptr, seg1, 1, nullptr, nullptr, seed_cap, &p, nullptr, event_cap,
                               nullptr, nullptr, nullptr, nullptr, nullptr, &ws_ev, nullptr, nullptr);
    if (rc != TT_OK) { std::free(c); return rc; }
    // the run-merge path may need more than the radix path: leave head-room, checked again per call
    c->ws_bytes = max_sz(max_sz(ws_sort + ws_sort / 2, ws_trig), ws_ev) + (1u << 20);
    const size_t nn = max_n ? max_n : 1;
    bool ok = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) == cudaSuccess &&
              cudaMalloc(&c->d_in, nn * sizeof(tt_hit)) == cudaSuccess &&
              cudaMalloc(&c->d_sorted, nn * sizeof(tt_hit)) == cudaSuccess &&
              cudaMalloc(&c->d_flags, nn) == cudaSuccess &&
              cudaMalloc(&c->d_seg, ((size_t)max_seg + 1) * 4) == cudaSuccess &&
              cudaMalloc(&c->d_runs, ((size_t)max_runs + 1) * 4) == cudaSuccess &&
              cudaMalloc(&c->d_seeds, ((size_t)seed_cap + 1) * 4) == cudaSuccess &&
              cudaMalloc(&c->d_counts, 4 * 4) == cudaSuccess &&
              cudaMalloc(&c->d_events, ((size_t)event_cap + 1) * sizeof(tt_event)) == cudaSuccess &&
              cudaMalloc(&c->d_ws, c->ws_bytes) == cudaSuccess;
    if (!ok) { tt_host_ctx_destroy(c); return TT_E_CUDA; }
    *out = c;
    return TT_OK;
}

extern "C" int tt_process_host(tt_host_ctx* c, const tt_hit* h_in, tt_hit* h_sorted, uint8_t* h_flags, uint32_t n,
                               const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* h_run_offsets,
                               uint32_t n_runs, const tt_geometry* g, const tt_params* p, uint32_t* h_seeds,
                               tt_event* h_events, uint32_t* h_counts) {
    if (!c || !h_seg_offsets || !g || !p || !h_counts || (n && !h_in)) return TT_E_INVAL;
    if (n > c->max_n || n_seg > c->max_seg || n_seg < 1 || (h_run_offsets && n_runs > c->max_runs)) return TT_E_INVAL;
    cudaStream_t s = c->stream;
    int32_t* d_status = (int32_t*)(c->d_counts + 2);
    TT_CUDA_OK(cudaMemsetAsync(c->d_counts, 0, 16, s));
    TT_CUDA_OK(cudaMemcpyAsync(c->d_seg, h_seg_offsets, ((size_t)n_seg + 1) * 4, cudaMemcpyHostToDevice, s));
    if (h_run_offsets)
        TT_CUDA_OK(cudaMemcpyAsync(c->d_runs, h_run_offsets, ((size_t)n_runs + 1) * 4, cudaMemcpyHostToDevice, s));
    if (n) TT_CUDA_OK(cudaMemcpyAsync(c->d_in, h_in, (size_t)n * sizeof(tt_hit), cudaMemcpyHostToDevice, s));
    size_t ws = c->ws_bytes;
    int rc = tt_sort_slice(c->d_in, c->d_sorted, nullptr, n, c->d_seg, h_seg_offsets, n_seg,
                           h_run_offsets ? c->d_runs : nullptr, h_run_offsets, h_run_offsets ? n_runs : 0, c->d_ws, &ws,
                           d_status, s);
    if (rc != TT_OK) return rc;
    ws = c->ws_bytes;
    rc = tt_trigger_slice(c->d_sorted, n, c->d_seg, h_seg_offsets, n_seg, g, p, c->d_flags, c->d_seeds, c->seed_cap,
                          c->d_counts, c->d_ws, &ws, d_status, s);
    if (rc != TT_OK) return rc;
    ws = c->ws_bytes;
    rc = tt_extract_events(c->d_sorted, n, c->d_seg, h_seg_offsets, n_seg, c->d_seeds, c->d_counts, c->seed_cap, p,
                           c->d_events, c->event_cap, c->d_counts + 1, c->d_flags, nullptr, nullptr, c->d_ws, &ws,
                           d_status, s);
    if (rc != TT_OK) return rc;
    TT_CUDA_OK(cudaMemcpyAsync(h_counts, c->d_counts, 12, cudaMemcpyDeviceToHost, s));
    if (h_sorted && n) TT_CUDA_OK(cudaMemcpyAsync(h_sorted, c->d_sorted, (size_t)n * sizeof(tt_hit), cudaMemcpyDeviceToHost, s));
    if (h_flags && n) TT_CUDA_OK(cudaMemcpyAsync(h_flags, c->d_flags, n, cudaMemcpyDeviceToHost, s));
    TT_CUDA_OK(cudaStreamSynchronize(s));
    const uint32_t ns = h_counts[0] < c->seed_cap ? h_counts[0] : c->seed_cap;
    const uint32_t ne = h_counts[1] < c->event_cap ? h_counts[1] : c->event_cap;
    if (h_seeds && ns) TT_CUDA_OK(cudaMemcpyAsync(h_seeds, c->d_seeds, (size_t)ns * 4, cudaMemcpyDeviceToHost, s));
    if (h_events && ne)
        TT_CUDA_OK(cudaMemcpyAsync(h_events, c->d_events, (size_t)ne * sizeof(tt_event), cudaMemcpyDeviceToHost, s));
    TT_CUDA_OK(cudaStreamSynchronize(s));
    return TT_OK;
}
