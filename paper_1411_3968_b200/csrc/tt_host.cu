// tt_host.cu -- host-buffer wrapper over the hot calls (end-to-end path): tt_sort_trigger_slice -> tt_extract_events
// with the copies around them.  Successive slices arrive back to back, so the context is two slots deep:
// tt_host_submit enqueues the upload of a slice on a copy stream, its compute on a compute stream and the read-back of
// its results on a third stream and returns; the upload of slice k + 1 then runs while slice k computes and slice k - 1
// is read back (PCIe is full duplex).  tt_host_wait returns the oldest submitted slice.  tt_process_host = submit + wait.
#include <cstdlib>

#include "tt_common.cuh"

namespace {

struct Slot {
    tt_hit* d_in;
    uint8_t* d_flags;
    uint32_t *d_seg, *d_runs, *d_seeds, *d_counts;  // d_counts: n_seeds, n_events, status
    tt_event* d_events;
    cudaEvent_t up_done, cmp_done, down_done;
    bool busy, wants_sorted;
    uint32_t* h_seeds;
    tt_event* h_events;
    uint32_t* h_counts;
    uint32_t* h_counts_pinned;  // [4] pinned staging of the counts
};

}  // namespace

struct tt_host_ctx {
    uint32_t max_n, max_seg, max_runs, seed_cap, event_cap;
    cudaStream_t s_up, s_cmp, s_down, s_tail;  // s_tail: the seeds / events read-back of tt_host_wait (must not queue
                                                // behind the NEXT slice's read-back on s_down)
    tt_hit* d_sorted;
    void* d_ws;
    size_t ws_bytes;
    Slot slot[2];
    uint32_t head, tail;  // submitted slices are head .. tail - 1 (mod 2 slots)
    bool sorted_in_flight;  // the last submitted slice reads d_sorted back: the next compute waits for it
    cudaEvent_t sorted_read;
};

static size_t max_sz(size_t a, size_t b) { return a > b ? a : b; }

extern "C" int tt_host_ctx_destroy(tt_host_ctx* c) {
    if (!c) return TT_OK;
    cudaDeviceSynchronize();
    for (int k = 0; k < 2; ++k) {
        Slot& s = c->slot[k];
        cudaFree(s.d_in); cudaFree(s.d_flags); cudaFree(s.d_seg); cudaFree(s.d_runs); cudaFree(s.d_seeds);
        cudaFree(s.d_counts); cudaFree(s.d_events);
        if (s.h_counts_pinned) cudaFreeHost(s.h_counts_pinned);
        if (s.up_done) cudaEventDestroy(s.up_done);
        if (s.cmp_done) cudaEventDestroy(s.cmp_done);
        if (s.down_done) cudaEventDestroy(s.down_done);
    }
    cudaFree(c->d_sorted); cudaFree(c->d_ws);
    if (c->sorted_read) cudaEventDestroy(c->sorted_read);
    if (c->s_up) cudaStreamDestroy(c->s_up);
    if (c->s_cmp) cudaStreamDestroy(c->s_cmp);
    if (c->s_down) cudaStreamDestroy(c->s_down);
    if (c->s_tail) cudaStreamDestroy(c->s_tail);
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
    // first workspace: the radix path of the fused call and the events; the run-merge plan of a real slice may need
    // more -- checked per call, and the workspace grows then (not a hot path: once per new plan)
    uint32_t seg1[2] = {0, max_n};
    size_t ws_f = 0, ws_ev = 0;
    tt_params p = {20000, 3000000, 3000000, 5, 0, 300, 0};
    tt_geometry dummy = {};
    int rc = tt_sort_trigger_slice(nullptr, nullptr, nullptr, max_n, nullptr, seg1, 1, nullptr, nullptr, 0, &dummy, &p, nullptr,
                                   nullptr, seed_cap, nullptr, nullptr, &ws_f, nullptr, nullptr);
    if (rc == TT_OK)
        rc = tt_extract_events(nullptr, max_n, nullptr, seg1, 1, nullptr, nullptr, seed_cap, &p, nullptr, event_cap,
                               nullptr, nullptr, nullptr, nullptr, nullptr, &ws_ev, nullptr, nullptr);
    if (rc != TT_OK) { std::free(c); return rc; }
    c->ws_bytes = max_sz(ws_f, ws_ev) + (1u << 20);
    const size_t nn = max_n ? max_n : 1;
    bool ok = cudaStreamCreateWithFlags(&c->s_up, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_cmp, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_down, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_tail, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->sorted_read, cudaEventDisableTiming) == cudaSuccess &&
              cudaMalloc(&c->d_sorted, nn * sizeof(tt_hit)) == cudaSuccess && cudaMalloc(&c->d_ws, c->ws_bytes) == cudaSuccess;
    for (int k = 0; ok && k < 2; ++k) {
        Slot& s = c->slot[k];
        ok = cudaMalloc(&s.d_in, nn * sizeof(tt_hit)) == cudaSuccess && cudaMalloc(&s.d_flags, nn) == cudaSuccess &&
             cudaMalloc(&s.d_seg, ((size_t)max_seg + 1) * 4) == cudaSuccess &&
             cudaMalloc(&s.d_runs, ((size_t)max_runs + 1) * 4) == cudaSuccess &&
             cudaMalloc(&s.d_seeds, ((size_t)seed_cap + 1) * 4) == cudaSuccess &&
             cudaMalloc(&s.d_counts, 4 * 4) == cudaSuccess &&
             cudaMalloc(&s.d_events, ((size_t)event_cap + 1) * sizeof(tt_event)) == cudaSuccess &&
             cudaMallocHost(&s.h_counts_pinned, 4 * 4) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.up_done, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.cmp_done, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.down_done, cudaEventDisableTiming) == cudaSuccess;
    }
    if (!ok) { tt_host_ctx_destroy(c); return TT_E_CUDA; }
    *out = c;
    return TT_OK;
}

extern "C" int tt_host_submit(tt_host_ctx* c, const tt_hit* h_in, tt_hit* h_sorted, uint8_t* h_flags, uint32_t n,
                              const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* h_run_offsets,
                              uint32_t n_runs, const tt_geometry* g, const tt_params* p, uint32_t* h_seeds,
                              tt_event* h_events, uint32_t* h_counts) {
    if (!c || !h_seg_offsets || !g || !p || !h_counts || (n && !h_in)) return TT_E_INVAL;
    if (n > c->max_n || n_seg > c->max_seg || n_seg < 1 || (h_run_offsets && n_runs > c->max_runs)) return TT_E_INVAL;
    if (c->tail - c->head >= 2u) return TT_E_INVAL;  // both slots in flight: tt_host_wait first
    Slot& sl = c->slot[c->tail & 1u];
    // workspace for this slice's plan
    size_t need_f = 0, need_e = 0;
    int rc = tt_sort_trigger_slice(nullptr, nullptr, nullptr, n, nullptr, h_seg_offsets, n_seg,
                                   h_run_offsets ? (const uint32_t*)sl.d_runs : nullptr, h_run_offsets,
                                   h_run_offsets ? n_runs : 0, g, p, nullptr, nullptr, c->seed_cap, nullptr, nullptr, &need_f,
                                   nullptr, nullptr);
    if (rc != TT_OK) return rc;
    rc = tt_extract_events(nullptr, n, nullptr, h_seg_offsets, n_seg, nullptr, nullptr, c->seed_cap, p, nullptr,
                           c->event_cap, nullptr, nullptr, nullptr, nullptr, nullptr, &need_e, nullptr, nullptr);
    if (rc != TT_OK) return rc;
    if (max_sz(need_f, need_e) > c->ws_bytes) {  // a deeper merge plan than the context was sized for: grow once
        TT_CUDA_OK(cudaDeviceSynchronize());
        cudaFree(c->d_ws);
        c->d_ws = nullptr;
        c->ws_bytes = max_sz(need_f, need_e) + (1u << 20);
        TT_CUDA_OK(cudaMalloc(&c->d_ws, c->ws_bytes));
    }
    int32_t* d_status = (int32_t*)(sl.d_counts + 2);
    // upload
    TT_CUDA_OK(cudaMemcpyAsync(sl.d_seg, h_seg_offsets, ((size_t)n_seg + 1) * 4, cudaMemcpyHostToDevice, c->s_up));
    if (h_run_offsets)
        TT_CUDA_OK(cudaMemcpyAsync(sl.d_runs, h_run_offsets, ((size_t)n_runs + 1) * 4, cudaMemcpyHostToDevice, c->s_up));
    if (n) TT_CUDA_OK(cudaMemcpyAsync(sl.d_in, h_in, (size_t)n * sizeof(tt_hit), cudaMemcpyHostToDevice, c->s_up));
    TT_CUDA_OK(cudaEventRecord(sl.up_done, c->s_up));
    // compute (one compute stream: slices run one after the other and share d_sorted and the workspace)
    TT_CUDA_OK(cudaStreamWaitEvent(c->s_cmp, sl.up_done, 0));
    if (c->sorted_in_flight) TT_CUDA_OK(cudaStreamWaitEvent(c->s_cmp, c->sorted_read, 0));
    TT_CUDA_OK(cudaMemsetAsync(sl.d_counts, 0, 16, c->s_cmp));
    size_t ws = c->ws_bytes;
    rc = tt_sort_trigger_slice(sl.d_in, c->d_sorted, nullptr, n, sl.d_seg, h_seg_offsets, n_seg,
                               h_run_offsets ? sl.d_runs : nullptr, h_run_offsets, h_run_offsets ? n_runs : 0, g, p,
                               sl.d_flags, sl.d_seeds, c->seed_cap, sl.d_counts, c->d_ws, &ws, d_status, c->s_cmp);
    if (rc != TT_OK) return rc;
    ws = c->ws_bytes;
    rc = tt_extract_events(c->d_sorted, n, sl.d_seg, h_seg_offsets, n_seg, sl.d_seeds, sl.d_counts, c->seed_cap, p,
                           sl.d_events, c->event_cap, sl.d_counts + 1, sl.d_flags, nullptr, nullptr, c->d_ws, &ws, d_status,
                           c->s_cmp);
    if (rc != TT_OK) return rc;
    TT_CUDA_OK(cudaEventRecord(sl.cmp_done, c->s_cmp));
    // read-back of what has a size known on the host; seeds and events follow in tt_host_wait
    TT_CUDA_OK(cudaStreamWaitEvent(c->s_down, sl.cmp_done, 0));
    TT_CUDA_OK(cudaMemcpyAsync(sl.h_counts_pinned, sl.d_counts, 12, cudaMemcpyDeviceToHost, c->s_down));
    if (h_flags && n) TT_CUDA_OK(cudaMemcpyAsync(h_flags, sl.d_flags, n, cudaMemcpyDeviceToHost, c->s_down));
    c->sorted_in_flight = false;
    if (h_sorted && n) {
        TT_CUDA_OK(cudaMemcpyAsync(h_sorted, c->d_sorted, (size_t)n * sizeof(tt_hit), cudaMemcpyDeviceToHost, c->s_down));
        TT_CUDA_OK(cudaEventRecord(c->sorted_read, c->s_down));
        c->sorted_in_flight = true;
    }
    TT_CUDA_OK(cudaEventRecord(sl.down_done, c->s_down));
    sl.busy = true;
    sl.h_seeds = h_seeds; sl.h_events = h_events; sl.h_counts = h_counts;
    ++c->tail;
    return TT_OK;
}

extern "C" int tt_host_wait(tt_host_ctx* c) {
    if (!c || c->head == c->tail) return TT_E_INVAL;
    Slot& sl = c->slot[c->head & 1u];
    TT_CUDA_OK(cudaEventSynchronize(sl.down_done));
    for (int k = 0; k < 3; ++k) sl.h_counts[k] = sl.h_counts_pinned[k];
    const uint32_t ns = sl.h_counts[0] < c->seed_cap ? sl.h_counts[0] : c->seed_cap;
    const uint32_t ne = sl.h_counts[1] < c->event_cap ? sl.h_counts[1] : c->event_cap;
    if (sl.h_seeds && ns) TT_CUDA_OK(cudaMemcpyAsync(sl.h_seeds, sl.d_seeds, (size_t)ns * 4, cudaMemcpyDeviceToHost, c->s_tail));
    if (sl.h_events && ne)
        TT_CUDA_OK(cudaMemcpyAsync(sl.h_events, sl.d_events, (size_t)ne * sizeof(tt_event), cudaMemcpyDeviceToHost, c->s_tail));
    TT_CUDA_OK(cudaStreamSynchronize(c->s_tail));
    sl.busy = false;
    ++c->head;
    return TT_OK;
}

extern "C" int tt_process_host(tt_host_ctx* c, const tt_hit* h_in, tt_hit* h_sorted, uint8_t* h_flags, uint32_t n,
                               const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* h_run_offsets,
                               uint32_t n_runs, const tt_geometry* g, const tt_params* p, uint32_t* h_seeds,
                               tt_event* h_events, uint32_t* h_counts) {
    if (c && c->head != c->tail) return TT_E_INVAL;  // slices in flight: this call is the synchronous form
    const int rc = tt_host_submit(c, h_in, h_sorted, h_flags, n, h_seg_offsets, n_seg, h_run_offsets, n_runs, g, p, h_seeds,
                                  h_events, h_counts);
    if (rc != TT_OK) return rc;
    return tt_host_wait(c);
}
