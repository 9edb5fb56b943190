// tt_events.cu -- event-window merge, INEVT tagging and the optional gather.
//   PAPER.md:23 "a 6 us time window of the tower data (centered at the time of the trigger seed) is sent
//   to the Event Manager"; "all hits within +-3 us are tagged to be saved".
//   Readings R11-R13: every L2 hit is a seed; closed windows, merge <=> gap <= 2H;
//   never across a segment; t_start / t_end unclipped.
#include "tt_common.cuh"

#include <mutex>

namespace tt {

constexpr int kEvBlocks = 592;  // fixed grid: the seed count lives on the device
constexpr int kEvThreads = 256;

__device__ __forceinline__ void ev_chunk(uint32_t m, uint32_t& c0, uint32_t& c1) {
    const uint32_t per = (m + gridDim.x - 1) / gridDim.x;
    const uint64_t a = (uint64_t)blockIdx.x * per;
    c0 = a < m ? (uint32_t)a : m;
    c1 = a + per < m ? (uint32_t)(a + per) : m;
}

struct SegCtx {
    const uint32_t* off;
    uint32_t n_seg, n;
};

// seed k opens a new event?
__device__ __forceinline__ bool is_head(const uint4* __restrict__ hits, const uint32_t* __restrict__ seeds, uint32_t k,
                                        const SegCtx& sc, uint64_t twoH) {
    if (k == 0) return true;
    const uint32_t i0 = seeds[k - 1], i1 = seeds[k];
    if (sc.n_seg > 1 && find_segment(sc.off, sc.n_seg, i0) != find_segment(sc.off, sc.n_seg, i1)) return true;
    return udiff(hit_time(__ldg(hits + i1)), hit_time(__ldg(hits + i0))) > twoH;
}

__global__ void __launch_bounds__(kEvThreads) ev_count_kernel(const uint4* __restrict__ hits,
                                                              const uint32_t* __restrict__ seeds,
                                                              const uint32_t* __restrict__ n_seeds_ptr, uint32_t seed_cap,
                                                              SegCtx sc, uint64_t twoH, uint32_t* __restrict__ cnt,
                                                              uint8_t* __restrict__ head) {
    const uint32_t ns = min(*n_seeds_ptr, seed_cap);
    uint32_t c0, c1;
    ev_chunk(ns, c0, c1);
    uint32_t c = 0;
    for (uint32_t k = c0 + threadIdx.x; k < c1; k += kEvThreads) {  // the only pass that gathers the seed times
        const bool h = is_head(hits, seeds, k, sc, twoH);
        head[k] = h ? 1 : 0;
        c += h ? 1u : 0u;
    }
    __shared__ uint32_t sm[33];
    uint32_t total;
    block_exclusive_scan(c, sm, &total);
    if (threadIdx.x == 0) cnt[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) ev_scan_kernel(uint32_t* __restrict__ cnt, uint32_t nb,
                                                       uint32_t* __restrict__ n_out, uint32_t cap,
                                                       int32_t* __restrict__ status) {
    __shared__ uint32_t sm[33];
    uint32_t carry = 0;
    for (uint32_t base = 0; base < nb; base += 1024) {
        const uint32_t i = base + threadIdx.x;
        const uint32_t v = i < nb ? cnt[i] : 0u;
        uint32_t total;
        const uint32_t ex = block_exclusive_scan(v, sm, &total);
        if (i < nb) cnt[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) {
        *n_out = carry;
        if (carry > cap) atomicOr(status, TT_S_EVENT_OVERFLOW);
    }
}

// lower_bound: first i in [a, b) with t[i] >= v  (signed compare)
__device__ __forceinline__ uint32_t lb_time(const uint4* __restrict__ hits, uint32_t a, uint32_t b, int64_t v) {
    while (a < b) {
        const uint32_t mid = a + ((b - a) >> 1);
        if (hit_time(__ldg(hits + mid)) < v) a = mid + 1; else b = mid;
    }
    return a;
}
// upper_bound: first i in [a, b) with t[i] > v
__device__ __forceinline__ uint32_t ub_time(const uint4* __restrict__ hits, uint32_t a, uint32_t b, int64_t v) {
    while (a < b) {
        const uint32_t mid = a + ((b - a) >> 1);
        if (hit_time(__ldg(hits + mid)) <= v) a = mid + 1; else b = mid;
    }
    return a;
}

// heads write {t_start, hit_begin, seed_begin}; tails write {t_end, hit_end, n_seeds := k+1 (fixed below)}
__global__ void __launch_bounds__(kEvThreads) ev_write_kernel(const uint4* __restrict__ hits,
                                                              const uint32_t* __restrict__ seeds,
                                                              const uint32_t* __restrict__ n_seeds_ptr, uint32_t seed_cap,
                                                              SegCtx sc, uint64_t twoH, int64_t H,
                                                              const uint32_t* __restrict__ off,
                                                              const uint8_t* __restrict__ head_flag,
                                                              tt_event* __restrict__ events, uint32_t event_cap) {
    __shared__ uint32_t sm[33];
    const uint32_t ns = min(*n_seeds_ptr, seed_cap);
    uint32_t c0, c1;
    ev_chunk(ns, c0, c1);
    uint32_t run = off[blockIdx.x];
    for (uint32_t base = c0; base < c1; base += kEvThreads) {
        const uint32_t k = base + threadIdx.x;
        const bool valid = k < c1;
        const bool head = valid && head_flag[k] != 0;
        uint32_t total;
        const uint32_t r = block_exclusive_scan(head ? 1u : 0u, sm, &total);
        if (valid) {
            const uint32_t e = run + r + (head ? 1u : 0u) - 1u;  // inclusive count - 1 (event 0 starts at seed 0)
            const bool tail = (k + 1 == ns) || head_flag[k + 1] != 0;
            if ((head || tail) && e < event_cap) {
                const uint32_t i = seeds[k];
                const int64_t t = hit_time(__ldg(hits + i));
                // the hit ranges are searched by ev_fix_kernel (one thread per event, all in parallel): here only
                // the seed's own hit index is left in hit_begin / hit_end
                if (head) {
                    events[e].t_start = (int64_t)((uint64_t)t - (uint64_t)H);
                    events[e].hit_begin = i;
                    events[e].seed_begin = k;
                }
                if (tail) {
                    events[e].t_end = (int64_t)((uint64_t)t + (uint64_t)H);
                    events[e].hit_end = i;
                    events[e].n_seeds = k + 1;  // end index; turned into a count by ev_fix_kernel
                }
            }
        }
        run += total;
    }
}

// one thread per event: seed count, and the hit range by galloping outwards from the first / last seed's hit
// (the window is +-H around it: a few thousand hits, so the probes stay close together)
__global__ void __launch_bounds__(256) ev_fix_kernel(const uint4* __restrict__ hits, SegCtx sc, int64_t H,
                                                     tt_event* __restrict__ events, const uint32_t* __restrict__ n_events_ptr,
                                                     uint32_t event_cap) {
    const uint32_t ne = min(*n_events_ptr, event_cap);
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < ne; e += gridDim.x * blockDim.x) {
        tt_event ev = events[e];
        ev.n_seeds -= ev.seed_begin;
        const uint32_t i0 = ev.hit_begin, i1 = ev.hit_end;  // hits of the first and of the last seed
        uint32_t sa = 0, sb = sc.n;
        if (sc.n_seg > 1) {
            const uint32_t s = find_segment(sc.off, sc.n_seg, i0);
            sa = __ldg(sc.off + s);
            sb = __ldg(sc.off + s + 1);
        }
        const int64_t tf = (int64_t)((uint64_t)ev.t_start + (uint64_t)H), tl = (int64_t)((uint64_t)ev.t_end - (uint64_t)H);
        if (ev.t_start <= tf) {  // first index of [sa, i0] with t >= t_start (t[i0] is one)
            uint32_t hi = i0, lo, step = 32;
            while (true) {
                lo = hi - sa > step ? hi - step : sa;
                if (lo == sa || hit_time(__ldg(hits + lo)) < ev.t_start) break;
                hi = lo;
                step <<= 1;
            }
            ev.hit_begin = lb_time(hits, lo, hi, ev.t_start);
        } else {
            ev.hit_begin = sa;  // wrapped below INT64_MIN: whole prefix
        }
        if (ev.t_end >= tl) {  // first index of (i1, sb) with t > t_end
            uint32_t lo = i1 + 1, hi, step = 32;
            while (true) {
                hi = sb - lo > step ? lo + step : sb;
                if (hi == sb || hit_time(__ldg(hits + (hi - 1))) > ev.t_end) break;
                lo = hi;
                step <<= 1;
            }
            ev.hit_end = ub_time(hits, lo, hi, ev.t_end);
        } else {
            ev.hit_end = sb;
        }
        events[e] = ev;
    }
}

// ---- gather offsets: exclusive scan of event lengths (count on the device) ------------------------
__global__ void __launch_bounds__(kEvThreads) len_count_kernel(const tt_event* __restrict__ events,
                                                               const uint32_t* __restrict__ n_events_ptr,
                                                               uint32_t event_cap, uint32_t* __restrict__ cnt) {
    const uint32_t ne = min(*n_events_ptr, event_cap);
    uint32_t c0, c1;
    ev_chunk(ne, c0, c1);
    uint32_t c = 0;
    for (uint32_t e = c0 + threadIdx.x; e < c1; e += kEvThreads) c += events[e].hit_end - events[e].hit_begin;
    __shared__ uint32_t sm[33];
    uint32_t total;
    block_exclusive_scan(c, sm, &total);
    if (threadIdx.x == 0) cnt[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) len_scan_kernel(uint32_t* __restrict__ cnt, uint32_t nb,
                                                        uint32_t* __restrict__ n_out) {
    __shared__ uint32_t sm[33];
    uint32_t carry = 0;
    for (uint32_t base = 0; base < nb; base += 1024) {
        const uint32_t i = base + threadIdx.x;
        const uint32_t v = i < nb ? cnt[i] : 0u;
        uint32_t total;
        const uint32_t ex = block_exclusive_scan(v, sm, &total);
        if (i < nb) cnt[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0 && n_out) *n_out = carry;
}

__global__ void __launch_bounds__(kEvThreads) len_write_kernel(const tt_event* __restrict__ events,
                                                               const uint32_t* __restrict__ n_events_ptr,
                                                               uint32_t event_cap, const uint32_t* __restrict__ off,
                                                               uint32_t* __restrict__ goff) {
    __shared__ uint32_t sm[33];
    const uint32_t ne = min(*n_events_ptr, event_cap);
    uint32_t c0, c1;
    ev_chunk(ne, c0, c1);
    uint32_t run = off[blockIdx.x];
    for (uint32_t base = c0; base < c1; base += kEvThreads) {
        const uint32_t e = base + threadIdx.x;
        const uint32_t v = e < c1 ? events[e].hit_end - events[e].hit_begin : 0u;
        uint32_t total;
        const uint32_t r = block_exclusive_scan(v, sm, &total);
        if (e < c1) goff[e] = run + r;
        run += total;
    }
}

// ---- tag + gather: 16 hits per thread; the events are ascending and disjoint in hit range ----------
constexpr int kTagThreads = 256;
constexpr int kTagPer = 16;

__global__ void __launch_bounds__(kTagThreads) tag_gather_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                                 const tt_event* __restrict__ events,
                                                                 const uint32_t* __restrict__ n_events_ptr,
                                                                 uint32_t event_cap, uint8_t* __restrict__ flags,
                                                                 uint4* __restrict__ gather,
                                                                 const uint32_t* __restrict__ goff) {
    const uint32_t ne = min(*n_events_ptr, event_cap);
    if (ne == 0) return;
    const uint64_t i0l = ((uint64_t)blockIdx.x * kTagThreads + threadIdx.x) * kTagPer;
    // first event with hit_end > i0: lane 0 of the warp searches for its index, the others walk on from there
    uint32_t a = 0;
    {
        const uint64_t w0l = i0l - (uint64_t)(threadIdx.x & 31u) * kTagPer;  // first hit of the warp
        if (w0l >= n) return;                                                // warp-uniform
        if ((threadIdx.x & 31u) == 0) {
            const uint32_t w0 = (uint32_t)w0l;
            uint32_t b = ne;
            while (a < b) {
                const uint32_t mid = a + ((b - a) >> 1);
                if (events[mid].hit_end <= w0) a = mid + 1; else b = mid;
            }
        }
        a = __shfl_sync(0xffffffffu, a, 0);
    }
    if (i0l >= n) return;
    const uint32_t i0 = (uint32_t)i0l;
    const uint32_t i1 = min(n, i0 + (uint32_t)kTagPer);
    while (a < ne && events[a].hit_end <= i0) ++a;
    uint32_t mask = 0;
    for (uint32_t e = a; e < ne; ++e) {
        const uint32_t hb = events[e].hit_begin, he = events[e].hit_end;
        if (hb >= i1) break;
        const uint32_t lo = max(hb, i0), hi = min(he, i1);
        if (hi > lo) mask |= (0xFFFFFFFFu >> (32u - (hi - lo))) << (lo - i0);  // bits [lo - i0, hi - i0), at most 16
        if (gather)
            for (uint32_t i = lo; i < hi; ++i) gather[goff[e] + (i - hb)] = __ldg(hits + i);
    }
    if (flags && mask) {
        if (i1 - i0 == kTagPer && (((uintptr_t)(flags + i0)) & 15) == 0) {
            uint4 v = *reinterpret_cast<uint4*>(flags + i0);
            uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int b8 = 0; b8 < 4; ++b8)
                    if (mask & (1u << (q * 4 + b8))) w[q] |= (uint32_t)TT_INEVT << (8 * b8);
            *reinterpret_cast<uint4*>(flags + i0) = make_uint4(w[0], w[1], w[2], w[3]);
        } else {
            for (uint32_t i = i0; i < i1; ++i)
                if (mask & (1u << (i - i0))) flags[i] |= (uint8_t)TT_INEVT;
        }
    }
}

struct EventsPlan {
    uint32_t *cnt, *cnt2, *goff, *n_gathered_dummy;
    uint8_t* head;  // [seed_cap] seed k opens an event
};
static void events_plan(Arena& a, uint32_t event_cap, uint32_t seed_cap, bool gather, EventsPlan& p) {
    p.cnt = a.take<uint32_t>(kEvBlocks);
    p.cnt2 = a.take<uint32_t>(kEvBlocks);
    p.n_gathered_dummy = a.take<uint32_t>(1);
    p.goff = a.take<uint32_t>(gather ? (size_t)event_cap : 1);
    p.head = a.take<uint8_t>((size_t)seed_cap + 1);
}

}  // namespace tt

using namespace tt;

extern "C" int tt_extract_events(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                                 const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* d_seeds,
                                 const uint32_t* d_n_seeds, uint32_t seed_cap, const tt_params* p,
                                 tt_event* d_events, uint32_t event_cap, uint32_t* d_n_events, uint8_t* d_flags,
                                 tt_hit* d_gather, uint32_t* d_n_gathered, void* d_ws, size_t* ws_bytes,
                                 int32_t* d_status, void* stream) {
    if (!ws_bytes || !p || n_seg < 1 || !h_seg_offsets) return TT_E_INVAL;
    if (p->event_half_ps < 0) return TT_E_INVAL;
    if (n >= 0xFFF00000u) return TT_E_INVAL;
    if (h_seg_offsets[0] != 0 || h_seg_offsets[n_seg] != n) return TT_E_INVAL;
    Arena sizing(nullptr);
    EventsPlan plan;
    events_plan(sizing, event_cap, seed_cap, true, plan);
    if (!d_ws) {
        *ws_bytes = sizing.off;
        return TT_OK;
    }
    if (*ws_bytes < sizing.off) return TT_E_WORKSPACE;
    if (!d_n_events || !d_status || !d_n_seeds || (!d_events && event_cap) || (!d_seeds && seed_cap) ||
        (n && (!d_sorted || !d_seg_offsets)))
        return TT_E_INVAL;
    if (((uintptr_t)d_ws & 255) || ((uintptr_t)d_sorted & 15) || ((uintptr_t)d_gather & 15)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    Arena a(d_ws);
    events_plan(a, event_cap, seed_cap, true, plan);
    if (n == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_n_events, 0, sizeof(uint32_t), s));
        if (d_n_gathered) TT_CUDA_OK(cudaMemsetAsync(d_n_gathered, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    const SegCtx sc{d_seg_offsets, n_seg, n};
    const uint64_t twoH = 2ull * (uint64_t)p->event_half_ps;
    const uint4* hits = (const uint4*)d_sorted;
    prof_mark(s, "ev.merge");
    TT_K(ev_count_kernel)<<<kEvBlocks, kEvThreads, 0, s>>>(hits, d_seeds, d_n_seeds, seed_cap, sc, twoH, plan.cnt, plan.head);
    TT_K(ev_scan_kernel)<<<1, 1024, 0, s>>>(plan.cnt, kEvBlocks, d_n_events, event_cap, d_status);
    TT_K(ev_write_kernel)<<<kEvBlocks, kEvThreads, 0, s>>>(hits, d_seeds, d_n_seeds, seed_cap, sc, twoH, p->event_half_ps,
                                                     plan.cnt, plan.head, d_events, event_cap);
    TT_K(ev_fix_kernel)<<<(uint32_t)sm_count(), 256, 0, s>>>(hits, sc, p->event_half_ps, d_events, d_n_events, event_cap);
    if (d_gather || d_n_gathered) {
        prof_mark(s, "ev.gather_scan");
        TT_K(len_count_kernel)<<<kEvBlocks, kEvThreads, 0, s>>>(d_events, d_n_events, event_cap, plan.cnt2);
        TT_K(len_scan_kernel)<<<1, 1024, 0, s>>>(plan.cnt2, kEvBlocks, d_n_gathered ? d_n_gathered : plan.n_gathered_dummy);
        if (d_gather)
            TT_K(len_write_kernel)<<<kEvBlocks, kEvThreads, 0, s>>>(d_events, d_n_events, event_cap, plan.cnt2, plan.goff);
    }
    if (d_flags || d_gather) {
        const uint32_t nb = div_up(n, kTagThreads * kTagPer);
        prof_mark(s, "ev.tag_gather");
        TT_K(tag_gather_kernel)<<<nb, kTagThreads, 0, s>>>(hits, n, d_events, d_n_events, event_cap, d_flags,
                                                     (uint4*)d_gather, plan.goff);
    }
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

// ---- the same call with its scratch in a static device array (tt.h: tt_extract_events_noalloc) -------------------
// In host code `g_noalloc_ws` is a host-side stand-in for the symbol, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, looked up once per device with that device current.
static __device__ __align__(256) unsigned char g_noalloc_ws[TT_NOALLOC_WS_BYTES];

static int noalloc_ws_address(void** out) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static void* addr[kMaxDev];  // zero-initialised
    int dev = -1;
    TT_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDev) return TT_E_CUDA;
    std::lock_guard<std::mutex> lk(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        TT_CUDA_OK(cudaGetSymbolAddress(&p, g_noalloc_ws));
        if (!p || ((uintptr_t)p & 255)) return TT_E_CUDA;
        addr[dev] = p;
    }
    *out = addr[dev];
    return TT_OK;
}

extern "C" int tt_extract_events_noalloc(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                                         const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* d_seeds,
                                         const uint32_t* d_n_seeds, uint32_t seed_cap, const tt_params* p,
                                         tt_event* d_events, uint32_t event_cap, uint32_t* d_n_events,
                                         uint8_t* d_flags, tt_hit* d_gather, uint32_t* d_n_gathered,
                                         int32_t* d_status, void* stream) {
    // argument errors first (the size query of the general call checks them), then the limit
    size_t need = 0;
    int rc = tt_extract_events(d_sorted, n, d_seg_offsets, h_seg_offsets, n_seg, d_seeds, d_n_seeds, seed_cap, p, d_events,
                               event_cap, d_n_events, d_flags, d_gather, d_n_gathered, nullptr, &need, d_status, stream);
    if (rc != TT_OK) return rc;
    if (need > (size_t)TT_NOALLOC_WS_BYTES) return TT_E_LIMIT;
    void* ws = nullptr;
    rc = noalloc_ws_address(&ws);
    if (rc != TT_OK) return rc;
    size_t have = TT_NOALLOC_WS_BYTES;
    return tt_extract_events(d_sorted, n, d_seg_offsets, h_seg_offsets, n_seg, d_seeds, d_n_seeds, seed_cap, p, d_events,
                             event_cap, d_n_events, d_flags, d_gather, d_n_gathered, ws, &have, d_status, stream);
}
