// tt_trigger.cu -- L1 (charge over threshold | same-floor coincidence), ordered L1 list, L2
// (time-space causality coincidence: star count + exact clique test), ordered seed list.
//
//   L1   PAPER.md:64 (QTRIG: hit[i].Charge > QTRIG; reading R3: >= q_thresh)
//        (coincidence between two hits in two PMTs of one floor; BASELINE.json configs[0]: 20 ns)
//   L2   PAPER.md:27-29 ("time-space correlation between PMT hits within a time interval less than
//        3 us"); north_star: ">= N L1 hits pairwise satisfying |dt| <= dt_max(pmt_i, pmt_j)"
//   seeds PAPER.md:67, 81 ("sends all trigger seeds")
#include "tt_common.cuh"

namespace tt {

// ------------------------------------------------------------------------------------------------
// L1: one thread per hit, neighbours read through L1/L2 cache (adjacent records).
// ------------------------------------------------------------------------------------------------
constexpr int kL1Threads = 256;

struct L1Rec {  // compact L1 hit, 16 bytes
    int64_t t;
    uint32_t idx;  // index in the sorted hit array
    uint32_t pmt;
};

__global__ void __launch_bounds__(kL1Threads) l1_flags_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                              const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                              uint64_t lc, uint32_t q_thresh,
                                                              uint8_t* __restrict__ flags,
                                                              uint32_t* __restrict__ blk_cnt) {
    const uint32_t i = blockIdx.x * kL1Threads + threadIdx.x;
    uint32_t f = 0;
    if (i < n) {
        const HitView h = unpack(__ldg(hits + i));
        uint32_t a = 0, b = n;
        if (n_seg > 1) {
            const uint32_t s = find_segment(seg_off, n_seg, i);
            a = __ldg(seg_off + s);
            b = __ldg(seg_off + s + 1);
        }
        if (h.charge >= q_thresh) f |= TT_Q;
        bool lcb = false;
        for (uint32_t j = i; j > a && !lcb;) {
            --j;
            const HitView o = unpack(__ldg(hits + j));
            if (udiff(h.t, o.t) > lc) break;
            lcb = (o.floor == h.floor) & (o.pmt != h.pmt);
        }
        for (uint32_t j = i + 1; j < b && !lcb; ++j) {
            const HitView o = unpack(__ldg(hits + j));
            if (udiff(o.t, h.t) > lc) break;
            lcb = (o.floor == h.floor) & (o.pmt != h.pmt);
        }
        if (lcb) f |= TT_LC;
        if (f) f |= TT_L1;
        flags[i] = (uint8_t)f;
    }
    const int c = __syncthreads_count(f != 0);
    if (threadIdx.x == 0) blk_cnt[blockIdx.x] = (uint32_t)c;
}

// ordered compaction of the L1 hits (block offsets from the scan of blk_cnt)
__global__ void __launch_bounds__(kL1Threads) l1_compact_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                                const uint8_t* __restrict__ flags,
                                                                const uint32_t* __restrict__ blk_off,
                                                                L1Rec* __restrict__ l1) {
    __shared__ uint32_t sm[33];
    const uint32_t i = blockIdx.x * kL1Threads + threadIdx.x;
    const bool is = i < n && (flags[i] & TT_L1);
    uint32_t total;
    const uint32_t r = block_exclusive_scan(is ? 1u : 0u, sm, &total);
    if (is) {
        const HitView h = unpack(__ldg(hits + i));
        L1Rec rec;
        rec.t = h.t;
        rec.idx = i;
        rec.pmt = h.pmt;
        l1[blk_off[blockIdx.x] + r] = rec;
    }
}

// ------------------------------------------------------------------------------------------------
// L2: one warp per L1 hit.
// ------------------------------------------------------------------------------------------------
constexpr int kL2Warps = 4;
constexpr int kMaxNb = TT_MAX_NEIGHBOURS;  // 256
constexpr int kMaxWords = kMaxNb / 32;     // 8

struct L2Smem {
    int64_t nb_t[kMaxNb];
    uint32_t nb_p[kMaxNb];
    uint32_t adj[kMaxNb * kMaxWords];
};

// dtmax lookup; -1 = never an edge.  a, b < n_pmt.
__device__ __forceinline__ int32_t dtmax_of(const tt_geometry_dev& g, uint32_t a, uint32_t b) {
    uint32_t ra = a, rb = b, blk = 0;
    if (g.n_tower > 1) {
        const uint32_t ta = a / g.ppt, tb = b / g.ppt;
        const int32_t bi = __ldg(g.pair_block + ta * g.n_tower + tb);
        if (bi < 0) return -1;
        blk = (uint32_t)bi;
        ra = a - ta * g.ppt;
        rb = b - tb * g.ppt;
    } else {
        const int32_t bi = __ldg(g.pair_block);
        if (bi < 0) return -1;
        blk = (uint32_t)bi;
    }
    return __ldg(g.blocks + ((size_t)blk * g.ppt + ra) * g.ppt + rb);
}

__device__ __forceinline__ bool edge_of(const tt_geometry_dev& g, uint64_t W, int64_t ta, uint32_t pa, int64_t tb,
                                        uint32_t pb) {
    if (pa >= g.n_pmt || pb >= g.n_pmt) return false;
    const int32_t lim = dtmax_of(g, pa, pb);
    if (lim < 0) return false;
    const uint64_t d = ta >= tb ? udiff(ta, tb) : udiff(tb, ta);
    const uint64_t l = (uint64_t)lim < W ? (uint64_t)lim : W;
    return d <= l;
}

// Is there a clique of `K` vertices in the graph (deg vertices, adjacency rows of `words` words)?
// Each lane starts from its own smallest vertex; iterative DFS on candidate bitmasks.
__device__ bool warp_has_clique(const uint32_t* adj, int deg, int words, int K, uint32_t lane) {
    bool found = false;
    if (K <= 0) found = true;
    uint32_t cand[TT_MAX_MULTIPLICITY][kMaxWords];
    for (int u = (int)lane; u < deg && !found; u += 32) {
        if (K == 1) { found = true; break; }
        const int need = K - 1;  // vertices still to choose after u
        // cand[0] = adj[u] restricted to vertices > u
        int cnt = 0;
        for (int w = 0; w < words; ++w) {
            uint32_t m = adj[u * words + w];
            if (w < (u >> 5)) m = 0;
            else if (w == (u >> 5)) m &= ~((2u << (u & 31)) - 1u);
            cand[0][w] = m;
            cnt += __popc(m);
        }
        (void)cnt;
        int d = 0;
        while (true) {
            const int rem = need - d;
            if (rem == 0) { found = true; break; }
            int pc = 0;
            for (int w = 0; w < words; ++w) pc += __popc(cand[d][w]);
            if (pc < rem) {
                if (d == 0) break;
                --d;
                continue;
            }
            // pick the lowest candidate v, remove it, descend with cand & adj[v]
            int v = -1;
            for (int w = 0; w < words; ++w) {
                if (cand[d][w]) {
                    const int bit = __ffs(cand[d][w]) - 1;
                    cand[d][w] &= cand[d][w] - 1u;
                    v = w * 32 + bit;
                    break;
                }
            }
            for (int w = 0; w < words; ++w) cand[d + 1][w] = cand[d][w] & adj[v * words + w];
            ++d;
        }
    }
    return __any_sync(0xffffffffu, found);
}

__global__ void __launch_bounds__(kL2Warps * 32) l2_kernel(const L1Rec* __restrict__ l1,
                                                           const uint32_t* __restrict__ m_ptr,
                                                           const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                           uint32_t n, tt_geometry_dev g, uint64_t W, uint32_t N,
                                                           uint32_t mode, uint8_t* __restrict__ flags,
                                                           uint8_t* __restrict__ l2bit, int32_t* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    L2Smem& sm = reinterpret_cast<L2Smem*>(smem_raw)[warp];
    const uint32_t m = *m_ptr;
    const uint32_t nwarps = gridDim.x * kL2Warps;
    // effective scan window: no edge can be longer than the largest table entry
    const bool any_edge = g.max_dt >= 0;
    const uint64_t Weff = any_edge ? ((uint64_t)g.max_dt < W ? (uint64_t)g.max_dt : W) : 0;
    for (uint32_t x = blockIdx.x * kL2Warps + warp; x < m; x += nwarps) {
        const L1Rec rx = l1[x];
        uint32_t sa = 0, sb = n;
        if (n_seg > 1) {
            const uint32_t s = find_segment(seg_off, n_seg, rx.idx);
            sa = __ldg(seg_off + s);
            sb = __ldg(seg_off + s + 1);
        }
        const bool bad = rx.pmt >= g.n_pmt;
        if (bad && lane == 0) atomicOr(status, TT_S_BAD_PMT);
        uint32_t deg = 0;
        if (!bad && any_edge) {
            // backward
            for (uint32_t base = x; base > 0;) {
                const bool valid = base > lane;  // y = base-1-lane >= 0
                const uint32_t y = valid ? base - 1 - lane : 0;
                bool in = false, e = false;
                L1Rec ry;
                if (valid) {
                    ry = l1[y];
                    in = ry.idx >= sa && udiff(rx.t, ry.t) <= Weff;
                    if (in) e = edge_of(g, W, rx.t, rx.pmt, ry.t, ry.pmt);
                }
                const uint32_t eb = __ballot_sync(0xffffffffu, e);
                const uint32_t ib = __ballot_sync(0xffffffffu, in);
                if (e) {
                    const uint32_t pos = deg + __popc(eb & lanemask_lt());
                    if (pos < (uint32_t)kMaxNb) { sm.nb_t[pos] = ry.t; sm.nb_p[pos] = ry.pmt; }
                }
                deg += __popc(eb);
                if (ib != 0xffffffffu) break;
                base -= 32;  // ib full => base > 31
            }
            // forward
            for (uint32_t base = x + 1; base < m; base += 32) {
                const uint32_t y = base + lane;
                const bool valid = y < m;
                bool in = false, e = false;
                L1Rec ry;
                if (valid) {
                    ry = l1[y];
                    in = ry.idx < sb && udiff(ry.t, rx.t) <= Weff;
                    if (in) e = edge_of(g, W, rx.t, rx.pmt, ry.t, ry.pmt);
                }
                const uint32_t eb = __ballot_sync(0xffffffffu, e);
                const uint32_t ib = __ballot_sync(0xffffffffu, in);
                if (e) {
                    const uint32_t pos = deg + __popc(eb & lanemask_lt());
                    if (pos < (uint32_t)kMaxNb) { sm.nb_t[pos] = ry.t; sm.nb_p[pos] = ry.pmt; }
                }
                deg += __popc(eb);
                if (ib != 0xffffffffu) break;
            }
        }
        const bool star = deg + 1 >= N;
        bool l2 = star;
        if (star && mode == 0 && N > 2) {
            if (deg > (uint32_t)kMaxNb) {
                l2 = false;
                if (lane == 0) atomicOr(status, TT_S_DENSITY);
            } else {
                __syncwarp();
                const int words = (int)((deg + 31) >> 5);
                for (uint32_t u = 0; u < deg; ++u) {
                    const int64_t tu = sm.nb_t[u];
                    const uint32_t pu = sm.nb_p[u];
                    for (int w = 0; w < words; ++w) {
                        const uint32_t v = w * 32 + lane;
                        const bool e = v < deg && v != u && edge_of(g, W, tu, pu, sm.nb_t[v], sm.nb_p[v]);
                        const uint32_t eb = __ballot_sync(0xffffffffu, e);
                        if (lane == 0) sm.adj[u * words + w] = eb;
                    }
                }
                __syncwarp();
                l2 = warp_has_clique(sm.adj, (int)deg, words, (int)N - 1, lane);
                __syncwarp();
            }
        }
        if (lane == 0) {
            uint32_t f = 0;
            if (star) f |= TT_L2STAR;
            if (l2) f |= TT_L2;
            if (f) flags[rx.idx] |= (uint8_t)f;
            l2bit[x] = l2 ? 1 : 0;
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------
// Ordered seed compaction over the L1 list (length known on the device only): fixed grid, each
// block owns one contiguous chunk; count -> one-block scan -> ordered write.
// ------------------------------------------------------------------------------------------------
constexpr int kSeedBlocks = 592;  // 4 x 148
constexpr int kSeedThreads = 256;

__device__ __forceinline__ void chunk_bounds(uint32_t m, uint32_t& c0, uint32_t& c1) {
    const uint32_t per = (m + gridDim.x - 1) / gridDim.x;
    const uint64_t a = (uint64_t)blockIdx.x * per;
    c0 = a < m ? (uint32_t)a : m;
    c1 = a + per < m ? (uint32_t)(a + per) : m;
}

__global__ void __launch_bounds__(kSeedThreads) seed_count_kernel(const uint8_t* __restrict__ l2bit,
                                                                  const uint32_t* __restrict__ m_ptr,
                                                                  uint32_t* __restrict__ cnt) {
    uint32_t c0, c1;
    chunk_bounds(*m_ptr, c0, c1);
    uint32_t c = 0;
    for (uint32_t x = c0 + threadIdx.x; x < c1; x += kSeedThreads) c += l2bit[x];
    __shared__ uint32_t sm[33];
    uint32_t total;
    block_exclusive_scan(c, sm, &total);
    if (threadIdx.x == 0) cnt[blockIdx.x] = total;
}

// one block: exclusive scan of cnt[nb] in place, true total to *n_out, overflow bit to status
__global__ void __launch_bounds__(1024) count_scan_kernel(uint32_t* __restrict__ cnt, uint32_t nb,
                                                          uint32_t* __restrict__ n_out, uint32_t cap, int32_t bit,
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
        if (carry > cap) atomicOr(status, bit);
    }
}

__global__ void __launch_bounds__(kSeedThreads) seed_write_kernel(const uint8_t* __restrict__ l2bit,
                                                                  const L1Rec* __restrict__ l1,
                                                                  const uint32_t* __restrict__ m_ptr,
                                                                  const uint32_t* __restrict__ off,
                                                                  uint32_t* __restrict__ seeds, uint32_t cap) {
    __shared__ uint32_t sm[33];
    uint32_t c0, c1;
    chunk_bounds(*m_ptr, c0, c1);
    uint32_t run = off[blockIdx.x];
    for (uint32_t base = c0; base < c1; base += kSeedThreads) {
        const uint32_t x = base + threadIdx.x;
        const bool is = x < c1 && l2bit[x];
        uint32_t total;
        const uint32_t r = block_exclusive_scan(is ? 1u : 0u, sm, &total);
        if (is && run + r < cap) seeds[run + r] = l1[x].idx;
        run += total;
    }
}

// ------------------------------------------------------------------------------------------------
struct TriggerPlan {
    uint32_t *blk_cnt, *scan_scratch, *m_total, *seed_cnt;
    L1Rec* l1;
    uint8_t* l2bit;
    uint32_t nblk;
};

static void trigger_plan(Arena& a, uint32_t n, TriggerPlan& p) {
    p.nblk = div_up(n, kL1Threads);
    p.blk_cnt = a.take<uint32_t>(p.nblk + 1);
    p.scan_scratch = a.take<uint32_t>(scan_ws_count(p.nblk + 1));
    p.m_total = a.take<uint32_t>(1);
    p.seed_cnt = a.take<uint32_t>(kSeedBlocks);
    p.l1 = a.take<L1Rec>(n);
    p.l2bit = a.take<uint8_t>(n);
}

}  // namespace tt

using namespace tt;

extern "C" int tt_trigger_slice(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                                const uint32_t* h_seg_offsets, uint32_t n_seg, const tt_geometry* g,
                                const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds, uint32_t seed_cap,
                                uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes, int32_t* d_status, void* stream) {
    if (!ws_bytes || !p || !g || n_seg < 1 || !h_seg_offsets) return TT_E_INVAL;
    if (p->l2_multiplicity < 1 || p->l2_multiplicity > TT_MAX_MULTIPLICITY || p->l2_mode > 1 || p->reserved != 0 ||
        p->lc_window_ps < 0 || p->l2_window_ps < 0 || p->event_half_ps < 0)
        return TT_E_INVAL;
    if (n >= 0xFFF00000u) return TT_E_INVAL;
    if (h_seg_offsets[0] != 0 || h_seg_offsets[n_seg] != n) return TT_E_INVAL;
    for (uint32_t s = 0; s < n_seg; ++s)
        if (h_seg_offsets[s] > h_seg_offsets[s + 1]) return TT_E_INVAL;
    Arena sizing(nullptr);
    TriggerPlan plan;
    trigger_plan(sizing, n, plan);
    if (!d_ws) {
        *ws_bytes = sizing.off;
        return TT_OK;
    }
    if (*ws_bytes < sizing.off) return TT_E_WORKSPACE;
    if (!d_flags || !d_n_seeds || !d_status || (!d_seeds && seed_cap) || (n && (!d_sorted || !d_seg_offsets)))
        return TT_E_INVAL;
    if (((uintptr_t)d_ws & 255) || ((uintptr_t)d_sorted & 15)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (n == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_n_seeds, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    Arena a(d_ws);
    trigger_plan(a, n, plan);
    static bool attr_done = false;
    if (!attr_done) {
        TT_CUDA_OK(cudaFuncSetAttribute(l2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)(sizeof(L2Smem) * kL2Warps)));
        attr_done = true;
    }
    prof_mark(s, "trig.l1_flags");
    TT_K(l1_flags_kernel)<<<plan.nblk, kL1Threads, 0, s>>>((const uint4*)d_sorted, n, d_seg_offsets, n_seg,
                                                     (uint64_t)p->lc_window_ps, p->q_thresh, d_flags, plan.blk_cnt);
    prof_mark(s, "trig.l1_scan");
    int rc = exclusive_scan_u32(plan.blk_cnt, plan.blk_cnt, plan.nblk, plan.scan_scratch, plan.m_total, s);
    if (rc != TT_OK) return rc;
    prof_mark(s, "trig.l1_compact");
    TT_K(l1_compact_kernel)<<<plan.nblk, kL1Threads, 0, s>>>((const uint4*)d_sorted, n, d_flags, plan.blk_cnt, plan.l1);
    prof_mark(s, "trig.l2");
    TT_K(l2_kernel)<<<kSMs * 8, kL2Warps * 32, sizeof(L2Smem) * kL2Warps, s>>>(
        plan.l1, plan.m_total, d_seg_offsets, n_seg, n, g->dev, (uint64_t)p->l2_window_ps, p->l2_multiplicity,
        p->l2_mode, d_flags, plan.l2bit, d_status);
    prof_mark(s, "trig.seeds");
    TT_K(seed_count_kernel)<<<kSeedBlocks, kSeedThreads, 0, s>>>(plan.l2bit, plan.m_total, plan.seed_cnt);
    TT_K(count_scan_kernel)<<<1, 1024, 0, s>>>(plan.seed_cnt, kSeedBlocks, d_n_seeds, seed_cap, TT_S_SEED_OVERFLOW, d_status);
    TT_K(seed_write_kernel)<<<kSeedBlocks, kSeedThreads, 0, s>>>(plan.l2bit, plan.l1, plan.m_total, plan.seed_cnt, d_seeds,
                                                           seed_cap);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}
