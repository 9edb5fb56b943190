// tt_trigger.cu -- L1 (charge over threshold | same-floor coincidence), ordered L1 list, L2
// (time-space causality coincidence: star count + exact clique test), ordered seed list.
//
//   L1   PAPER.md:64 (QTRIG: hit[i].Charge > QTRIG; reading R3: >= q_thresh)
//        (coincidence between two hits in two PMTs of one floor; BASELINE.json configs[0]: 20 ns)
//   L2   PAPER.md:27-29 ("time-space correlation between PMT hits within a time interval less than
//        3 us"); north_star: ">= N L1 hits pairwise satisfying |dt| <= dt_max(pmt_i, pmt_j)"
//   seeds PAPER.md:67, 81 ("sends all trigger seeds")
#include "tt_merge.cuh"

namespace tt {

// ------------------------------------------------------------------------------------------------
// L1.  One CTA per tile of kL1Tile consecutive sorted hits, staged in shared memory (with a halo of
// kL1Halo hits on both sides) as (32-bit time relative to the first staged hit, floor << 16 | pmt).
// Every staged hit scans FORWARD while t_j - t_i <= LC and marks both partners of a same-floor /
// other-PMT pair, so each pair is tested once.  What the staged window cannot decide (a neighbourhood
// reaching past the halo, a tile spanning >= 2^32 ps, a segment boundary) is finished by exact scans
// of global memory, so the result is the plain definition for any input.
// ------------------------------------------------------------------------------------------------
constexpr int kL1Threads = 256;
constexpr int kL1Per = 16;                        // in-tile hits per thread
constexpr int kL1Tile = kL1Threads * kL1Per;      // 4096
constexpr int kL1Halo = kL1Threads;               // staged hits before and after the tile
constexpr int kL1Stage = kL1Tile + 2 * kL1Halo;   // 4608

struct L1Rec {  // compact L1 hit, 16 bytes
    int64_t t;
    uint32_t idx;  // index in the sorted hit array
    uint32_t tp;   // tower << 16 | pmt index inside the tower; 0xFFFFFFFF = pmt_id out of range
};
constexpr uint32_t kBadTp = 0xFFFFFFFFu;

// exact LC bit of hit i by scanning global memory outwards from (below, above): partners j < below and
// j >= above inside [a, b)
__device__ __forceinline__ bool lc_scan_global(const uint4* __restrict__ hits, int64_t t, uint32_t fp, uint32_t below,
                                               uint32_t above, uint32_t a, uint32_t b, uint64_t lc) {
    for (uint32_t j = below; j > a;) {
        --j;
        const uint4 v = __ldg(hits + j);
        if (udiff(t, hit_time(v)) > lc) break;
        const uint32_t x = v.z ^ fp;
        if (x - 1u < 0xFFFFu) return true;  // same floor (high half equal), other pmt (low half differs)
    }
    for (uint32_t j = above; j < b; ++j) {
        const uint4 v = __ldg(hits + j);
        if (udiff(hit_time(v), t) > lc) break;
        const uint32_t x = v.z ^ fp;
        if (x - 1u < 0xFFFFu) return true;
    }
    return false;
}

constexpr int kL1Pad = 64;  // readable slack behind the staged arrays (speculative key reads)

struct L1Smem {
    uint32_t f[kL1Tile / 4];
    uint32_t t[kL1Stage + kL1Pad];
    uint32_t k[kL1Stage + kL1Pad];
    uint32_t red[kL1Threads / 32];
};

__global__ void __launch_bounds__(kL1Threads) l1_tile_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                             const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                             uint64_t lc, uint32_t q_thresh,
                                                             uint8_t* __restrict__ flags,
                                                             uint32_t* __restrict__ tile_cnt) {
    extern __shared__ __align__(16) unsigned char l1_smem_raw[];
    L1Smem& l1s = *reinterpret_cast<L1Smem*>(l1_smem_raw);
    uint32_t* const s_t = l1s.t;     // time relative to the first staged hit
    uint32_t* const s_k = l1s.k;     // floor << 16 | pmt
    uint32_t* const s_f = l1s.f;     // flag bytes of the in-tile hits
    uint32_t* const s_red = l1s.red;
    const uint32_t tid = threadIdx.x, lane = tid & 31;
    const uint32_t tb = blockIdx.x * (uint32_t)kL1Tile;                 // first in-tile hit
    const uint32_t te = min(n, tb + (uint32_t)kL1Tile);                 // end of the tile
    const uint32_t glo = tb >= (uint32_t)kL1Halo ? tb - kL1Halo : 0u;   // first staged hit
    const uint32_t ghi = min(n, te + (uint32_t)kL1Halo);                // end of the staged hits
    // staged slot e <-> global index g0 + e (g0 = tb - kL1Halo, modulo 2^32); slot kL1Halo = first in-tile hit
    const uint32_t g0 = tb - (uint32_t)kL1Halo;
    const uint32_t e_lo = glo - g0, e_hi = ghi - g0, e_te = te - g0;
    uint32_t seg_a = 0, seg_b = n;
    bool one_seg = true;
    if (n_seg > 1) {
        const uint32_t s = find_segment(seg_off, n_seg, glo);
        seg_a = __ldg(seg_off + s);
        seg_b = __ldg(seg_off + s + 1);
        one_seg = seg_b >= ghi;
    }
    const int64_t t0 = hit_time(__ldg(hits + glo));
    bool wide = false;  // some staged time is not t0 + (a 32-bit offset): sparse data, or an earlier time of another segment
    uint8_t* s_fb = reinterpret_cast<uint8_t*>(s_f);
    // batches of six unconditional loads (slots outside the staged range read the first staged hit and are
    // discarded): all six are in flight before the first is used
    constexpr int kBatch = 6;
    static_assert((kL1Per + 2) % kBatch == 0, "staging batches");
#pragma unroll
    for (int k0 = 0; k0 < kL1Per + 2; k0 += kBatch) {
        uint4 v[kBatch];
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const uint32_t e = tid + (k0 + u) * kL1Threads;
            const bool in = e >= e_lo && e < e_hi;
            v[u] = __ldg(hits + (in ? g0 + e : glo));
        }
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int k = k0 + u;
            const uint32_t e = tid + k * kL1Threads;
            uint32_t tr = 0xFFFFFFFFu, ky = 0xFFFFFFFFu, q = 0;
            if (e >= e_lo && e < e_hi) {
                const uint64_t d64 = udiff(hit_time(v[u]), t0);
                wide |= d64 >= 0xFFFFFFFFull;
                tr = (uint32_t)d64;
                ky = v[u].z;
                q = (v[u].w & 0xFFFFu) >= q_thresh ? (uint32_t)TT_Q : 0u;
            }
            s_t[e] = tr;
            s_k[e] = ky;
            if (k >= 1 && k <= kL1Per) s_fb[e - kL1Halo] = (uint8_t)q;
        }
    }
    if (tid < kL1Pad) { s_t[kL1Stage + tid] = 0xFFFFFFFFu; s_k[kL1Stage + tid] = 0xFFFFFFFFu; }
    const bool fits32 = !__syncthreads_or(wide);
    const uint32_t lc32 = lc > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)lc;
    if (fits32) {
        const uint32_t t_last = s_t[e_hi - 1];
        // chunk k = 0: the halo before the tile (marks its in-tile partners only); k = 1..16: the tile
#pragma unroll 1
        for (int k = 0; k <= kL1Per; ++k) {
            const uint32_t e = tid + k * kL1Threads;
            const uint32_t w0 = e - lane;                       // first slot of this warp's chunk
            if (w0 >= e_te) break;                              // warp-uniform
            const bool valid = e >= e_lo && e < e_te;
            const uint32_t ti = s_t[e], ki = s_k[e];
            uint32_t jmax = e_hi, sa = seg_a, sb = seg_b;
            if (!one_seg && valid) {
                const uint32_t s = find_segment(seg_off, n_seg, g0 + e);
                sa = __ldg(seg_off + s);
                sb = __ldg(seg_off + s + 1);
                if (sb < ghi) jmax = sb - g0;
            }
            bool found = false;
            const uint32_t dmax = e_hi - w0;                    // warp-uniform bound on the offsets
            for (uint32_t d0 = 1; d0 < dmax; d0 += 4) {
                // does any hit of the chunk still have offset d0 inside its window?
                if (!__any_sync(0xffffffffu, valid && (s_t[e + d0] - ti <= lc32))) break;
                // four offsets at once: a hit of the same floor is rare (cfg4: 18 neighbours, 1400 floors)
                const uint32_t x0 = s_k[e + d0] ^ ki, x1 = s_k[e + d0 + 1] ^ ki, x2 = s_k[e + d0 + 2] ^ ki, x3 = s_k[e + d0 + 3] ^ ki;
                if ((x0 - 1u < 0xFFFFu) | (x1 - 1u < 0xFFFFu) | (x2 - 1u < 0xFFFFu) | (x3 - 1u < 0xFFFFu)) {  // same floor, other PMT
                    // the time tests, straight-line, before anything diverges: with few floors (one tower: 14) the
                    // floor filter fires in almost every warp step, a real pair (floor AND window) stays rare
                    const uint32_t j0 = e + d0;
                    const bool m0 = (x0 - 1u < 0xFFFFu) && (s_t[j0] - ti <= lc32);
                    const bool m1 = (x1 - 1u < 0xFFFFu) && (s_t[j0 + 1] - ti <= lc32);
                    const bool m2 = (x2 - 1u < 0xFFFFu) && (s_t[j0 + 2] - ti <= lc32);
                    const bool m3 = (x3 - 1u < 0xFFFFu) && (s_t[j0 + 3] - ti <= lc32);
                    if (valid && (m0 | m1 | m2 | m3)) {
                        const uint32_t mm = (m0 ? 1u : 0u) | (m1 ? 2u : 0u) | (m2 ? 4u : 0u) | (m3 ? 8u : 0u);
#pragma unroll
                        for (uint32_t q = 0; q < 4; ++q) {
                            const uint32_t j = j0 + q;
                            if (((mm >> q) & 1u) && j < jmax) {
                                found = true;
                                if (j >= (uint32_t)kL1Halo && j < e_te)
                                    atomicOr(&s_f[(j - kL1Halo) >> 2], (uint32_t)TT_LC << (8 * ((j - kL1Halo) & 3)));
                            }
                        }
                    }
                }
            }
            if (k == 0 || !valid) continue;
            // what the staged window leaves open: partners beyond its end / before its start
            const bool open_fwd = jmax == e_hi && ghi < sb && t_last - ti <= lc32;
            const bool open_bwd = max(glo, sa) > sa && (uint64_t)ti <= lc;  // the first staged hit is inside the window
            if (!found && (open_fwd || open_bwd)) {
                const int64_t t = (int64_t)((uint64_t)t0 + ti);
                found = lc_scan_global(hits, t, ki, open_bwd ? glo : sa, open_fwd ? ghi : sb, sa, sb, lc);
            }
            if (found) atomicOr(&s_f[(e - kL1Halo) >> 2], (uint32_t)TT_LC << (8 * ((e - kL1Halo) & 3)));
        }
    } else {
        // ---- sparse tile (>= 2^32 ps across the staged hits): exact scans of global memory ------------
#pragma unroll 1
        for (int k = 1; k <= kL1Per; ++k) {
            const uint32_t e = tid + k * kL1Threads;
            if (e >= e_te) break;
            const uint32_t g = g0 + e;
            uint32_t sa = seg_a, sb = seg_b;
            if (!one_seg) {
                const uint32_t s = find_segment(seg_off, n_seg, g);
                sa = __ldg(seg_off + s);
                sb = __ldg(seg_off + s + 1);
            }
            const uint4 v = __ldg(hits + g);
            if (lc_scan_global(hits, hit_time(v), v.z, g, g + 1, sa, sb, lc))
                atomicOr(&s_f[(e - kL1Halo) >> 2], (uint32_t)TT_LC << (8 * ((e - kL1Halo) & 3)));
        }
    }
    __syncthreads();
    // thread t writes the 16 flag bytes [16 t, 16 t + 16) of the tile: L1 = Q | LC
    uint32_t cnt = 0;
    {
        uint4 v = reinterpret_cast<const uint4*>(s_f)[tid];
        uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint32_t any = (w[q] | (w[q] >> 1)) & 0x01010101u;  // Q = 1, LC = 2
            w[q] |= any << 2;                                          // L1 = 4
            cnt += __popc(any);
        }
        const uint32_t i0 = tb + tid * 16u;
        if (i0 + 16u <= te && (((uintptr_t)(flags + i0)) & 15) == 0) {
            *reinterpret_cast<uint4*>(flags + i0) = make_uint4(w[0], w[1], w[2], w[3]);
        } else {
            cnt = 0;
            for (uint32_t b8 = 0; b8 < 16u && i0 + b8 < te; ++b8) {
                const uint32_t f = (w[b8 >> 2] >> (8 * (b8 & 3))) & 0xFFu;
                flags[i0 + b8] = (uint8_t)f;
                cnt += f ? 1u : 0u;
            }
        }
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0) s_red[tid >> 5] = cnt;
    __syncthreads();
    if (tid == 0) {
        uint32_t c = 0;
#pragma unroll
        for (int w = 0; w < kL1Threads / 32; ++w) c += s_red[w];
        tile_cnt[blockIdx.x] = c;
    }
}

// ---- fused path (tt_sort_trigger_slice): the last merge level wrote Q / LC / L1 for every hit from what its own
// time tile holds (merge_fast_kernel<.., true>).  A partner in a neighbouring tile was not visible there, so the
// hits within LC of the last hit before their tile or of the first hit after it -- and every hit of a tile the general
// merge kernel sorted (tile_open) -- get their flag byte from an exact scan of the sorted array here.  One warp per
// tile.  At the last level a group is a whole segment, so [gs, ge) bounds the scans.
constexpr int kBndWarps = 8;

__device__ __forceinline__ void l1_exact(const uint4* __restrict__ hits, uint32_t i, uint32_t gs, uint32_t ge, uint64_t lc,
                                         uint32_t q_thresh, uint8_t* __restrict__ flags) {
    const uint4 v = __ldg(hits + i);
    uint32_t f = (v.w & 0xFFFFu) >= q_thresh ? (uint32_t)TT_Q : 0u;
    if (lc_scan_global(hits, hit_time(v), v.z, i, i + 1, gs, ge, lc)) f |= TT_LC;
    if (f) f |= TT_L1;
    flags[i] = (uint8_t)f;
}

__global__ void __launch_bounds__(kBndWarps * 32) l1_boundary_kernel(LevelDev lv, uint32_t n_tiles,
                                                                     const uint4* __restrict__ hits, uint64_t lc,
                                                                     uint32_t q_thresh, uint8_t* __restrict__ flags) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t tile = blockIdx.x * kBndWarps + (threadIdx.x >> 5);
    if (tile >= n_tiles) return;
    const uint4 td = lv.tile_desc[tile];
    const uint2 td2 = lv.tile_desc2[tile];
    const uint32_t gs = lv.roff[td.y], ge = lv.roff[td.y + td.z];
    const uint32_t tb0 = lv.tile_base[td2.y], tb1 = lv.tile_base[td2.y + 1];
    uint32_t b0 = gs + tb0, b1 = gs + tb1;  // the tile's range of the sorted array
    if (b0 > ge) b0 = ge;                    // only with unsorted runs (output unspecified, accesses stay in range)
    if (b1 > ge) b1 = ge;
    if (b1 <= b0) return;
    if (lv.tile_open[tile]) {
        for (uint32_t i = b0 + lane; i < b1; i += 32) l1_exact(hits, i, gs, ge, lc, q_thresh, flags);
        return;
    }
    const bool has_prev = b0 > gs, has_next = b1 < ge;
    const int64_t t_prev = has_prev ? hit_time(__ldg(hits + b0 - 1)) : 0;
    const int64_t t_next = has_next ? hit_time(__ldg(hits + b1)) : 0;
    if (has_prev) {  // head: hits within LC of the last hit before the tile
        for (uint32_t base = b0; base < b1; base += 32) {
            const uint32_t i = base + lane;
            const bool open = i < b1 && udiff(hit_time(__ldg(hits + i)), t_prev) <= lc;
            if (open) l1_exact(hits, i, gs, ge, lc, q_thresh, flags);
            if (!__all_sync(0xffffffffu, open)) break;
        }
    }
    if (has_next) {  // tail: hits within LC of the first hit after the tile (not those the head loop already did)
        for (uint32_t base = b1; base > b0;) {
            const bool valid = base - b0 > lane;
            const uint32_t i = base - 1u - lane;
            bool open = false;
            if (valid) {
                const int64_t t = hit_time(__ldg(hits + i));
                open = udiff(t_next, t) <= lc;
                if (open && !(has_prev && udiff(t, t_prev) <= lc)) l1_exact(hits, i, gs, ge, lc, q_thresh, flags);
            }
            if (!__all_sync(0xffffffffu, open)) break;
            base -= 32;
        }
    }
}

// L1 hits per block of kL1Tile flag bytes (the fused path has no l1_tile_kernel to count them)
__global__ void __launch_bounds__(kL1Threads) l1_count_kernel(const uint8_t* __restrict__ flags, uint32_t n,
                                                              uint32_t* __restrict__ tile_cnt) {
    __shared__ uint32_t s_red[kL1Threads / 32];
    const uint32_t i0 = blockIdx.x * (uint32_t)kL1Tile + threadIdx.x * kL1Per;
    uint32_t cnt = 0;
    if (i0 < n) {
        if (i0 + kL1Per <= n && (((uintptr_t)(flags + i0)) & 15) == 0) {
            const uint4 v = *reinterpret_cast<const uint4*>(flags + i0);
            cnt = __popc(v.x & 0x04040404u) + __popc(v.y & 0x04040404u) + __popc(v.z & 0x04040404u) + __popc(v.w & 0x04040404u);
        } else {
            for (uint32_t k = 0; k < (uint32_t)kL1Per && i0 + k < n; ++k) cnt += (flags[i0 + k] & TT_L1) ? 1u : 0u;
        }
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t c = 0;
#pragma unroll
        for (int w = 0; w < kL1Threads / 32; ++w) c += s_red[w];
        tile_cnt[blockIdx.x] = c;
    }
}

// ordered compaction of the L1 hits, one CTA per L1 tile (tile offsets from the scan of tile_cnt):
// thread t owns the 16 consecutive flag bytes [16 t, 16 t + 16) of the tile.
__global__ void __launch_bounds__(kL1Threads) l1_compact_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                                const uint8_t* __restrict__ flags,
                                                                const uint32_t* __restrict__ tile_off,
                                                                L1Rec* __restrict__ l1, uint32_t cap,
                                                                uint32_t* __restrict__ m_total, uint32_t n_pmt,
                                                                uint32_t ppt, int32_t* __restrict__ status) {
    __shared__ uint32_t sm[33];
    // the list holds cap records (tt_params.l1_capacity): later L1 hits keep their flags but are not listed.  No block of
    // this kernel reads *m_total; the L2 kernels that follow see the clamped count.
    if (blockIdx.x == 0 && threadIdx.x == 0 && *m_total > cap) {
        *m_total = cap;
        atomicOr(status, TT_S_L1_OVERFLOW);
    }
    const uint32_t i0 = blockIdx.x * (uint32_t)kL1Tile + threadIdx.x * kL1Per;
    uint32_t mask = 0;
    if (i0 < n) {
        if (i0 + kL1Per <= n && (((uintptr_t)(flags + i0)) & 15) == 0) {
            const uint4 v = *reinterpret_cast<const uint4*>(flags + i0);
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int b8 = 0; b8 < 4; ++b8)
                    if ((w[q] >> (8 * b8)) & TT_L1) mask |= 1u << (q * 4 + b8);
        } else {
            for (uint32_t k = 0; k < (uint32_t)kL1Per && i0 + k < n; ++k)
                if (flags[i0 + k] & TT_L1) mask |= 1u << k;
        }
    }
    // the block's L1 hits as a dense list of tile positions in shared memory (a tile holds ~2 % L1 hits: most threads
    // have none, a few have one), then one thread per list entry: the record gathers are all in flight at once and
    // the 16-byte list records leave coalesced
    __shared__ uint16_t s_pos[kL1Tile];
    uint32_t total;
    uint32_t r = block_exclusive_scan(__popc(mask), sm, &total);
    while (mask) {
        const uint32_t k = __ffs(mask) - 1;
        mask &= mask - 1;
        s_pos[r++] = (uint16_t)(threadIdx.x * kL1Per + k);
    }
    __syncthreads();
    const uint32_t base = tile_off[blockIdx.x], tb = blockIdx.x * (uint32_t)kL1Tile;
    bool bad = false;
    for (uint32_t q = threadIdx.x; q < total; q += kL1Threads) {
        const uint32_t i = tb + s_pos[q];
        const HitView h = unpack(__ldg(hits + i));
        L1Rec rec;
        rec.t = h.t;
        rec.idx = i;
        if (h.pmt >= n_pmt) { rec.tp = kBadTp; bad = true; }
        else { const uint32_t tw = h.pmt / ppt; rec.tp = (tw << 16) | (h.pmt - tw * ppt); }
        if (base + q < cap) l1[base + q] = rec;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(status, TT_S_BAD_PMT);
}

// ------------------------------------------------------------------------------------------------
// L2.  Causality edge between two L1 hits; tp = tower << 16 | local pmt.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool edge_tp(const tt_geometry_dev& g, uint64_t W, uint64_t dt, uint32_t tpa, uint32_t tpb) {
    if (tpa == kBadTp || tpb == kBadTp) return false;
    uint32_t blk = 0;
    if (g.n_tower > 1) {
        const int32_t bi = __ldg(g.pair_block + (tpa >> 16) * g.n_tower + (tpb >> 16));
        if (bi < 0) return false;
        blk = (uint32_t)bi;
    } else {
        const int32_t bi = __ldg(g.pair_block);
        if (bi < 0) return false;
        blk = (uint32_t)bi;
    }
    const int32_t lim = __ldg(g.blocks + ((size_t)blk * g.ppt + (tpa & 0xFFFFu)) * g.ppt + (tpb & 0xFFFFu));
    if (lim < 0) return false;
    const uint64_t l = (uint64_t)lim < W ? (uint64_t)lim : W;
    return dt <= l;
}
__device__ __forceinline__ uint64_t absdiff(int64_t a, int64_t b) { return a >= b ? udiff(a, b) : udiff(b, a); }

// ---- fast path, pass 1: neighbour rows.  One CTA per tile of 256 L1 hits x; the candidates (L1 hits of the
// same segment within +-Weff) are staged in shared memory.  Row of x: a bit mask of its causal neighbours over
// the L1 list, in a frame of kRowWords 32-bit words that starts at the word-aligned list index 32 f (so two rows
// are brought to a common frame by a word offset, no bit shifts).  Three steps per tile:
//   (1) thread per x: window [lo, hi) by binary search; which candidates sit on a tower that is connected to
//       x's tower at all (a byte table of the tower pairs in shared memory, no global gather; cfg4: 27 %
//       survive).  A pair inside the tile is owned by its earlier hit, so it is tested once.
//   (2) the surviving (x, y) pairs of the whole tile are written to a dense list;
//   (3) thread per pair: table entry + time test, result bits OR-ed into the rows of both hits.
// A hit with more than kRowSpan candidates ("wide") goes to the slow list instead.
constexpr int kRowTile = 256;
constexpr int kRowSpan = 256;            // candidates a row can hold
constexpr int kRowHalo = kRowSpan;       // a window of <= kRowSpan hits never leaves [x - 255, x + 256]
constexpr int kRowStage = kRowTile + 2 * kRowHalo;  // staged records per tile: always [x0 - 256, x0 + 512)
constexpr int kRowPer = kRowStage / kRowTile;  // 3
constexpr int kRowWords = 10;            // (31 + kRowSpan) / 32 + 1 = 9, padded to a 48-byte row
constexpr int kPairList = 256 * 16;       // pair lists of one round: 8 warps x (32 hits x 16 offsets)
constexpr int kPairBytesMax = 16384;     // tower-pair byte table in shared memory: n_tower <= 128
constexpr uint32_t kWide = 0xFFFFFFFFu;

struct Row {  // 48 bytes
    uint32_t w[kRowWords];
    uint32_t f;    // frame: bit b of w[k] <=> L1 list index 32 (f + k) + b;  kWide = no row (slow list)
    uint32_t deg;  // number of neighbours | (number of words in use) << 16
};

struct RowSmem {
    int64_t t[kRowStage];
    uint32_t idx[kRowStage];
    uint32_t tp[kRowStage];
    uint32_t row[kRowWords][kRowTile];   // step 3: causal neighbours (x's frame)
    uint32_t lo[kRowTile];               // window start (staged index); kWide = wide / not staged
    uint32_t boff[kRowTile];             // bit of candidate y in x's frame: boff + (y - lo)
    uint16_t list[kPairList];            // pair of the current round: stream << 12 | (x - x0) << 4 | offset in the round
    uint32_t next;                       // next tile of this CTA (dynamic schedule: dense tiles cost 10x)
};

__global__ void __launch_bounds__(kRowTile) l2_rows_kernel(const L1Rec* __restrict__ l1, const uint32_t* __restrict__ m_ptr,
                                                           const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                           uint32_t n, tt_geometry_dev g, uint64_t W, uint32_t N,
                                                           uint32_t mode, uint32_t pair_smem, uint8_t* __restrict__ flags,
                                                           uint8_t* __restrict__ l2bit, Row* __restrict__ rows,
                                                           uint32_t* __restrict__ slow_list, uint32_t* __restrict__ slow_cnt) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RowSmem& sm = *reinterpret_cast<RowSmem*>(smem_raw);
    unsigned char* s_pair = smem_raw + sizeof(RowSmem);  // [n_tower * n_tower] block id, 0xFF = unconnected
    const uint32_t m = *m_ptr;
    const uint32_t tid = threadIdx.x;
    const bool any_edge = g.max_dt >= 0;
    const uint64_t Weff = any_edge ? ((uint64_t)g.max_dt < W ? (uint64_t)g.max_dt : W) : 0;
    const uint32_t ntiles = (m + kRowTile - 1) / kRowTile;
    const uint32_t nt = g.n_tower;
    if (pair_smem && blockIdx.x < ntiles) {
        for (uint32_t i = tid; i < nt * nt; i += kRowTile) {
            const int32_t bi = __ldg(g.pair_block + i);
            s_pair[i] = bi < 0 ? (unsigned char)0xFF : (unsigned char)bi;
        }
    }
    const int32_t blk_single = nt == 1 ? __ldg(g.pair_block) : -1;
    // staged slot e of a tile <-> list index x0 - kRowHalo + e; slots outside [0, m) hold a record that is in no window
    L1Rec pre[kRowPer];
    auto fetch = [&](uint32_t tile) {
        const uint32_t x0 = tile * kRowTile;
#pragma unroll
        for (int k = 0; k < kRowPer; ++k) {
            const uint32_t e = tid + k * kRowTile;
            const uint32_t y = x0 - (uint32_t)kRowHalo + e;  // wraps below 0: then y >= m
            L1Rec r;
            r.t = 0; r.idx = 0xFFFFFFFFu; r.tp = kBadTp;
            if (y < m) r = l1[y];
            pre[k] = r;
        }
    };
    if (blockIdx.x < ntiles) fetch(blockIdx.x);
    uint32_t* const tile_ctr = slow_cnt + 1;  // zeroed with slow_cnt
    for (uint32_t tile = blockIdx.x; tile < ntiles;) {
        const uint32_t x0 = tile * kRowTile, x1 = min(m, x0 + kRowTile);
        const uint32_t ylo = x0 - (uint32_t)kRowHalo;          // list index of staged slot 0 (modulo 2^32)
        const uint32_t e_lo = x0 >= (uint32_t)kRowHalo ? 0u : (uint32_t)kRowHalo - x0;  // first real slot
        const uint32_t e_hi = min((uint32_t)kRowStage, m - ylo);                       // end of the real slots
#pragma unroll
        for (int k = 0; k < kRowPer; ++k) {
            const uint32_t e = tid + k * kRowTile;
            sm.t[e] = pre[k].t; sm.idx[e] = pre[k].idx; sm.tp[e] = pre[k].tp;
        }
        __syncthreads();
        if (tid == 0) sm.next = gridDim.x + atomicAdd(tile_ctr, 1u);
        const bool staged = true;
        const uint32_t x = x0 + tid;
        const uint32_t xl = x - ylo;   // staged index of x
        const uint32_t t0l = x0 - ylo, t1l = x1 - ylo;  // staged range of the tile
        // ---- step 1a: windows ----------------------------------------------------------------------------
        uint32_t lo = 0, hi = 0, f = kWide, boff = 0, words = 0;
        bool wide = false;
        if (x < x1) {
            wide = !staged;
            if (staged) {
                const uint32_t cnt = e_hi;
                const int64_t tx = sm.t[xl];
                uint32_t sa = 0, sb = n;
                if (n_seg > 1) {
                    const uint32_t s = find_segment(seg_off, n_seg, sm.idx[xl]);
                    sa = __ldg(seg_off + s); sb = __ldg(seg_off + s + 1);
                }
                // first y <= x with idx >= sa and tx - t_y <= Weff (monotone false..true on [0, xl])
                uint32_t a = e_lo, b = xl;
                while (a < b) { const uint32_t mid = (a + b) >> 1; if (sm.idx[mid] >= sa && udiff(tx, sm.t[mid]) <= Weff) b = mid; else a = mid + 1; }
                lo = a;
                // first y > x that is out (idx >= sb or t_y - tx > Weff): monotone true..false on (xl, cnt)
                a = xl + 1; b = cnt;
                while (a < b) { const uint32_t mid = (a + b) >> 1; if (sm.idx[mid] < sb && udiff(sm.t[mid], tx) <= Weff) a = mid + 1; else b = mid; }
                hi = a;
                if (hi - lo > (uint32_t)kRowSpan) wide = true;
                else {
                    f = (ylo + lo) >> 5;
                    boff = (ylo + lo) & 31u;
                    words = (boff + (hi - lo) + 31u) >> 5;  // <= 9
                }
            }
        }
        sm.lo[tid] = (x < x1 && !wide) ? lo : kWide;
        sm.boff[tid] = boff;
#pragma unroll
        for (int k = 0; k < kRowWords; ++k) sm.row[k][tid] = 0;
        __syncthreads();
        const uint32_t next_tile = sm.next;
        if (next_tile < ntiles) fetch(next_tile);  // in flight while this tile is worked on
        // ---- steps 1b-3 in rounds of 16 list offsets: every warp walks its 32 hits in lockstep over the later
        // candidates y = x + 1 + d (a pair inside the tile is owned by its earlier hit, with or without a row, so it
        // is tested once) and over the candidates before the tile, y = lo + d; the ones on connected towers
        // (cfg4: ~27 %) are appended to the tile's pair list with one shared-memory atomic per warp and step,
        // then tested one thread per pair.  256 hits x 16 offsets always fit the list.
        const uint32_t tpx = (x < x1 && staged) ? sm.tp[xl] : kBadTp;
        const uint32_t prow = (tpx >> 16) * nt;
        const bool emits = x < x1 && any_edge && tpx != kBadTp && (nt > 1 || blk_single >= 0);
        const uint32_t fwd_end = emits ? (wide ? min(hi, t1l) : hi) : 0u;   // later candidates: [xl + 1, fwd_end)
        const uint32_t reach = fwd_end > xl + 1u ? fwd_end - xl - 1u : 0u;
        const uint32_t lane = tid & 31u, warp = tid >> 5;
        // Every warp keeps its own pair list and tests its own pairs: the rounds need no block-wide barrier and no
        // shared counter (the row bits are OR-ed with atomics anyway), so a warp with a short reach does not wait for
        // the dense ones round by round.
        uint16_t* const wlist = sm.list + warp * (uint32_t)(kPairList / (kRowTile / 32));
        // the listed pairs, one thread per pair, four in flight (the table gather is the latency).  mode 0: entry =
        // tile index of x << 4 | offset, y = x + 1 + base + offset; mode 1: entry = tile index << 3 | offset,
        // y = lo(x) + base + offset
        auto test_pairs = [&](uint32_t np, uint32_t mode, uint32_t base) {
            for (uint32_t p0 = lane; p0 < np; p0 += 4u * 32u) {
                uint32_t xt4[4], y4[4];
                int32_t lim4[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t p = p0 + (uint32_t)u * 32u;
                    lim4[u] = -1; xt4[u] = 0; y4[u] = 0;
                    if (p < np) {
                        const uint32_t pr = wlist[p];
                        const uint32_t xt = mode ? pr >> 3 : pr >> 4, xs = t0l + xt;  // tile index / staged index of x
                        const uint32_t y = (mode ? sm.lo[xt] + (pr & 7u) : xs + 1u + (pr & 15u)) + base;  // staged index of y
                        const uint32_t tpa = sm.tp[xs], tpb = sm.tp[y];
                        int32_t bi;
                        if (nt == 1) bi = blk_single;
                        else if (pair_smem) { const uint32_t v = s_pair[(tpa >> 16) * nt + (tpb >> 16)]; bi = v == 0xFF ? -1 : (int32_t)v; }
                        else bi = __ldg(g.pair_block + (tpa >> 16) * nt + (tpb >> 16));
                        xt4[u] = xt; y4[u] = y;
                        if (bi >= 0) lim4[u] = __ldg(g.blocks + ((size_t)(uint32_t)bi * g.ppt + (tpa & 0xFFFFu)) * g.ppt + (tpb & 0xFFFFu));
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int32_t lim = lim4[u];
                    if (lim < 0) continue;
                    const uint32_t xt = xt4[u], y = y4[u], xs = t0l + xt;
                    const uint64_t l = (uint64_t)lim < W ? (uint64_t)lim : W;
                    if (absdiff(sm.t[xs], sm.t[y]) > l) continue;
                    const uint32_t xlo2 = sm.lo[xt];
                    if (xlo2 != kWide) {
                        const uint32_t bx = sm.boff[xt] + (y - xlo2);
                        atomicOr(&sm.row[bx >> 5][xt], 1u << (bx & 31u));
                    }
                    if (y >= t0l && y < t1l) {  // the partner is in the tile: its row gets the mirrored bit
                        const uint32_t yt = y - t0l, ylo2 = sm.lo[yt];
                        if (ylo2 != kWide) {
                            const uint32_t by = sm.boff[yt] + (xs - ylo2);
                            atomicOr(&sm.row[by >> 5][yt], 1u << (by & 31u));
                        }
                    }
                }
            }
        };
        // ---- phase A: every warp walks its own 32 hits in lockstep over the LATER candidates y = x + 1 + d, 16
        // offsets per round (a pair inside the tile is owned by its earlier hit, so it is tested once)
        for (uint32_t r = 0;; ++r) {
            if (!__any_sync(0xffffffffu, reach > 16u * r)) break;
            uint32_t np = 0;  // warp-uniform
            const uint32_t y0 = xl + 1u + 16u * r;
            // the 16 offsets of the round in three straight-line sweeps (16 independent loads each, no early exit)
            uint32_t tp16[16];
#pragma unroll
            for (uint32_t dd = 0; dd < 16u; ++dd) tp16[dd] = y0 + dd < fwd_end ? sm.tp[y0 + dd] : kBadTp;
            uint32_t cm = 0;  // bit dd: candidate on a connected tower
#pragma unroll
            for (uint32_t dd = 0; dd < 16u; ++dd) {
                bool c = tp16[dd] != kBadTp;
                if (c && pair_smem) c = s_pair[prow + (tp16[dd] >> 16)] != 0xFF;
                cm |= (c ? 1u : 0u) << dd;
            }
#pragma unroll
            for (uint32_t dd = 0; dd < 16u; ++dd) {
                const bool c = (cm >> dd) & 1u;
                const uint32_t mk = __ballot_sync(0xffffffffu, c);
                if (c) wlist[np + (uint32_t)__popc(mk & ((1u << lane) - 1u))] = (uint16_t)((tid << 4) | dd);
                np += (uint32_t)__popc(mk);
            }
            __syncwarp();
            test_pairs(np, 0u, 16u * r);
            __syncwarp();  // the list is rewritten in the next round
        }
        // ---- phase B: the candidates BEFORE the tile, y = lo(x) + d < first hit of the tile.  Only the first hits of
        // a tile have them (the whole load of an extra pass for the first warp, and the rest of the block waited for
        // it at the barrier below): now shared by all warps -- batch by batch of 32 hits, warp w takes the offsets
        // d with (d / 8) % 8 == w.
        for (uint32_t bq = 0; bq < (uint32_t)kRowTile / 32u; ++bq) {
            const uint32_t xt = 32u * bq + lane;
            uint32_t lo_b = 0, cnt_b = 0, prow_b = 0;
            if (x0 + xt < x1) {
                const uint32_t l0 = sm.lo[xt], tpb = sm.tp[t0l + xt];
                if (l0 != kWide && l0 < t0l && any_edge && tpb != kBadTp && (nt > 1 || blk_single >= 0)) {
                    lo_b = l0; cnt_b = t0l - l0; prow_b = (tpb >> 16) * nt;
                }
            }
            if (!__any_sync(0xffffffffu, cnt_b > 0u)) break;  // windows move forward: no later batch has any either
            for (uint32_t base = 8u * warp;; base += 8u * (uint32_t)(kRowTile / 32)) {
                if (!__any_sync(0xffffffffu, cnt_b > base)) break;
                uint32_t np = 0;
#pragma unroll
                for (uint32_t dd = 0; dd < 8u; ++dd) {
                    bool c = base + dd < cnt_b;
                    if (c) {
                        const uint32_t tpy = sm.tp[lo_b + base + dd];
                        c = tpy != kBadTp && !(pair_smem && s_pair[prow_b + (tpy >> 16)] == 0xFF);
                    }
                    const uint32_t mk = __ballot_sync(0xffffffffu, c);
                    if (c) wlist[np + (uint32_t)__popc(mk & ((1u << lane) - 1u))] = (uint16_t)((xt << 3) | dd);
                    np += (uint32_t)__popc(mk);
                }
                __syncwarp();
                test_pairs(np, 1u, base);
                __syncwarp();
            }
        }
        __syncthreads();  // all rows complete (bits come from other warps too)
        // ---- rows out -------------------------------------------------------------------------------------
        if (x < x1) {
            uint32_t deg = 0;
            Row row;
#pragma unroll
            for (int k = 0; k < kRowWords; ++k) {
                row.w[k] = wide ? 0u : sm.row[k][tid];
                deg += __popc(row.w[k]);
            }
            row.f = wide ? kWide : f;
            row.deg = deg | (words << 16);
            rows[x] = row;
            if (wide) {
                l2bit[x] = 0;
                slow_list[atomicAdd(slow_cnt, 1u)] = x;
            } else {
                const bool star = deg + 1 >= N;
                const bool decided = mode == 1 || N <= 2 || !star;  // clique test needed only for star hits, N > 2
                uint32_t fl = 0;
                if (star) fl |= TT_L2STAR;
                if (decided && star) fl |= TT_L2;
                if (fl) flags[sm.idx[xl]] |= (uint8_t)fl;
                l2bit[x] = (decided && star) ? 1 : 0;
            }
        }
        __syncthreads();
        tile = next_tile;
    }
}

// ---- fast path, pass 2: exact clique test on the rows (no table lookups).  One thread per star hit; the
// rows of a tile of hits and of everything their masks can name (+-(kRowSpan - 1) list positions) are
// staged in shared memory, so a neighbour's row is a shared-memory read at a word offset.
constexpr int kClqTile = 256;

// The same depth-first search as the generic loop in l2_clique_kernel (lowest candidate first, remove it, descend
// with cand & adj(v) while enough candidates are left), written as a recursion over the number REM of vertices still
// wanted so that every candidate mask is a statically indexed register array: NW words cover the frame of x, and
// the depth is a template parameter.  Returns 0 = no clique, 1 = found, 2 = a wide row was met (slow list).
template <int NW, int REM>
struct CliqueDfs {
    static __device__ __forceinline__ int run(uint32_t (&c)[NW], int cnt, uint32_t fx, const Row* s_rows, uint32_t base) {
        while (cnt >= REM) {
            uint32_t v = 0;
            bool got = false;
#pragma unroll
            for (int i = 0; i < NW; ++i)
                if (!got && c[i]) { v = 32u * (uint32_t)i + (uint32_t)__ffs(c[i]) - 1u; got = true; }
#pragma unroll
            for (int i = 0; i < NW; ++i)
                if ((uint32_t)i == (v >> 5)) c[i] &= ~(1u << (v & 31u));
            --cnt;
            if (REM == 1) return 1;  // v completes the clique
            const Row& rv = s_rows[32u * fx + v - base];
            if (rv.f == kWide) return 2;
            const int off = (int)fx - (int)rv.f;  // word i of x's frame is word i + off of v's
            uint32_t nx[NW];
            int cn = 0;
#pragma unroll
            for (int i = 0; i < NW; ++i) {
                const int j = i + off;
                const uint32_t a = (j >= 0 && j < kRowWords) ? rv.w[j] : 0u;
                nx[i] = c[i] & a;
                cn += __popc(nx[i]);
            }
            if (cn >= REM - 1) {
                const int r = CliqueDfs<NW, REM - 1>::run(nx, cn, fx, s_rows, base);
                if (r) return r;
            }
        }
        return 0;
    }
};
template <int NW>
struct CliqueDfs<NW, 0> {
    static __device__ __forceinline__ int run(uint32_t (&)[NW], int, uint32_t, const Row*, uint32_t) { return 1; }
};
constexpr int kClqStage = kClqTile + 2 * (kRowSpan - 1);  // 766 rows, 36.8 KB

__global__ void __launch_bounds__(kClqTile) l2_clique_kernel(const L1Rec* __restrict__ l1, const uint32_t* __restrict__ m_ptr,
                                                             const Row* __restrict__ rows, uint32_t N, uint32_t mode,
                                                             uint8_t* __restrict__ flags, uint8_t* __restrict__ l2bit,
                                                             uint32_t* __restrict__ slow_list, uint32_t* __restrict__ slow_cnt) {
    if (mode != 0 || N <= 2) return;
    __shared__ __align__(16) Row s_rows[kClqStage];
    const uint32_t m = *m_ptr;
    const uint32_t tid = threadIdx.x;
    const int K = (int)N - 1;  // clique size wanted among the neighbours of x
    const uint32_t ntiles = (m + kClqTile - 1) / kClqTile;
    __shared__ uint32_t s_next;
    uint32_t* const tile_ctr = slow_cnt + 2;  // zeroed with slow_cnt
    for (uint32_t tile = blockIdx.x; tile < ntiles;) {
        if (tid == 0) s_next = gridDim.x + atomicAdd(tile_ctr, 1u);
        const uint32_t x0 = tile * kClqTile, x1 = min(m, x0 + kClqTile);
        // rows the masks of this tile can name: windows move forward with x, so the first and the last row of the
        // tile bound them (a wide row at either end: the full +-(kRowSpan - 1))
        uint32_t base = x0 >= (uint32_t)(kRowSpan - 1) ? x0 - (kRowSpan - 1) : 0u;
        uint32_t top = min(m, x1 + (uint32_t)(kRowSpan - 1));
        {
            const uint32_t f0 = rows[x0].f, f1 = rows[x1 - 1].f, nw1 = rows[x1 - 1].deg >> 16;
            if (f0 != kWide) base = max(base, min(x0, 32u * f0));
            if (f1 != kWide) top = min(top, max(x1, 32u * (f1 + nw1)));
        }
        {   // rows [base, top) as 16-byte pieces, coalesced
            const uint4* src = reinterpret_cast<const uint4*>(rows + base);
            uint4* dst = reinterpret_cast<uint4*>(s_rows);
            const uint32_t pieces = (top - base) * (uint32_t)(sizeof(Row) / 16);
            for (uint32_t i = tid; i < pieces; i += kClqTile) dst[i] = src[i];
        }
        __syncthreads();
        const uint32_t x = x0 + tid;
        if (x < x1) {
            const Row& rx = s_rows[x - base];
            if (rx.f != kWide && (rx.deg & 0xFFFFu) + 1 >= N && (rx.deg >> 16) <= 3u && K <= 4) {
                // the usual case (a window of <= 96 candidates, N <= 5): masks in registers
                uint32_t c0[3] = {rx.w[0], rx.w[1], rx.w[2]};
                const int cnt0 = (int)(rx.deg & 0xFFFFu);
                int r = 0;
                switch (K) {
                    case 2: r = CliqueDfs<3, 2>::run(c0, cnt0, rx.f, s_rows, base); break;
                    case 3: r = CliqueDfs<3, 3>::run(c0, cnt0, rx.f, s_rows, base); break;
                    default: r = CliqueDfs<3, 4>::run(c0, cnt0, rx.f, s_rows, base); break;
                }
                if (r == 2) {
                    slow_list[atomicAdd(slow_cnt, 1u)] = x;
                } else if (r == 1) {
                    flags[l1[x].idx] |= (uint8_t)TT_L2;
                    l2bit[x] = 1;
                }
            } else if (rx.f != kWide && (rx.deg & 0xFFFFu) + 1 >= N) {
                uint32_t cand[TT_MAX_MULTIPLICITY][kRowWords];
                const int nw = (int)(rx.deg >> 16);  // words of the frame that can hold a neighbour of x
                for (int i = 0; i < nw; ++i) cand[0][i] = rx.w[i];
                const uint32_t fx = rx.f;
                int cnt[TT_MAX_MULTIPLICITY + 1];  // candidates left on every level
                cnt[0] = (int)(rx.deg & 0xFFFFu);
                int d = 0;
                bool found = false, punt = false;
                while (true) {
                    const int rem = K - d;
                    if (rem == 0) { found = true; break; }
                    if (cnt[d] < rem) {
                        if (d == 0) break;
                        --d;
                        continue;
                    }
                    // lowest candidate v, remove it, descend with cand & adj(v)
                    uint32_t v = 0;
                    for (int i = 0; i < nw; ++i)
                        if (cand[d][i]) { v = 32u * (uint32_t)i + (uint32_t)__ffs(cand[d][i]) - 1u; break; }
                    cand[d][v >> 5] &= ~(1u << (v & 31u));
                    cnt[d] -= 1;
                    if (rem == 1) { found = true; break; }  // v completes the clique
                    const Row& rv = s_rows[32u * fx + v - base];
                    if (rv.f == kWide) { punt = true; break; }
                    const int off = (int)fx - (int)rv.f;  // word i of x's frame is word i + off of v's
                    int c = 0;
                    for (int i = 0; i < nw; ++i) {
                        const int j = i + off;
                        const uint32_t a = (j >= 0 && j < kRowWords) ? rv.w[j] : 0u;
                        const uint32_t w = cand[d][i] & a;
                        cand[d + 1][i] = w;
                        c += __popc(w);
                    }
                    if (c >= rem - 1) { cnt[d + 1] = c; ++d; }  // else no clique through v on this level
                }
                if (punt) {
                    slow_list[atomicAdd(slow_cnt, 1u)] = x;
                } else if (found) {
                    flags[l1[x].idx] |= (uint8_t)TT_L2;
                    l2bit[x] = 1;
                }
            }
        }
        const uint32_t next_tile = s_next;  // written before the barrier after the staging
        __syncthreads();
        tile = next_tile;
    }
}

// ---- wide path: one warp per listed L1 hit (windows of more than 128 candidates: muon tracks, bursts).
// The window [lo, hi) of x is a bitmask of up to kMaxWin candidates in shared memory; the clique search is
// a lazy depth-first search: mask[d+1] = {c in mask[d] : edge(v, c)} is evaluated on demand for the picked
// vertex v only, so a dense clique (a track) is found after N-2 refinements instead of a full adjacency
// matrix.  A found clique marks ALL its members L2 (each of them is in an N-clique), which lets the other
// hits of the same track skip their own search.
constexpr int kL2Warps = 4;
constexpr int kMaxWin = TT_MAX_NEIGHBOURS;   // candidates per window
constexpr int kWinWords = kMaxWin / 32;

struct WideSmem {
    uint32_t mask[TT_MAX_MULTIPLICITY][kWinWords];
};

__global__ void __launch_bounds__(kL2Warps * 32) l2_wide_kernel(const L1Rec* __restrict__ l1,
                                                                const uint32_t* __restrict__ m_ptr,
                                                                const uint32_t* __restrict__ slow_list,
                                                                const uint32_t* __restrict__ slow_cnt,
                                                                const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                                uint32_t n, tt_geometry_dev g, uint64_t W, uint32_t N,
                                                                uint32_t mode, uint8_t* flags, volatile uint8_t* l2bit,
                                                                int32_t* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WideSmem& sm = reinterpret_cast<WideSmem*>(smem_raw)[warp];
    const uint32_t m = *m_ptr, nlist = *slow_cnt;
    const uint32_t nwarps = gridDim.x * kL2Warps;
    const bool any_edge = g.max_dt >= 0;
    const uint64_t Weff = any_edge ? ((uint64_t)g.max_dt < W ? (uint64_t)g.max_dt : W) : 0;
    const int K = (int)N - 1;
    for (uint32_t q = blockIdx.x * kL2Warps + warp; q < nlist; q += nwarps) {
        const uint32_t x = slow_list[q];
        const L1Rec rx = l1[x];
        uint32_t sa = 0, sb = n;
        if (n_seg > 1) {
            const uint32_t s = find_segment(seg_off, n_seg, rx.idx);
            sa = __ldg(seg_off + s);
            sb = __ldg(seg_off + s + 1);
        }
        // window extents
        uint32_t lo = x, hi = x + 1;
        for (uint32_t base = x; base > 0;) {
            const bool valid = base > lane;
            bool in = false;
            if (valid) { const L1Rec ry = l1[base - 1 - lane]; in = ry.idx >= sa && udiff(rx.t, ry.t) <= Weff; }
            const uint32_t ib = __ballot_sync(0xffffffffu, in);
            lo = base - __popc(ib);
            if (ib != 0xffffffffu) break;
            base -= 32;
        }
        for (uint32_t base = x + 1; base < m; base += 32) {
            const uint32_t y = base + lane;
            bool in = false;
            if (y < m) { const L1Rec ry = l1[y]; in = ry.idx < sb && udiff(ry.t, rx.t) <= Weff; }
            const uint32_t ib = __ballot_sync(0xffffffffu, in);
            hi = base + __popc(ib);
            if (ib != 0xffffffffu) break;
        }
        const uint32_t w = hi - lo;
        const bool fits = w <= (uint32_t)kMaxWin;
        const uint32_t nwords = (w + 31) >> 5;
        const bool live = rx.tp != kBadTp && any_edge;
        // neighbours of x
        uint32_t deg = 0;
        for (uint32_t k = 0; k < nwords; ++k) {
            const uint32_t y = lo + 32 * k + lane;
            bool e = false;
            if (live && y < hi && y != x) { const L1Rec ry = l1[y]; e = edge_tp(g, W, absdiff(rx.t, ry.t), rx.tp, ry.tp); }
            const uint32_t eb = __ballot_sync(0xffffffffu, e);
            if (fits && lane == 0) sm.mask[0][k] = eb;
            deg += __popc(eb);
        }
        __syncwarp();
        const bool star = deg + 1 >= N;
        bool l2 = star;
        if (star && mode == 0 && N > 2) {
            l2 = false;
            // lane 0 reads the byte another warp may be writing and shares it: the full-mask votes and shuffles of the
            // search below need every lane of the warp on the same path
            const uint32_t marked = __shfl_sync(0xffffffffu, lane == 0 ? (uint32_t)l2bit[x] : 0u, 0);
            if (!fits) {
                // more than TT_MAX_NEIGHBOURS candidates: the clique is not searched.  Fail open and deterministic: the
                // hit keeps its data (L2 := the exact L2STAR bit, a superset of the clique answer) and the status says so
                if (lane == 0) atomicOr(status, TT_S_DENSITY);
                l2 = true;
            } else if (marked) {
                l2 = true;  // already marked as a member of a clique found from another hit
            } else {
                // need K vertices of mask[0], pairwise adjacent
                uint32_t cnt[TT_MAX_MULTIPLICITY];
                uint32_t chosen[TT_MAX_MULTIPLICITY];
                cnt[0] = deg;
                int d = 0;
                while (true) {
                    const int rem = K - d;
                    if (cnt[d] < (uint32_t)rem) {
                        if (d == 0) break;
                        --d;
                        continue;
                    }
                    // lowest candidate v of mask[d]
                    uint32_t v = 0xFFFFFFFFu;
                    for (uint32_t k0 = 0; k0 < nwords; k0 += 32) {
                        const uint32_t k = k0 + lane;
                        const uint32_t wv = k < nwords ? sm.mask[d][k] : 0u;
                        const uint32_t nz = __ballot_sync(0xffffffffu, wv != 0);
                        if (nz) {
                            const uint32_t src = __ffs(nz) - 1;
                            const uint32_t word = __shfl_sync(0xffffffffu, wv, src);
                            v = (k0 + src) * 32 + (__ffs(word) - 1);
                            break;
                        }
                    }
                    chosen[d] = v;
                    if (rem == 1) { l2 = true; break; }
                    if (lane == 0) sm.mask[d][v >> 5] &= ~(1u << (v & 31));
                    cnt[d] -= 1;
                    __syncwarp();
                    const L1Rec rv = l1[lo + v];
                    uint32_t c = 0;
                    for (uint32_t k = 0; k < nwords; ++k) {
                        uint32_t nw = 0;
                        if (k >= (v >> 5)) {
                            const uint32_t bits = sm.mask[d][k];
                            bool e = false;
                            if ((bits >> lane) & 1u) {
                                const L1Rec ry = l1[lo + 32 * k + lane];
                                e = edge_tp(g, W, absdiff(rv.t, ry.t), rv.tp, ry.tp);
                            }
                            nw = __ballot_sync(0xffffffffu, e);
                        }
                        if (lane == 0) sm.mask[d + 1][k] = nw;
                        c += __popc(nw);
                    }
                    __syncwarp();
                    cnt[d + 1] = c;
                    ++d;
                }
                if (l2 && lane == 0) {  // mark the other members of the clique
                    for (int q2 = 0; q2 < K; ++q2) {
                        const uint32_t y = lo + chosen[q2];
                        l2bit[y] = 1;  // its TT_L2 flag is set by seed_write_kernel
                    }
                }
            }
        }
        if (lane == 0) {
            uint32_t f = 0;
            if (star) f |= TT_L2STAR;
            if (l2) f |= TT_L2;
            if (f) flags[rx.idx] |= (uint8_t)f;  // only this warp touches this byte here
            if (l2) l2bit[x] = 1;
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
                                                                  uint32_t* __restrict__ seeds, uint32_t cap,
                                                                  uint8_t* __restrict__ flags) {
    __shared__ uint32_t sm[33];
    uint32_t c0, c1;
    chunk_bounds(*m_ptr, c0, c1);
    uint32_t run = off[blockIdx.x];
    for (uint32_t base = c0; base < c1; base += kSeedThreads) {
        const uint32_t x = base + threadIdx.x;
        const bool is = x < c1 && l2bit[x];
        uint32_t total;
        const uint32_t r = block_exclusive_scan(is ? 1u : 0u, sm, &total);
        if (is) {
            const uint32_t i = l1[x].idx;
            flags[i] |= (uint8_t)TT_L2;  // idempotent; covers members marked by another hit's clique search
            if (run + r < cap) seeds[run + r] = i;
        }
        run += total;
    }
}

// ------------------------------------------------------------------------------------------------
struct TriggerPlan {
    uint32_t *blk_cnt, *scan_scratch, *m_total, *seed_cnt;
    L1Rec* l1;
    uint8_t* l2bit;
    Row* rows;
    uint32_t *slow_list, *slow_cnt;
    uint32_t nblk;
};

// cap: L1 hits the list arrays hold (n, or tt_params.l1_capacity if that is smaller)
static uint32_t l1_cap(uint32_t n, const tt_params* p) { return p->l1_capacity && p->l1_capacity < n ? p->l1_capacity : n; }

static void trigger_plan(Arena& a, uint32_t n, uint32_t cap, TriggerPlan& p) {
    p.nblk = div_up(n, kL1Tile);
    p.blk_cnt = a.take<uint32_t>(p.nblk + 1);
    p.scan_scratch = a.take<uint32_t>(scan_ws_count(p.nblk + 1));
    p.m_total = a.take<uint32_t>(1);
    p.seed_cnt = a.take<uint32_t>(kSeedBlocks);
    p.l1 = a.take<L1Rec>(cap);
    p.l2bit = a.take<uint8_t>(cap);
    p.rows = a.take<Row>(cap);
    p.slow_list = a.take<uint32_t>(cap);
    p.slow_cnt = a.take<uint32_t>(4);  // [0] slow-list length, [1] / [2] tile counters of the rows / clique kernels
}

}  // namespace tt

using namespace tt;

static int trigger_attrs() {
    TT_CUDA_OK(cudaFuncSetAttribute(l2_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(WideSmem) * kL2Warps)));
    TT_CUDA_OK(cudaFuncSetAttribute(l1_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(L1Smem)));
    TT_CUDA_OK(cudaFuncSetAttribute(l2_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(RowSmem) + kPairBytesMax)));
    return TT_OK;
}

static int trigger_args_ok(uint32_t n, const uint32_t* h_seg_offsets, uint32_t n_seg, const tt_geometry* g,
                           const tt_params* p) {
    if (!p || !g || n_seg < 1 || !h_seg_offsets) return TT_E_INVAL;
    if (p->l2_multiplicity < 1 || p->l2_multiplicity > TT_MAX_MULTIPLICITY || p->l2_mode > 1 ||
        p->lc_window_ps < 0 || p->l2_window_ps < 0 || p->event_half_ps < 0)
        return TT_E_INVAL;
    if (n >= 0xFFF00000u) return TT_E_INVAL;
    if (h_seg_offsets[0] != 0 || h_seg_offsets[n_seg] != n) return TT_E_INVAL;
    for (uint32_t s = 0; s < n_seg; ++s)
        if (h_seg_offsets[s] > h_seg_offsets[s + 1]) return TT_E_INVAL;
    return TT_OK;
}

static int trigger_l2(const TriggerPlan& plan, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                      const tt_geometry* g, const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds, uint32_t seed_cap,
                      uint32_t* d_n_seeds, int32_t* d_status, cudaStream_t s);

// Everything of tt_trigger_slice.  last == nullptr: L1 by l1_tile_kernel.  last != nullptr: the last merge level has
// written the in-tile L1 flags (fused call); the tile edges are finished here.
static int trigger_run(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                       const tt_geometry* g, const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds, uint32_t seed_cap,
                       uint32_t* d_n_seeds, void* d_ws, int32_t* d_status, cudaStream_t s, const MergeLast* last) {
    Arena a(d_ws);
    TriggerPlan plan;
    const uint32_t cap = l1_cap(n, p);
    trigger_plan(a, n, cap, plan);
    int rc = once_per_device(kSlotTrigger, trigger_attrs);
    if (rc != TT_OK) return rc;
    const uint32_t sms = (uint32_t)sm_count();
    if (!last) {
        prof_mark(s, "trig.l1_flags");
        TT_K(l1_tile_kernel)<<<plan.nblk, kL1Threads, sizeof(L1Smem), s>>>((const uint4*)d_sorted, n, d_seg_offsets, n_seg,
                                                        (uint64_t)p->lc_window_ps, p->q_thresh, d_flags, plan.blk_cnt);
    } else {
        prof_mark(s, "trig.l1_edges");
        if (last->tiles)
            TT_K(l1_boundary_kernel)<<<div_up(last->tiles, kBndWarps), kBndWarps * 32, 0, s>>>(
                last->lv, last->tiles, (const uint4*)d_sorted, (uint64_t)p->lc_window_ps, p->q_thresh, d_flags);
        TT_K(l1_count_kernel)<<<plan.nblk, kL1Threads, 0, s>>>(d_flags, n, plan.blk_cnt);
    }
    prof_mark(s, "trig.l1_scan");
    rc = exclusive_scan_u32(plan.blk_cnt, plan.blk_cnt, plan.nblk, plan.scan_scratch, plan.m_total, s);
    if (rc != TT_OK) return rc;
    prof_mark(s, "trig.l1_compact");
    TT_K(l1_compact_kernel)<<<plan.nblk, kL1Threads, 0, s>>>((const uint4*)d_sorted, n, d_flags, plan.blk_cnt, plan.l1,
                                                         cap, plan.m_total, g->dev.n_pmt, g->dev.ppt, d_status);
    return trigger_l2(plan, n, d_seg_offsets, n_seg, g, p, d_flags, d_seeds, seed_cap, d_n_seeds, d_status, s);
}

// L2 (rows, clique, wide) and the ordered seed list over the L1 list plan.l1[*plan.m_total].  `n` bounds the `idx`
// fields of the list (the sorted hit array, or the list itself in tt_l2_merged); flags / seeds are indexed by them.
static int trigger_l2(const TriggerPlan& plan, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                      const tt_geometry* g, const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds, uint32_t seed_cap,
                      uint32_t* d_n_seeds, int32_t* d_status, cudaStream_t s) {
    const uint32_t sms = (uint32_t)sm_count();
    prof_mark(s, "trig.l2_rows");
    TT_CUDA_OK(cudaMemsetAsync(plan.slow_cnt, 0, 4 * sizeof(uint32_t), s));
    const uint32_t nt2 = g->dev.n_tower * g->dev.n_tower;
    const uint32_t pair_smem = (g->dev.n_tower > 1 && nt2 <= (uint32_t)kPairBytesMax && g->dev.n_blocks <= 255u) ? 1u : 0u;
    const size_t rows_smem = sizeof(RowSmem) + (pair_smem ? ((nt2 + 15u) & ~15u) : 0);
    TT_K(l2_rows_kernel)<<<sms * 5, kRowTile, rows_smem, s>>>(
        plan.l1, plan.m_total, d_seg_offsets, n_seg, n, g->dev, (uint64_t)p->l2_window_ps, p->l2_multiplicity, p->l2_mode,
        pair_smem, d_flags, plan.l2bit, plan.rows, plan.slow_list, plan.slow_cnt);
    prof_mark(s, "trig.l2_clique");
    TT_K(l2_clique_kernel)<<<sms * 6, kClqTile, 0, s>>>(plan.l1, plan.m_total, plan.rows, p->l2_multiplicity, p->l2_mode,
                                                        d_flags, plan.l2bit, plan.slow_list, plan.slow_cnt);
    prof_mark(s, "trig.l2_wide");
    TT_K(l2_wide_kernel)<<<sms * 12, kL2Warps * 32, sizeof(WideSmem) * kL2Warps, s>>>(
        plan.l1, plan.m_total, plan.slow_list, plan.slow_cnt, d_seg_offsets, n_seg, n, g->dev, (uint64_t)p->l2_window_ps,
        p->l2_multiplicity, p->l2_mode, d_flags, plan.l2bit, d_status);
    prof_counter(s, "l1_hits", plan.m_total);
    prof_counter(s, "l2_slow_items", plan.slow_cnt);
    prof_mark(s, "trig.seeds");
    TT_K(seed_count_kernel)<<<kSeedBlocks, kSeedThreads, 0, s>>>(plan.l2bit, plan.m_total, plan.seed_cnt);
    TT_K(count_scan_kernel)<<<1, 1024, 0, s>>>(plan.seed_cnt, kSeedBlocks, d_n_seeds, seed_cap, TT_S_SEED_OVERFLOW, d_status);
    TT_K(seed_write_kernel)<<<kSeedBlocks, kSeedThreads, 0, s>>>(plan.l2bit, plan.l1, plan.m_total, plan.seed_cnt, d_seeds,
                                                           seed_cap, d_flags);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

extern "C" int tt_trigger_slice(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                                const uint32_t* h_seg_offsets, uint32_t n_seg, const tt_geometry* g,
                                const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds, uint32_t seed_cap,
                                uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes, int32_t* d_status, void* stream) {
    if (!ws_bytes) return TT_E_INVAL;
    int rc = trigger_args_ok(n, h_seg_offsets, n_seg, g, p);
    if (rc != TT_OK) return rc;
    Arena sizing(nullptr);
    TriggerPlan plan;
    trigger_plan(sizing, n, l1_cap(n, p), plan);
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
    return trigger_run(d_sorted, n, d_seg_offsets, n_seg, g, p, d_flags, d_seeds, seed_cap, d_n_seeds, d_ws, d_status, s,
                       nullptr);
}

// tt_sort_slice + tt_trigger_slice in one call (last bullet): same outputs, byte for byte.  With runs
// given, L1 is evaluated by the last merge level on its sorted tile in shared memory, so the sorted array is not read
// again for it; without runs (radix sort) the two calls simply run back to back.
extern "C" int tt_sort_trigger_slice(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n,
                                     const uint32_t* d_seg_offsets, const uint32_t* h_seg_offsets, uint32_t n_seg,
                                     const uint32_t* d_run_offsets, const uint32_t* h_run_offsets, uint32_t n_runs,
                                     const tt_geometry* g, const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds,
                                     uint32_t seed_cap, uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes,
                                     int32_t* d_status, void* stream) {
    if (!ws_bytes) return TT_E_INVAL;
    int rc = trigger_args_ok(n, h_seg_offsets, n_seg, g, p);
    if (rc != TT_OK) return rc;
    size_t ws_sort = 0, ws_trig = 0;
    rc = tt_sort_slice(nullptr, nullptr, nullptr, n, nullptr, h_seg_offsets, n_seg, d_run_offsets, h_run_offsets, n_runs,
                       nullptr, &ws_sort, nullptr, nullptr);
    if (rc != TT_OK) return rc;
    rc = tt_trigger_slice(nullptr, n, nullptr, h_seg_offsets, n_seg, g, p, nullptr, nullptr, seed_cap, nullptr, nullptr,
                          &ws_trig, nullptr, nullptr);
    if (rc != TT_OK) return rc;
    ws_sort = (ws_sort + 255) & ~size_t(255);
    if (!d_ws) {
        *ws_bytes = ws_sort + ws_trig;
        return TT_OK;
    }
    if (*ws_bytes < ws_sort + ws_trig) return TT_E_WORKSPACE;
    if (!d_flags || !d_n_seeds || !d_status || (!d_seeds && seed_cap)) return TT_E_INVAL;
    if (n && (!d_in || !d_out || !d_seg_offsets || d_in == d_out)) return TT_E_INVAL;
    if (((uintptr_t)d_ws & 255) || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (n == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_n_seeds, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    void* d_ws_trig = (char*)d_ws + ws_sort;
    const bool runs = d_run_offsets != nullptr || h_run_offsets != nullptr;
    if (!runs) {
        size_t w = ws_sort;
        rc = tt_sort_slice(d_in, d_out, d_perm, n, d_seg_offsets, h_seg_offsets, n_seg, nullptr, nullptr, 0, d_ws, &w,
                           d_status, stream);
        if (rc != TT_OK) return rc;
        return trigger_run(d_out, n, d_seg_offsets, n_seg, g, p, d_flags, d_seeds, seed_cap, d_n_seeds, d_ws_trig, d_status,
                           s, nullptr);
    }
    if (!d_run_offsets || !h_run_offsets || n_runs < 1) return TT_E_INVAL;
    FuseL1 fz;
    fz.flags = d_flags;
    fz.lc = (uint64_t)p->lc_window_ps;
    fz.q_thresh = p->q_thresh;
    MergeLast last;
    last.tiles = 0;
    rc = merge_sort_runs(d_in, d_out, d_perm, n, d_seg_offsets, h_seg_offsets, n_seg, d_run_offsets, h_run_offsets, n_runs,
                         d_ws, d_status, s, &fz, &last);
    if (rc != TT_OK) return rc;
    return trigger_run(d_out, n, d_seg_offsets, n_seg, g, p, d_flags, d_seeds, seed_cap, d_n_seeds, d_ws_trig, d_status, s,
                       &last);
}

// ------------------------------------------------------------------------------------------------
// NEXT-4: the trigger of a multi-tower detector sharded BY TOWER over several GPUs, with ONE exchange (PAPER.md:81,
// sect. 5: "each TGPU finds the trigger seeds of its tower and sends them to a TCPU ... gets candidate times back";
// SURVEY.md 8(e)(ii)).  L1 is local to a floor, hence to a tower: every rank sorts and L1-tags the hits of its own
// towers (tt_sort_l1_slice), exports its L1 hits as 16-byte records (tt_l1_export), the ranks all-gather them
// (~2 % of the hits), merge the lists in time (tt_sort_slice: the record starts with the time, like a hit), and every
// rank evaluates the inter-tower L2 on the merged list (tt_l2_merged: the same kernels as tt_trigger_slice), takes the
// bits of its own hits (tt_l2_apply) and tags its hits inside the global event windows (tt_tag_windows).  The result
// is, hit for hit, what one GPU computes on the whole detector.
// ------------------------------------------------------------------------------------------------
namespace tt {

struct L1Hit {  // = tt_l1hit
    int64_t t;
    uint32_t idx;
    uint32_t ps;  // pmt_id | src << 16
};

__global__ void __launch_bounds__(kL1Threads) l1_export_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                               const uint8_t* __restrict__ flags,
                                                               const uint32_t* __restrict__ tile_off, uint32_t src,
                                                               L1Hit* __restrict__ out, uint32_t cap) {
    __shared__ uint32_t sm[33];
    const uint32_t i0 = blockIdx.x * (uint32_t)kL1Tile + threadIdx.x * kL1Per;
    uint32_t mask = 0;
    for (uint32_t k = 0; k < (uint32_t)kL1Per && i0 + k < n; ++k)
        if (flags[i0 + k] & TT_L1) mask |= 1u << k;
    uint32_t total;
    uint32_t r = tile_off[blockIdx.x] + block_exclusive_scan(__popc(mask), sm, &total);
    while (mask) {
        const uint32_t k = __ffs(mask) - 1;
        mask &= mask - 1;
        const uint32_t i = i0 + k;
        const uint4 v = __ldg(hits + i);
        L1Hit h;
        h.t = hit_time(v);
        h.idx = i;
        h.ps = (v.z & 0xFFFFu) | (src << 16);
        if (r < cap) out[r] = h;
        ++r;
    }
}

__global__ void __launch_bounds__(256) l1_export_finish_kernel(const uint32_t* __restrict__ m_total, uint32_t cap,
                                                               uint32_t* __restrict__ n_out, int32_t* __restrict__ status) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        *n_out = *m_total;
        if (*m_total > cap) atomicOr(status, TT_S_L1_OVERFLOW);
    }
}

__global__ void __launch_bounds__(256) l1hit_to_rec_kernel(const L1Hit* __restrict__ in, uint32_t m, uint32_t n_pmt,
                                                           uint32_t ppt, L1Rec* __restrict__ out,
                                                           uint32_t* __restrict__ m_total, int32_t* __restrict__ status) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x == 0) *m_total = m;
    bool bad = false;
    if (x < m) {
        const L1Hit h = in[x];
        L1Rec rec;
        rec.t = h.t;
        rec.idx = x;  // flags and seeds of tt_l2_merged are indexed by the position in the merged list
        const uint32_t pmt = h.ps & 0xFFFFu;
        if (pmt >= n_pmt) { rec.tp = kBadTp; bad = true; }
        else { const uint32_t tw = pmt / ppt; rec.tp = (tw << 16) | (pmt - tw * ppt); }
        out[x] = rec;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(status, TT_S_BAD_PMT);
}

__global__ void __launch_bounds__(kSeedThreads) l2_apply_count_kernel(const L1Hit* __restrict__ l1, const uint8_t* __restrict__ bits,
                                                                      uint32_t m, uint32_t src, uint32_t* __restrict__ cnt) {
    const uint32_t per = (m + gridDim.x - 1) / gridDim.x;
    const uint64_t a = (uint64_t)blockIdx.x * per;
    const uint32_t c0 = a < m ? (uint32_t)a : m, c1 = a + per < m ? (uint32_t)(a + per) : m;
    uint32_t c = 0;
    for (uint32_t x = c0 + threadIdx.x; x < c1; x += kSeedThreads)
        c += ((l1[x].ps >> 16) == src && (bits[x] & TT_L2)) ? 1u : 0u;
    __shared__ uint32_t sm[33];
    uint32_t total;
    block_exclusive_scan(c, sm, &total);
    if (threadIdx.x == 0) cnt[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kSeedThreads) l2_apply_write_kernel(const L1Hit* __restrict__ l1, const uint8_t* __restrict__ bits,
                                                                      uint32_t m, uint32_t src, const uint32_t* __restrict__ off,
                                                                      uint8_t* __restrict__ flags, uint32_t n,
                                                                      uint32_t* __restrict__ seeds, uint32_t cap) {
    __shared__ uint32_t sm[33];
    const uint32_t per = (m + gridDim.x - 1) / gridDim.x;
    const uint64_t a = (uint64_t)blockIdx.x * per;
    const uint32_t c0 = a < m ? (uint32_t)a : m, c1 = a + per < m ? (uint32_t)(a + per) : m;
    uint32_t run = off[blockIdx.x];
    for (uint32_t base = c0; base < c1; base += kSeedThreads) {
        const uint32_t x = base + threadIdx.x;
        bool is = false;
        uint32_t idx = 0;
        if (x < c1) {
            const L1Hit h = l1[x];
            if ((h.ps >> 16) == src && h.idx < n) {
                const uint32_t b = bits[x] & (uint32_t)(TT_L2STAR | TT_L2);
                idx = h.idx;
                flags[idx] = (uint8_t)((flags[idx] & ~(uint32_t)(TT_L2STAR | TT_L2)) | b);  // one record per hit: no race
                is = (b & TT_L2) != 0;
            }
        }
        uint32_t total;
        const uint32_t r = block_exclusive_scan(is ? 1u : 0u, sm, &total);
        if (is && run + r < cap) seeds[run + r] = idx;
        run += total;
    }
}

// INEVT for the hits of a sorted slice that lie inside one of the (ascending, disjoint) event windows
// [t_first - H, t_last + H], t_first = t_start + H and t_last = t_end - H (exact for any int64: unsigned differences)
__global__ void __launch_bounds__(256) tag_windows_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                          const tt_event* __restrict__ events,
                                                          const uint32_t* __restrict__ n_events_ptr, uint32_t event_cap,
                                                          uint64_t H, uint8_t* __restrict__ flags) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t ne = min(*n_events_ptr, event_cap);
    if (i >= n || ne == 0) return;
    const int64_t t = hit_time(__ldg(hits + i));
    uint32_t a = 0, b = ne;  // first event with t <= t_last + H
    while (a < b) {
        const uint32_t mid = a + ((b - a) >> 1);
        const int64_t t_last = (int64_t)((uint64_t)events[mid].t_end - H);
        if (t <= t_last || udiff(t, t_last) <= H) b = mid; else a = mid + 1;
    }
    if (a < ne) {
        const int64_t t_first = (int64_t)((uint64_t)events[a].t_start + H);
        if (t >= t_first || udiff(t_first, t) <= H) flags[i] |= (uint8_t)TT_INEVT;
    }
}

struct ExportPlan {
    uint32_t *blk_cnt, *scan_scratch, *m_total;
    uint32_t nblk;
};
static void export_plan(Arena& a, uint32_t n, ExportPlan& p) {
    p.nblk = div_up(n, kL1Tile);
    p.blk_cnt = a.take<uint32_t>(p.nblk + 1);
    p.scan_scratch = a.take<uint32_t>(scan_ws_count(p.nblk + 1));
    p.m_total = a.take<uint32_t>(1);
}

}  // namespace tt

extern "C" int tt_sort_l1_slice(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n,
                                const uint32_t* d_seg_offsets, const uint32_t* h_seg_offsets, uint32_t n_seg,
                                const uint32_t* d_run_offsets, const uint32_t* h_run_offsets, uint32_t n_runs,
                                const tt_params* p, uint8_t* d_flags, void* d_ws, size_t* ws_bytes, int32_t* d_status,
                                void* stream) {
    if (!ws_bytes || !p || p->lc_window_ps < 0 || !h_run_offsets || n_runs < 1) return TT_E_INVAL;
    size_t need = 0;
    int rc = tt_sort_slice(nullptr, nullptr, nullptr, n, nullptr, h_seg_offsets, n_seg, d_run_offsets ? d_run_offsets : h_run_offsets,
                           h_run_offsets, n_runs, nullptr, &need, nullptr, nullptr);
    if (rc != TT_OK) return rc;
    if (!d_ws) {
        *ws_bytes = need;
        return TT_OK;
    }
    if (*ws_bytes < need) return TT_E_WORKSPACE;
    if (n == 0) return TT_OK;
    if (!d_in || !d_out || !d_seg_offsets || !d_run_offsets || !d_flags || !d_status || d_in == d_out) return TT_E_INVAL;
    if (((uintptr_t)d_ws & 255) || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    FuseL1 fz;
    fz.flags = d_flags;
    fz.lc = (uint64_t)p->lc_window_ps;
    fz.q_thresh = p->q_thresh;
    MergeLast last;
    last.tiles = 0;
    rc = merge_sort_runs(d_in, d_out, d_perm, n, d_seg_offsets, h_seg_offsets, n_seg, d_run_offsets, h_run_offsets, n_runs,
                         d_ws, d_status, s, &fz, &last);
    if (rc != TT_OK) return rc;
    prof_mark(s, "trig.l1_edges");
    if (last.tiles)
        TT_K(l1_boundary_kernel)<<<div_up(last.tiles, kBndWarps), kBndWarps * 32, 0, s>>>(
            last.lv, last.tiles, (const uint4*)d_out, (uint64_t)p->lc_window_ps, p->q_thresh, d_flags);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

extern "C" int tt_l1_export(const tt_hit* d_sorted, uint32_t n, const uint8_t* d_flags, uint32_t src, tt_l1hit* d_l1,
                            uint32_t l1_cap, uint32_t* d_n_l1, void* d_ws, size_t* ws_bytes, int32_t* d_status,
                            void* stream) {
    if (!ws_bytes || src > 0xFFFFu || n >= 0xFFF00000u) return TT_E_INVAL;
    Arena sizing(nullptr);
    ExportPlan plan;
    export_plan(sizing, n, plan);
    if (!d_ws) {
        *ws_bytes = sizing.off;
        return TT_OK;
    }
    if (*ws_bytes < sizing.off) return TT_E_WORKSPACE;
    if (!d_n_l1 || !d_status || (n && (!d_sorted || !d_flags)) || (l1_cap && !d_l1) || ((uintptr_t)d_ws & 255)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (n == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_n_l1, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    Arena a(d_ws);
    export_plan(a, n, plan);
    prof_mark(s, "towers.l1_export");
    TT_K(l1_count_kernel)<<<plan.nblk, kL1Threads, 0, s>>>(d_flags, n, plan.blk_cnt);
    int rc = exclusive_scan_u32(plan.blk_cnt, plan.blk_cnt, plan.nblk, plan.scan_scratch, plan.m_total, s);
    if (rc != TT_OK) return rc;
    TT_K(l1_export_kernel)<<<plan.nblk, kL1Threads, 0, s>>>((const uint4*)d_sorted, n, d_flags, plan.blk_cnt, src,
                                                         reinterpret_cast<L1Hit*>(d_l1), l1_cap);
    TT_K(l1_export_finish_kernel)<<<1, 32, 0, s>>>(plan.m_total, l1_cap, d_n_l1, d_status);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

extern "C" int tt_l2_merged(const tt_l1hit* d_l1, uint32_t m, const tt_geometry* g, const tt_params* p, uint8_t* d_bits,
                            uint32_t* d_seeds, uint32_t seed_cap, uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes,
                            int32_t* d_status, void* stream) {
    if (!ws_bytes) return TT_E_INVAL;
    const uint32_t seg1[2] = {0, m};
    int rc = trigger_args_ok(m, seg1, 1, g, p);
    if (rc != TT_OK) return rc;
    Arena sizing(nullptr);
    TriggerPlan plan;
    trigger_plan(sizing, m, m, plan);
    if (!d_ws) {
        *ws_bytes = sizing.off;
        return TT_OK;
    }
    if (*ws_bytes < sizing.off) return TT_E_WORKSPACE;
    if (!d_n_seeds || !d_status || (!d_seeds && seed_cap) || (m && (!d_l1 || !d_bits)) || ((uintptr_t)d_ws & 255)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (m == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_n_seeds, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    Arena a(d_ws);
    trigger_plan(a, m, m, plan);
    rc = once_per_device(kSlotTrigger, trigger_attrs);
    if (rc != TT_OK) return rc;
    prof_mark(s, "towers.l2_prepare");
    TT_CUDA_OK(cudaMemsetAsync(d_bits, 0, m, s));
    TT_K(l1hit_to_rec_kernel)<<<div_up(m, 256), 256, 0, s>>>(reinterpret_cast<const L1Hit*>(d_l1), m, g->dev.n_pmt, g->dev.ppt,
                                                            plan.l1, plan.m_total, d_status);
    return trigger_l2(plan, m, nullptr, 1, g, p, d_bits, d_seeds, seed_cap, d_n_seeds, d_status, s);
}

extern "C" int tt_l2_apply(const tt_l1hit* d_l1, const uint8_t* d_bits, uint32_t m, uint32_t src, uint8_t* d_flags, uint32_t n,
                           uint32_t* d_seeds, uint32_t seed_cap, uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes,
                           int32_t* d_status, void* stream) {
    if (!ws_bytes || src > 0xFFFFu) return TT_E_INVAL;
    Arena sizing(nullptr);
    (void)sizing.take<uint32_t>(kSeedBlocks);
    if (!d_ws) {
        *ws_bytes = sizing.off;
        return TT_OK;
    }
    if (*ws_bytes < sizing.off) return TT_E_WORKSPACE;
    if (!d_n_seeds || !d_status || (!d_seeds && seed_cap) || (m && (!d_l1 || !d_bits || !d_flags)) || ((uintptr_t)d_ws & 255))
        return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (m == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_n_seeds, 0, sizeof(uint32_t), s));
        return TT_OK;
    }
    Arena a(d_ws);
    uint32_t* cnt = a.take<uint32_t>(kSeedBlocks);
    prof_mark(s, "towers.l2_apply");
    TT_K(l2_apply_count_kernel)<<<kSeedBlocks, kSeedThreads, 0, s>>>(reinterpret_cast<const L1Hit*>(d_l1), d_bits, m, src, cnt);
    TT_K(count_scan_kernel)<<<1, 1024, 0, s>>>(cnt, kSeedBlocks, d_n_seeds, seed_cap, TT_S_SEED_OVERFLOW, d_status);
    TT_K(l2_apply_write_kernel)<<<kSeedBlocks, kSeedThreads, 0, s>>>(reinterpret_cast<const L1Hit*>(d_l1), d_bits, m, src, cnt,
                                                                   d_flags, n, d_seeds, seed_cap);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

extern "C" int tt_tag_windows(const tt_hit* d_sorted, uint32_t n, const tt_event* d_events, const uint32_t* d_n_events,
                              uint32_t event_cap, const tt_params* p, uint8_t* d_flags, void* stream) {
    if (!p || p->event_half_ps < 0 || n >= 0xFFF00000u) return TT_E_INVAL;
    if (n == 0) return TT_OK;
    if (!d_sorted || !d_events || !d_n_events || !d_flags) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    prof_mark(s, "towers.tag_windows");
    TT_K(tag_windows_kernel)<<<div_up(n, 256), 256, 0, s>>>((const uint4*)d_sorted, n, d_events, d_n_events, event_cap,
                                                           (uint64_t)p->event_half_ps, d_flags);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}
