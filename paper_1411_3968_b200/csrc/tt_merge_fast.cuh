// tt_merge_fast.cuh -- the tile kernel of the run merge for the usual tile (included by tt_merge.cu inside namespace tt,
// after its shared-memory / TMA helpers).  PAPER.md:51-53: the sort; L1 on the sorted tile (fused call).
//
// One CTA per time tile, as merge_tile_kernel, but only the case that covers all but a handful of tiles of a real
// slice: <= kFCap hits in the tile's pieces, a tile narrower than 2^32 key units and wider than kFCap.  Everything
// else (skew, massive ties, >= 2^32 ps across a tile) is appended to a list that merge_slow_kernel works off with the
// general code.  What is different from merge_tile_kernel:
//   * the bucket map's multiplier comes from the plan (no 64-bit division per thread), the run-order check compares
//     the 32-bit key offsets of neighbouring lanes (one shuffle) instead of re-reading 64-bit keys;
//   * hits that are alone in their fine bucket (the majority) skip the in-bucket ordering;
//   * every thread then holds its records in registers, and after ONE barrier writes them to their ranks in the SAME
//     tile buffer (in-place permutation): the sorted tile is in shared memory, and leaves with one TMA bulk store;
//   * kFuse (last level of tt_sort_trigger_slice): Q and the same-floor coincidences are evaluated on that sorted tile
//     (32-bit relative times, forward scan, both partners marked) and the flag bytes are written with the records.
//     Partners in a neighbouring tile are not visible here: l1_boundary_kernel (tt_trigger.cu) finishes the hits
//     within LC of a tile edge with exact scans of the sorted array.

constexpr int kFThreads = 512;
constexpr int kFItems = 8;
constexpr int kFCap = kFThreads * kFItems;  // 4096 hits per tile at most; also the number of fine buckets
static_assert(kFCap <= 4096, "12-bit element ids / bucket ids");

struct FastSmem {
    uint4 tile[kFCap];               // staged run-major by TMA, then the sorted tile (in place)        64 KB
    uint32_t cs[kFCap + 4];          // buckets: count, then start << 16 | count; later relative times + 4 sentinels
    uint32_t list[kFCap + 4];        // bucket members (composites); later perm values / floor|pmt (+ 4 readable)
    uint32_t fl[kFCap / 4 + 8];      // kFuse: flag bytes, shifted so that 16-byte groups match the global array
    uint32_t segstart[kMaxFan + 1];  // tile-local start of every run piece
    uint32_t cur[kMaxFan];           // absolute index of the first hit of every piece
    uint32_t pstart[kFCap / 32];     // bitmap of piece starts (run-order check)
    uint32_t scan[64];
    uint32_t emit[4];                // EmitRange of this tile (thread kFThreads - 1 computes it while the tile is loading)
    uint64_t mbar;
};
static_assert(2 * (sizeof(FastSmem) + 1024) <= 233472, "two CTAs per SM");
static_assert(offsetof(FastSmem, fl) % 16 == 0 && offsetof(FastSmem, cs) % 16 == 0 && offsetof(FastSmem, list) % 16 == 0, "16-byte accesses");
static_assert(kFItems == 8 && kFCap == 8 * kFThreads && kFCap < 65536, "the bucket scan: two uint4 per thread, two 16-bit partial sums in one word");

__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

__device__ __forceinline__ uint64_t tile_key(const uint4* tile, uint32_t e) {
    const uint2 v = *reinterpret_cast<const uint2*>(&tile[e]);
    return (((uint64_t)v.y << 32) | v.x) ^ 0x8000000000000000ull;
}

template <bool kPerm, bool kFuse>
__global__ void __launch_bounds__(kFThreads, 2) merge_fast_kernel(LevelDev lv, LevelDev nx, int has_next,
                                                                  const uint4* __restrict__ in, uint4* __restrict__ out,
                                                                  const uint32_t* __restrict__ perm_in,
                                                                  uint32_t* __restrict__ perm_out, int check_runs,
                                                                  FuseL1 fz, int32_t* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FastSmem& sm = *reinterpret_cast<FastSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31u;
    if (tid == 0) mbar_init(&sm.mbar, 1);
    {   // buckets and piece-start bitmap cleared while the tile's description is on its way
        uint4* z = reinterpret_cast<uint4*>(sm.cs);
#pragma unroll
        for (int i = 0; i < kFCap / 4 / kFThreads; ++i) z[tid + i * kFThreads] = make_uint4(0, 0, 0, 0);
        if (tid < (uint32_t)kFCap / 32) sm.pstart[tid] = 0;
    }
    const uint4 td = lv.tile_desc[blockIdx.x];
    const uint2 td2 = lv.tile_desc2[blockIdx.x];
    const uint32_t g = td.x, r0 = td.y, K = td.z, k = td.w;
    uint32_t my_a = 0, my_len = 0;
    if (tid < K) {
        const uint32_t* row0 = lv.splits + td2.x;
        const uint32_t a = row0[tid];
        uint32_t b = row0[K + tid];
        if (b < a) { b = a; atomicOr(status, TT_S_RUN_UNSORTED); }  // the split rows disagree: only with unsorted runs
        my_a = a;
        my_len = b - a;
        sm.cur[tid] = a;
    }
    const uint32_t out_base = lv.roff[r0] + lv.tile_base[td2.y];
    const uint32_t out_end = lv.roff[r0 + K];  // end of the group's output range
    const uint64_t T0 = lv.gT0[g], DT = lv.gDT[g];
    const uint32_t scale = lv.gScale[g];
    uint32_t total;
    const uint32_t my_s0 = block_scan1(my_len, sm.scan, &total);  // one barrier (orders the clearing above too)
    if (total == 0 || total > (uint32_t)kFCap || scale == 0u || out_base > out_end) {
        if (tid == 0) {
            if (total) lv.slow_list[atomicAdd(lv.slow_cnt, 1u)] = blockIdx.x;  // merge_slow_kernel sorts it (and emits)
            if (kFuse) lv.tile_open[blockIdx.x] = total ? 1 : 0;
        }
        if (!kFuse && has_next && total == 0) {  // an empty tile still owns the next level's boundaries of its key range
            const EmitRange er = emit_range(lv, nx, g, k);
            emit_next_splits(nx, er, lv.roff[r0], out_end, min(out_base, out_end), 0u, [](uint32_t) { return 0ull; });
        }
        return;
    }
    // fused L1 needs the window to end inside 32-bit offsets from Ta: lc + width < 2^32.  A wider window (far wider
    // than a tile anyway) leaves all L1 bits of the tile to l1_boundary_kernel's exact scans.
    const bool l1_here = kFuse && fz.lc < 0xFFFFFFFFull - (uint32_t)DT;
    if (tid < K) {
        sm.segstart[tid] = my_s0;
        if (my_len) atomicOr(&sm.pstart[my_s0 >> 5], 1u << (my_s0 & 31u));
    }
    if (tid == 0) {
        sm.segstart[K] = total;
        if (kFuse) lv.tile_open[blockIdx.x] = l1_here ? 0 : 1;
        mbar_expect_tx(&sm.mbar, total * 16u);
    }
    __syncthreads();
    {   // one TMA bulk copy per run piece; piece j is issued by lane j / 16 of warp j % 16 (spread over all warps)
        const uint32_t jj = lane * (uint32_t)(kFThreads / 32) + (tid >> 5);
        if (jj < K) {
            const uint32_t s0 = sm.segstart[jj], len = sm.segstart[jj + 1] - s0;
            if (len) bulk_g2s(&sm.tile[s0], in + sm.cur[jj], len * 16u, &sm.mbar);
        }
    }
    if (!kFuse && has_next && tid == kFThreads - 1) {  // while the tile is on its way; read after later barriers
        const EmitRange er = emit_range(lv, nx, g, k);
        sm.emit[0] = er.k_lo; sm.emit[1] = er.k_hi; sm.emit[2] = er.g1; sm.emit[3] = er.j1;
    }
    uint64_t Ta = T0 + (uint64_t)k * DT;
    if (Ta < T0) Ta = ~0ull;
    const uint32_t Ta_lo = (uint32_t)Ta, Ta_hi = (uint32_t)(Ta >> 32);
    const uint32_t width = (uint32_t)DT;  // kFCap < DT < 2^32 (scale != 0)
    mbar_wait(&sm.mbar, 0);
    // ---- histogram over kFCap fine buckets of the key offset d = key - Ta: bucket = hi32(d * scale); the top 20 bits
    // of lo32(d * scale) order two different offsets of one bucket (scale >= 2^12), the element id below them breaks
    // ties in input order
    uint32_t fb[kFItems];    // composite high part (20 bits) << 12 | bucket
    uint32_t slot[kFItems];  // arrival position in the bucket, later start << 16 | count of the bucket
    bool unsorted = false;
#pragma unroll
    for (int i = 0; i < kFItems; ++i) {
        const uint32_t e = tid + i * kFThreads;
        const bool in_tile = e < total;
        // key - Ta as (hi, d); a hit outside [0, width) can only come from unsorted runs (the splits assume sorted
        // runs): it is flagged, and its bucket is clamped so that the ranks stay a permutation of the tile
        const uint2 v = *reinterpret_cast<const uint2*>(&sm.tile[in_tile ? e : 0u]);
        const uint32_t d = v.x - Ta_lo;
        const uint32_t hi = (v.y ^ 0x80000000u) - Ta_hi - (v.x < Ta_lo ? 1u : 0u);
        bool bad = hi != 0u || d >= width;
        if (check_runs) {
            // order inside a run piece: the offset of the staged predecessor = the lane below; lane 0 reads it (if the
            // predecessor is outside [0, width) its own thread flags it, so comparing the low words is enough)
            uint32_t dp = __shfl_up_sync(0xffffffffu, d, 1);
            if (lane == 0u && e > 0u) dp = sm.tile[e - 1u].x - Ta_lo;
            const uint32_t ps = sm.pstart[(tid >> 5) + i * (kFThreads / 32)];  // one word per warp: a broadcast
            bad |= e > 0u && !((ps >> lane) & 1u) && dp > d;
        }
        unsorted |= in_tile && bad;
        const uint64_t pr = (uint64_t)d * scale;
        const uint32_t b = min((uint32_t)(pr >> 32), (uint32_t)kFCap - 1u);
        fb[i] = ((uint32_t)pr & 0xFFFFF000u) | b;
        slot[i] = 0;
        if (in_tile) slot[i] = atomicAdd(&sm.cs[b], 1u);
    }
    if (__syncthreads_or(unsorted) && tid == 0) atomicOr(status, TT_S_RUN_UNSORTED);
    // ---- exclusive scan of the bucket counts -> start << 16 | count.  Every thread takes four consecutive buckets of
    // the lower half and four of the upper half (two conflict-free 16-byte accesses; 8 consecutive buckets would be a
    // 32-byte stride = two-way bank conflicts); both partial sums (<= kFCap each) ride in one 32-bit scan.
    {
        uint4* c4 = reinterpret_cast<uint4*>(sm.cs);
        const uint4 w0 = c4[tid], w1 = c4[tid + kFThreads];
        uint32_t c[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
        const uint32_t sum_lo = c[0] + c[1] + c[2] + c[3], sum_hi = c[4] + c[5] + c[6] + c[7];
        uint32_t tot;
        const uint32_t ex2 = block_scan1(sum_lo | (sum_hi << 16), sm.scan + 16, &tot);
        uint32_t ex = ex2 & 0xFFFFu;
#pragma unroll
        for (int i = 0; i < 4; ++i) { const uint32_t t = c[i]; c[i] = (ex << 16) | t; ex += t; }
        ex = (tot & 0xFFFFu) + (ex2 >> 16);
#pragma unroll
        for (int i = 4; i < 8; ++i) { const uint32_t t = c[i]; c[i] = (ex << 16) | t; ex += t; }
        c4[tid] = make_uint4(c[0], c[1], c[2], c[3]);
        c4[tid + kFThreads] = make_uint4(c[4], c[5], c[6], c[7]);
    }
    __syncthreads();
    // ---- members of shared buckets go to the bucket's list
#pragma unroll
    for (int i = 0; i < kFItems; ++i) {
        const uint32_t e = tid + i * kFThreads;
        // (slots past the tile's end read bucket fb = garbage & 0xFFF: in range, and their cb/rank are never used)
        const uint32_t w = sm.cs[fb[i] & 0xFFFu];
        if (e < total && (w & 0xFFFFu) > 1u) sm.list[(w >> 16) + slot[i]] = (fb[i] & 0xFFFFF000u) | e;
        slot[i] = e < total ? w : 0u;
    }
    __syncthreads();
    // ---- rank = bucket start + members of the bucket that order before this hit.  Four members in a straight line (99 %
    // of the hits at a bucket load of 0.875), the loads of four hits issued together and predicated, no branch around
    // them: a branch per hit serialised its four dependent shared-memory reads; the loop is for the rare fuller buckets
    uint32_t rk[kFItems];
#pragma unroll
    for (int h = 0; h < kFItems; h += 4) {
        uint32_t o[4][4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t s0 = slot[h + u] >> 16, cb = slot[h + u] & 0xFFFFu;
            const uint32_t* const lp = sm.list + s0;
#pragma unroll
            for (int q = 0; q < 4; ++q) o[u][q] = (cb > 1u && cb > (uint32_t)q) ? lp[q] : 0xFFFFFFFFu;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t e = tid + (h + u) * kFThreads;
            const uint32_t s0 = slot[h + u] >> 16, cb = slot[h + u] & 0xFFFFu;
            const uint32_t c = (fb[h + u] & 0xFFFFF000u) | e;
            uint32_t r = s0 + (o[u][0] < c ? 1u : 0u) + (o[u][1] < c ? 1u : 0u) + (o[u][2] < c ? 1u : 0u) + (o[u][3] < c ? 1u : 0u);
            if (cb > 4u) {
                const uint32_t* const lp = sm.list + s0;
#pragma unroll 1
                for (uint32_t q = 4u; q < cb; ++q) r += lp[q] < c ? 1u : 0u;
            }
            rk[h + u] = r;
        }
    }
    // ---- in-place permutation: all records to registers, one barrier, all records to their ranks
    uint4 rec[kFItems];
#pragma unroll
    for (int i = 0; i < kFItems; ++i) {
        const uint32_t e = tid + i * kFThreads;
        rec[i] = e < total ? sm.tile[e] : make_uint4(0, 0, 0, 0);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kFItems; ++i) {
        const uint32_t e = tid + i * kFThreads;
        if (e < total) sm.tile[rk[i]] = rec[i];
    }
    if (kPerm) {
#pragma unroll
        for (int i = 0; i < kFItems; ++i) {
            const uint32_t e = tid + i * kFThreads;
            if (e < total) {
                uint32_t lo = 0, hi = K;  // piece j with segstart[j] <= e < segstart[j+1]
                while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (sm.segstart[mid] <= e) lo = mid; else hi = mid; }
                const uint32_t src = sm.cur[lo] + (e - sm.segstart[lo]);
                sm.list[rk[i]] = perm_in ? perm_in[src] : src;
            }
        }
    }
    fence_proxy_async();  // the generic-proxy writes of the tile before the bulk store reads it
    __syncthreads();
    const uint32_t n_store = min(total, out_end - out_base);
    if (tid == 0 && n_store) bulk_s2g(out + out_base, sm.tile, n_store * 16u);
    if (!kFuse && has_next) {  // the next level's split rows from the sorted tile (see emit_next_splits in tt_merge.cu)
        EmitRange er;
        er.k_lo = sm.emit[0]; er.k_hi = sm.emit[1]; er.g1 = sm.emit[2]; er.j1 = sm.emit[3];
        emit_next_splits(nx, er, lv.roff[r0], out_end, out_base, total, [&](uint32_t q) { return tile_key(sm.tile, q); });
    }
    if (kPerm) {
        for (uint32_t r = tid; r < n_store; r += kFThreads) perm_out[out_base + r] = sm.list[r];
        if (kFuse) __syncthreads();  // list is reused below
    }
    if (kFuse && l1_here) {
        // ---- L1 on the sorted tile.  cs[] <- time offset from Ta (exact in 32 bits: the tile spans < 2^32), list[] <-
        // floor << 16 | pmt, fl bytes <- Q.  Flag byte of tile hit r sits at byte sh + r, sh = the global address's
        // offset in its 16-byte group, so whole groups leave with 16-byte stores.
        uint8_t* const gfl = fz.flags + out_base;
        const uint32_t sh = (uint32_t)((uintptr_t)gfl & 15u);
        uint8_t* const fbytes = reinterpret_cast<uint8_t*>(sm.fl);
        const uint32_t lc32 = (uint32_t)fz.lc;  // lc < 2^32 - width here (else the tile is left to the exact scans)
#pragma unroll
        for (int i = 0; i < kFItems; ++i) {
            const uint32_t r = tid + i * kFThreads;
            if (r < total) {
                const uint4 v = sm.tile[r];
                sm.cs[r] = min(v.x - Ta_lo, width - 1u);  // (the clamp only acts on unsorted input: the scans below end at the sentinels)
                sm.list[r] = v.z;
                fbytes[sh + r] = (v.w & 0xFFFFu) >= fz.q_thresh ? (uint8_t)TT_Q : (uint8_t)0;
            }
        }
        if (tid < 4u) sm.cs[total + tid] = 0xFFFFFFFFu;  // sentinels: outside every window (offsets are < width)
        __syncthreads();
        // Every hit scans FORWARD over the hits inside its window and marks both partners of a same-floor / other-PMT
        // pair, so a pair is tested once.  Two loops, chosen per tile from its density (block-uniform):
        //   sparse (under ~1.5 hits per window: one tower): one hit per step, the time test first -- most hits leave at once;
        //   dense (many superimposed towers: ~9 hits ahead inside 20 ns): four hits per step, the floor filter first (a
        //   same-floor hit among them is rare), the time test only on a match and for the loop condition.
        if ((uint64_t)total * lc32 < (uint64_t)width + (width >> 1)) {
#pragma unroll 2
            for (int i = 0; i < kFItems; ++i) {
                const uint32_t e = tid + i * kFThreads;
                if (e >= total) break;
                const uint32_t ti = sm.cs[e], ki = sm.list[e];
                bool found = false;
                for (uint32_t j = e + 1; sm.cs[j] - ti <= lc32; ++j) {  // ends at the sentinel
                    const uint32_t x = sm.list[j] ^ ki;
                    if (x - 1u < 0xFFFFu) {  // same floor (high half equal), other pmt (low half differs)
                        found = true;
                        atomicOr(&sm.fl[(sh + j) >> 2], (uint32_t)TT_LC << (8u * ((sh + j) & 3u)));
                    }
                }
                if (found) atomicOr(&sm.fl[(sh + e) >> 2], (uint32_t)TT_LC << (8u * ((sh + e) & 3u)));
            }
        } else {
#pragma unroll 2
            for (int i = 0; i < kFItems; ++i) {
                const uint32_t e = tid + i * kFThreads;
                if (e >= total) break;
                const uint32_t ti = sm.cs[e], ki = sm.list[e];
                bool found = false;
                uint32_t j = e + 1;
                bool more;
                do {
                    const uint32_t x0 = sm.list[j] ^ ki, x1 = sm.list[j + 1] ^ ki, x2 = sm.list[j + 2] ^ ki, x3 = sm.list[j + 3] ^ ki;
                    more = sm.cs[j + 3] - ti <= lc32;
                    if ((x0 - 1u < 0xFFFFu) | (x1 - 1u < 0xFFFFu) | (x2 - 1u < 0xFFFFu) | (x3 - 1u < 0xFFFFu)) {
                        const uint32_t xs[4] = {x0, x1, x2, x3};
#pragma unroll
                        for (uint32_t q = 0; q < 4u; ++q) {
                            if (xs[q] - 1u < 0xFFFFu && sm.cs[j + q] - ti <= lc32) {
                                found = true;
                                atomicOr(&sm.fl[(sh + j + q) >> 2], (uint32_t)TT_LC << (8u * ((sh + j + q) & 3u)));
                            }
                        }
                    }
                    j += 4;
                } while (more);
                if (found) atomicOr(&sm.fl[(sh + e) >> 2], (uint32_t)TT_LC << (8u * ((sh + e) & 3u)));
            }
        }
        __syncthreads();
        // flags out: L1 = Q | LC
        const uint32_t nvec = (sh + n_store + 15u) >> 4;
        for (uint32_t q = tid; q < nvec; q += kFThreads) {
            uint4 v = reinterpret_cast<const uint4*>(sm.fl)[q];
            uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) w[u] |= ((w[u] | (w[u] >> 1)) & 0x01010101u) << 2;
            const uint32_t b0 = 16u * q;  // smem byte of the group; global byte = gfl - sh + b0
            if (b0 >= sh && b0 + 16u <= sh + n_store) {
                *reinterpret_cast<uint4*>(gfl - sh + b0) = make_uint4(w[0], w[1], w[2], w[3]);
            } else {
                for (uint32_t b8 = 0; b8 < 16u; ++b8) {
                    const uint32_t sb = b0 + b8;
                    if (sb >= sh && sb < sh + n_store) gfl[sb - sh] = (uint8_t)(w[b8 >> 2] >> (8u * (b8 & 3u)));
                }
            }
        }
    }
    if (tid == 0 && n_store) bulk_wait_read();  // the bulk store has read the tile: shared memory may go
}
