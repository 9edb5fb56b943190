// tt_merge.cu -- time sort of P concatenated, individually time-ordered runs (the per-PMT streams:
// PAPER.md:23 "merges together the 16 PMT data streams", "our data ... is time-ordered
// for single PMT"; north_star: "a merge of the per-PMT time-ordered streams").
//
// One pass per level: the runs of a group (<= fan-in F consecutive runs of one segment) are cut at
// uniform time boundaries into tiles of ~3.5 k hits (binary search of every run at every boundary),
// one CTA stages the <= F short run pieces of its tile in shared memory (run-major = input order),
// ranks them with a counting sort on fine time buckets (shared-memory atomics for the histogram,
// exact (time, input order) comparison inside a bucket, so the result is the stable order), and
// writes the tile with coalesced 16-byte stores.  P <= 512 runs per segment: one level (32 B/hit of
// HBM traffic).  More runs (cfg4: 8400): ceil(log_512 P) levels with fan-in ceil(P^(1/levels)).
//
// The plan (groups, tile counts, split tables) is computed on the device from the offsets, so the
// call stays asynchronous and allocation-free; the host mirrors the same integer arithmetic only to
// size grids and the workspace.
//
// Robustness: a tile whose pieces hold more than kCap hits (non-uniform density, massive ties) is
// swept in time order in chunks of <= kCap hits found by bisection on the key; a single timestamp
// with more than kCap hits is emitted as the run-major concatenation (which is the stable order).
#include <algorithm>
#include <vector>

#include <cstring>

#include "tt_merge.cuh"

namespace tt {

constexpr int kMThreads = 512;
constexpr int kCap = 4096;                    // hits staged per chunk
constexpr int kMItems = kCap / kMThreads;     // 8
constexpr uint32_t kTileTarget = 3584;        // expected hits per tile (0.875 kCap)
constexpr int kMaxFan = 512;                  // runs per group
constexpr uint32_t kInterpFan = 192;
constexpr int kFastCap = 4096;                // = kFCap of tt_merge_fast.cuh (checked there)          // from this fan-in on the partition search interpolates over the whole run first

__host__ __device__ inline uint32_t tiles_for(uint32_t n_g) { return (n_g + kTileTarget - 1) / kTileTarget; }

__device__ __forceinline__ uint64_t key_at(const uint4* __restrict__ hits, uint32_t i) {
    return key_of(hit_time(__ldg(hits + i)));
}

// ---- plan step 1: groups.  Segment s owns the runs [lb(roff, seg[s]), lb(roff, seg[s+1])) and is cut into
// consecutive groups of F runs.  One block; loops over segments with a running carry.
__device__ __forceinline__ void merge_groups(const LevelDev& lv, const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                             uint32_t* sm) {
    uint32_t carry = 0;
    for (uint32_t base = 0; base < n_seg; base += 1024) {
        const uint32_t s = base + threadIdx.x;
        uint32_t r0 = 0, r1 = 0, ng = 0;
        if (s < n_seg) {
            const uint32_t a = seg_off[s], b = seg_off[s + 1];
            uint32_t lo = 0, hi = lv.R;  // first run index with roff[r] >= a
            while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (lv.roff[mid] < a) lo = mid + 1; else hi = mid; }
            r0 = lo;
            lo = r0; hi = lv.R;
            if (s + 1 == n_seg) r1 = lv.R;
            else { while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (lv.roff[mid] < b) lo = mid + 1; else hi = mid; } r1 = lo; }
            ng = (r1 - r0 + lv.F - 1) / lv.F;
        }
        uint32_t total;
        const uint32_t ex = block_exclusive_scan(ng, sm, &total);
        for (uint32_t q = 0; q < ng; ++q) lv.gfirst[carry + ex + q] = r0 + q * lv.F;
        carry += total;
    }
    if (threadIdx.x == 0) lv.gfirst[carry] = lv.R;  // carry == G
}

// ---- plan step 2: per group: hit count, tile count, key range, tile width; prefixes.  One block,
// one warp per group (lanes over the group's runs).
// run_kmin / run_kmax (nullable): the key range of every run when the runs are the previous level's groups whose hits
// are not written yet (the previous level's tile kernel emits this level's splits, see emit_next_splits)
__global__ void __launch_bounds__(1024) merge_plan_kernel(LevelDev lv, const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                          const uint4* __restrict__ hits, uint32_t n,
                                                          const uint64_t* __restrict__ run_kmin,
                                                          const uint64_t* __restrict__ run_kmax) {
    __shared__ uint32_t sm[33];
    merge_groups(lv, seg_off, n_seg, sm);
    __syncthreads();  // gfirst[] (global, written by this block) is visible to all its threads
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // pass A: per-group ranges (warp per group; a lane takes four runs at a time so that their loads overlap)
    for (uint32_t g = warp; g < lv.G; g += 32) {
        const uint32_t r0 = lv.gfirst[g], r1 = lv.gfirst[g + 1];
        uint64_t kmin = ~0ull, kmax = 0;
        for (uint32_t rb = r0; rb < r1; rb += 128) {
            uint32_t a[4], b[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t r = rb + lane + 32u * j;
                a[j] = 0; b[j] = 0;
                if (r < r1) { a[j] = lv.roff[r]; b[j] = lv.roff[r + 1]; lv.run_group[r] = g; }
            }
            uint64_t k0[4], k1[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t r = rb + lane + 32u * j;
                k0[j] = ~0ull; k1[j] = 0;
                if (b[j] > a[j]) {
                    k0[j] = run_kmin ? run_kmin[r] : key_at(hits, a[j]);
                    k1[j] = run_kmax ? run_kmax[r] : key_at(hits, b[j] - 1);
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                kmin = k0[j] < kmin ? k0[j] : kmin;
                kmax = k1[j] > kmax ? k1[j] : kmax;
            }
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            const uint64_t o0 = __shfl_xor_sync(0xffffffffu, kmin, d), o1 = __shfl_xor_sync(0xffffffffu, kmax, d);
            kmin = o0 < kmin ? o0 : kmin;
            kmax = o1 > kmax ? o1 : kmax;
        }
        if (lane == 0) {
            const uint32_t n_g = lv.roff[r1] - lv.roff[r0];
            const uint32_t nt = tiles_for(n_g);
            lv.gT0[g] = kmin;
            lv.gKmax[g] = kmax;
            uint64_t dt = nt ? (kmax >= kmin ? (kmax - kmin) / nt + 1 : 1) : 1;
            if (dt == 0) dt = ~0ull;  // one tile over the whole key range, 2^64 - 1: the + 1 wrapped
            lv.gDT[g] = dt;
            // the fast tile kernel's bucket map: bucket = hi32((key - Ta) * scale) < kFastCap for key - Ta < dt
            lv.gScale[g] = (dt > (uint64_t)kFastCap && dt <= 0xFFFFFFFFull) ? (uint32_t)(((uint64_t)kFastCap << 32) / dt) : 0u;
            lv.roff_next[g] = lv.roff[r0];
        }
    }
    if (threadIdx.x == 0) lv.roff_next[lv.G] = n;
    __syncthreads();
    // pass B: prefixes of tiles and split entries
    uint32_t carry_t = 0, carry_s = 0;
    for (uint32_t base = 0; base < lv.G; base += 1024) {
        const uint32_t g = base + threadIdx.x;
        uint32_t nt = 0, ns = 0;
        if (g < lv.G) {
            const uint32_t r0 = lv.gfirst[g], r1 = lv.gfirst[g + 1];
            nt = tiles_for(lv.roff[r1] - lv.roff[r0]);
            ns = nt ? (nt + 1) * (r1 - r0) : 0;
        }
        uint32_t tt_, ts_;
        const uint32_t et = block_exclusive_scan(nt, sm, &tt_);
        const uint32_t es = block_exclusive_scan(ns, sm, &ts_);
        if (g < lv.G) { lv.tbase[g] = carry_t + et; lv.sbase[g] = carry_s + es; }
        carry_t += tt_;
        carry_s += ts_;
    }
    if (threadIdx.x == 0) { lv.tbase[lv.G] = carry_t; lv.sbase[lv.G] = carry_s; }
}

// ---- plan step 3: split table.  Entry (g, k, j): first index of run j of group g with key >= T0 + k*DT
// (k = 0: run start; k = tiles: run end).
template <bool kInterp>  // kInterp: many runs per group (host: fan-in >= kInterpFan), see the two branches below
__global__ void __launch_bounds__(256, 8) merge_partition_kernel(LevelDev lv, const uint4* __restrict__ hits,
                                                                 uint32_t total) {
    const uint32_t id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    uint32_t lo = 0, hi = lv.G;  // group with sbase[g] <= id < sbase[g+1]
    while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (lv.sbase[mid] <= id) lo = mid; else hi = mid; }
    const uint32_t g = lo;
    const uint32_t r0 = lv.gfirst[g], K = lv.gfirst[g + 1] - r0;
    const uint32_t local = id - lv.sbase[g];
    const uint32_t nt = lv.tbase[g + 1] - lv.tbase[g];
    // consecutive threads take consecutive boundaries k of ONE run j: their searches share the upper levels
    // and end in neighbouring cache lines (the table itself stays [k][j], as the tile kernel reads it)
    const uint32_t j = local / (nt + 1), k = local - j * (nt + 1);
    uint32_t a = lv.roff[r0 + j], b = lv.roff[r0 + j + 1];
    uint32_t res;
    if (k == 0) res = a;
    else if (k >= nt) res = b;
    else {
        const uint64_t T0 = lv.gT0[g], DT = lv.gDT[g];
        const uint64_t add = (uint64_t)k * DT;  // k < 2^20, DT <= 2^64 / nt: no overflow of the product
        const uint64_t T = T0 + add < T0 ? ~0ull : T0 + add;
        // Down to a bracket of <= 128 hits (below), then ONE interpolated probe between the last keys seen below and
        // above T and a short gallop: the bottom of the search touches 1-2 sectors of DRAM instead of ~5.  Exact for
        // any data (only comparisons decide); the interpolations just pick the probes.
        uint64_t klo = 0, khi = 0;  // key[a - 1] < T and key[b] >= T once seen
        bool have_lo = false, have_hi = false;
        if (!kInterp) {
            // few runs per group: consecutive boundaries of a run lie ~kTileTarget / K hits (several cache lines)
            // apart, so what pays is that the threads of a warp SHARE the upper probes of a plain bisection
            // (measured on cfg3 / cfg4, K = 84 / 92: 0.10 / 0.15 ms against 0.13 / 0.18 ms for the branch below)
            while (b - a > 128u) {
                const uint32_t mid = a + ((b - a) >> 1);
                const uint64_t km = key_at(hits, mid);
                if (km < T) { a = mid + 1; klo = km; have_lo = true; } else { b = mid; khi = km; have_hi = true; }
            }
        } else if (b - a > 128u) {
            // many runs per group (cfg2: 420): neighbouring boundaries end in the same cache lines anyway, and the
            // runs are near-uniform in time (Poisson streams): interpolate over the WHOLE run first -- the two end
            // keys are shared by every boundary of the run -- then gallop with a step of the order of the expected
            // error (sqrt of the run length) to bracket the answer (cfg2: 0.118 -> 0.079 ms).  Only comparisons
            // decide, so any data gives the exact lower bound.
            const uint64_t k0 = key_at(hits, a), k1 = key_at(hits, b - 1);
            if (T <= k0) b = a;
            else if (T > k1) a = b;
            else {
                uint32_t L = a, R = b - 1;  // key[L] < T <= key[R]
                uint64_t kL = k0, kR = k1;
                uint32_t step = (uint32_t)(sqrtf((float)(R - L)) * 0.25f);
                step = step < 16u ? 16u : step;
                if (R - L > 1u) {
                    const float frac = (float)(T - kL) / (float)(kR - kL);  // in (0, 1]
                    uint32_t q = L + (uint32_t)(frac * (float)(R - L));
                    q = q <= L ? L + 1u : (q >= R ? R - 1u : q);
                    const uint64_t kq = key_at(hits, q);
                    if (kq < T) {
                        L = q; kL = kq;
                        while (R - L > step) {
                            const uint32_t u = L + step;
                            const uint64_t ku = key_at(hits, u);
                            if (ku < T) { L = u; kL = ku; step <<= 1; } else { R = u; kR = ku; break; }
                        }
                    } else {
                        R = q; kR = kq;
                        while (R - L > step) {
                            const uint32_t u = R - step;
                            const uint64_t ku = key_at(hits, u);
                            if (ku >= T) { R = u; kR = ku; step <<= 1; } else { L = u; kL = ku; break; }
                        }
                    }
                }
                while (R - L > 128u) {
                    const uint32_t mid = L + ((R - L) >> 1);
                    const uint64_t km = key_at(hits, mid);
                    if (km < T) { L = mid; kL = km; } else { R = mid; kR = km; }
                }
                a = L + 1u; b = R; klo = kL; khi = kR; have_lo = true; have_hi = true;
            }
        }
        if (have_lo && have_hi && b > a) {
            // keys rise from klo at a - 1 to khi at b: first guess for the first index with key >= T
            const float frac = (float)(T - klo) / (float)(khi - klo);  // in (0, 1]
            uint32_t p = a + (uint32_t)(frac * (float)(b - a + 1));
            p = p > a ? p - 1u : a;
            if (p >= b) p = b - 1u;
            uint32_t step = 2;
            if (key_at(hits, p) < T) {  // answer in (p, b]
                a = p + 1u;
                while (a < b) {
                    const uint32_t q = b - a > step ? a + step - 1u : b - 1u;
                    if (key_at(hits, q) < T) { a = q + 1u; step <<= 1; } else { b = q; break; }
                }
            } else {                     // answer in [a, p]
                b = p;
                while (a < b) {
                    const uint32_t q = b - a > step ? b - step : a;
                    if (key_at(hits, q) >= T) { b = q; step <<= 1; } else { a = q + 1u; break; }
                }
            }
        }
        while (a < b) { const uint32_t mid = a + ((b - a) >> 1); if (key_at(hits, mid) < T) a = mid + 1; else b = mid; }
        res = a;
    }
    lv.splits[lv.sbase[g] + (size_t)k * K + j] = res;
    if (res != lv.roff[r0 + j]) atomicAdd(&lv.tile_base[lv.tbase[g] + g + k], res - lv.roff[r0 + j]);
    if (j == 0 && k < nt) {
        lv.tile_desc[lv.tbase[g] + k] = make_uint4(g, r0, K, k);
        lv.tile_desc2[lv.tbase[g] + k] = make_uint2(lv.sbase[g] + k * K, lv.tbase[g] + g + k);
    }
}

// ---- the next level's split table without a partition pass -----------------------------------------------
// A merge level's tile kernel has every sorted tile in shared memory (or has just written it), and the next level's
// runs ARE this level's groups: the position of a next-level boundary T1 inside run j1 is the tile's output base plus a
// lower bound inside the one tile whose key range holds T1.  So the tile kernels of level l write level l + 1's
// split rows and tile-base sums themselves (a few dozen binary searches in shared memory per tile) and the
// partition kernel -- 0.16 ms and 0.6 GB of DRAM probes on the 100-tower config -- runs for level 0 only.
// merge_init_next_kernel writes what no tile writes: row 0 (run starts), the rows of empty runs, the tile descriptors.
__global__ void __launch_bounds__(256, 8) merge_init_next_kernel(LevelDev lv, uint32_t total) {
    const uint32_t id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    uint32_t lo = 0, hi = lv.G;  // group with sbase[g] <= id < sbase[g+1]
    while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (lv.sbase[mid] <= id) lo = mid; else hi = mid; }
    const uint32_t g = lo;
    const uint32_t r0 = lv.gfirst[g], K = lv.gfirst[g + 1] - r0;
    const uint32_t local = id - lv.sbase[g];
    const uint32_t nt = lv.tbase[g + 1] - lv.tbase[g];
    const uint32_t j = local / (nt + 1), k = local - j * (nt + 1);
    lv.splits[lv.sbase[g] + (size_t)k * K + j] = k == 0 ? lv.roff[r0 + j] : lv.roff[r0 + j + 1];
    if (j == 0 && k < nt) {
        lv.tile_desc[lv.tbase[g] + k] = make_uint4(g, r0, K, k);
        lv.tile_desc2[lv.tbase[g] + k] = make_uint2(lv.sbase[g] + k * K, lv.tbase[g] + g + k);
    }
}

__device__ __forceinline__ uint64_t sat_boundary(uint64_t T0, uint64_t k, uint64_t DT) {
    const uint64_t t = T0 + k * DT;  // k < 2^20, DT <= 2^64 / tiles: the product does not overflow
    return t < T0 ? ~0ull : t;
}

// Tile k (of nt) of group g of level lv holds the keys in [T_k, T_k+1) (T_0 = -inf, T_nt = +inf) and owns the next
// level's boundaries k1 = 1 .. nt1 (T1(nt1) = +inf: the run end) whose T1 lies in that range: [k_lo, k_hi).  ONE
// thread computes the range (two 64-bit divisions) -- emit_range -- and all threads then place their boundaries --
// emit_next_splits.
struct EmitRange {
    uint32_t k_lo, k_hi;  // boundaries [k_lo, k_hi) of next-level group g1
    uint32_t g1, j1;      // next-level group and this group's run index in it
};

__device__ __forceinline__ EmitRange emit_range(const LevelDev& lv, const LevelDev& nx, uint32_t g, uint32_t k) {
    EmitRange r;
    r.g1 = nx.run_group[g];
    r.j1 = g - nx.gfirst[r.g1];
    const uint32_t nt1 = nx.tbase[r.g1 + 1] - nx.tbase[r.g1];
    const uint32_t nt = lv.tbase[g + 1] - lv.tbase[g];
    r.k_lo = 1; r.k_hi = 0;
    if (nt1 == 0) return r;
    const uint64_t T0 = lv.gT0[g], DT = lv.gDT[g], T01 = nx.gT0[r.g1], DT1 = nx.gDT[r.g1];
    // first boundary index k1 >= 1 with T1(k1) >= T, capped at nt1 (T1(nt1) = +inf)
    auto first_at = [&](uint64_t T) -> uint32_t {
        if (T <= T01) return 1u;
        const uint64_t q = (T - T01 - 1ull) / DT1 + 1ull;
        return q < (uint64_t)nt1 ? (uint32_t)q : nt1;
    };
    r.k_lo = k == 0 ? 1u : first_at(sat_boundary(T0, k, DT));
    r.k_hi = k + 1 >= nt ? nt1 + 1u : first_at(sat_boundary(T0, k + 1, DT));
    return r;
}

// The tile's c sorted hits start at output index b0, key_at(i) is the key of the i-th; [gs, ge) is the group's output
// range.  Called by all threads of the block with the same (block-uniform) range.
template <class KeyAt>
__device__ __forceinline__ void emit_next_splits(const LevelDev& nx, const EmitRange& r, uint32_t gs, uint32_t ge,
                                                 uint32_t b0, uint32_t c, KeyAt key_at) {
    if (r.k_lo >= r.k_hi) return;
    const uint32_t g1 = r.g1;
    const uint32_t K1 = nx.gfirst[g1 + 1] - nx.gfirst[g1];
    const uint32_t nt1 = nx.tbase[g1 + 1] - nx.tbase[g1];
    const uint64_t T01 = nx.gT0[g1], DT1 = nx.gDT[g1];
    uint32_t* const srow = nx.splits + nx.sbase[g1] + r.j1;
    uint32_t* const tb = nx.tile_base + nx.tbase[g1] + g1;
    for (uint32_t k1 = r.k_lo + threadIdx.x; k1 < r.k_hi; k1 += blockDim.x) {
        uint32_t pos = ge;
        if (k1 < nt1) {
            const uint64_t T = sat_boundary(T01, k1, DT1);
            uint32_t a = 0, b = c;
            while (a < b) { const uint32_t mid = a + ((b - a) >> 1); if (key_at(mid) < T) a = mid + 1; else b = mid; }
            pos = b0 + a;
            pos = pos < gs ? gs : (pos > ge ? ge : pos);  // (only unsorted runs can push it outside)
        }
        srow[(size_t)k1 * K1] = pos;
        if (pos != gs) atomicAdd(tb + k1, pos - gs);
    }
}

// ---- the tile kernel ---------------------------------------------------------------------------------
struct MergeSmem {
    uint4 tile[kCap];             // staged records, run-major (filled by TMA bulk copies)   64 KB
    uint32_t cs[kCap];            // 32-bit-key path: per bucket start << 16 | count, later inv[] (u16)      16 KB
                                  // wide-key path:   packed 16-bit counters (8 KB) + inv[] (u16, 8 KB)
    uint32_t list[kCap];          // 32-bit-key path: bucket member composites; wide-key path: member ids (u16)  16 KB
    uint32_t segstart[kMaxFan + 1];  // tile-local start of every run piece
    uint32_t cur[kMaxFan];        // absolute index of the next unprocessed hit of every run
    uint32_t end[kMaxFan];        // absolute end of every run piece of this tile
    uint32_t mid[kMaxFan];        // scratch: chunk ends (overflow sweep)
    uint32_t pstart[kCap / 32];   // bitmap of piece starts (run check)
    uint32_t scan[33];
    uint64_t red64[2 * (kMThreads / 32)];
    uint64_t mbar;                // TMA completion barrier
};
static_assert(2 * (sizeof(MergeSmem) + 1024) <= 233472, "two CTAs per SM");

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D TMA bulk copy global -> shared (16-byte granules), completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ uint32_t block_sum(uint32_t v, uint32_t* sm) {
    uint32_t total;
    block_exclusive_scan(v, sm, &total);
    return total;
}

__device__ __forceinline__ uint64_t tile_key(const MergeSmem& sm, uint32_t e) {
    const uint2 v = *reinterpret_cast<const uint2*>(&sm.tile[e]);
    return (((uint64_t)v.y << 32) | v.x) ^ 0x8000000000000000ull;
}
__device__ __forceinline__ uint32_t bucket_start(const MergeSmem& sm, uint32_t b) {
    return (sm.cs[b >> 1] >> ((b & 1) * 16)) & 0xFFFFu;
}

// block-wide exclusive scan with ONE barrier (blockDim.x = kMThreads): warp scans, the warp totals through 16 words of
// shared memory, and every warp scans those itself.  buf must not be rewritten before a later barrier.
__device__ __forceinline__ uint32_t block_scan1(uint32_t v, uint32_t* buf, uint32_t* total) {
    const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= (uint32_t)d) inc += o;
    }
    if (lane == 31) buf[w] = inc;
    __syncthreads();
    const uint32_t s = lane < (uint32_t)(kMThreads / 32) ? buf[lane] : 0u;
    uint32_t si = s;
#pragma unroll
    for (int d = 1; d < kMThreads / 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, si, d);
        if (lane >= (uint32_t)d) si += o;
    }
    *total = __shfl_sync(0xffffffffu, si, kMThreads / 32 - 1);
    return __shfl_sync(0xffffffffu, si - s, w) + inc - v;
}

// ---- 32-bit-key chunk sort (the common case: the chunk spans < 2^32 ps) -----------------------------------
// Same contract as sort_chunk below.  Counting sort on kCap fine buckets of the 32-bit key offset d = key - Ta:
// bucket = hi32(d * scale), and the top 20 bits of lo32(d * scale) order the keys inside a bucket exactly
// (scale >= 2^12, so two different offsets of one bucket differ there); with the 12-bit element id below them
// one 32-bit composite per hit gives the stable order by a single unsigned compare.
template <bool kPerm>
__device__ uint32_t sort_chunk32(MergeSmem& sm, const uint4* __restrict__ in, uint4* __restrict__ out, uint32_t K,
                                 const uint32_t* chunk_end, uint64_t Ta, uint32_t width, uint32_t out_base, uint32_t out_end,
                                 const uint32_t* __restrict__ perm_in, uint32_t* __restrict__ perm_out, bool check_runs,
                                 const uint32_t* __restrict__ run_begin, const uint64_t* prev_pre,
                                 int32_t* __restrict__ status, uint32_t& phase, bool cs_zeroed) {
    const uint32_t tid = threadIdx.x;
    uint32_t my_len = tid < K ? chunk_end[tid] - sm.cur[tid] : 0u;
    uint32_t total;
    const uint32_t my_s0 = block_scan1(my_len, sm.scan, &total);
    if (total > (uint32_t)kCap) {  // the split table and the pieces disagree: only with unsorted runs
        if (tid == 0) atomicOr(status, TT_S_RUN_UNSORTED);
        return total;
    }
    if (tid < K) sm.segstart[tid] = my_s0;
    if (tid == 0) {
        sm.segstart[K] = total;
        if (total) mbar_expect_tx(&sm.mbar, total * 16u);
    }
    fence_proxy_async();  // earlier generic-proxy accesses of the tile buffer are ordered before the bulk copies
    __syncthreads();
    const uint32_t count = total;
    // stage the pieces: one TMA bulk copy per run piece, all in flight at once.  Piece j is issued by lane j / 16
    // of warp j % 16: a warp issues its lanes' copies one after the other, so the K copies are spread over all
    // 16 warps instead of the first K / 32 (the others would wait for them at the next barrier).
    {
        const uint32_t jj = (tid & 31u) * (uint32_t)(kMThreads / 32) + (tid >> 5);
        if (jj < K) {
            const uint32_t s0 = sm.segstart[jj], len = sm.segstart[jj + 1] - s0;
            if (len) bulk_g2s(&sm.tile[s0], in + sm.cur[jj], len * 16u, &sm.mbar);
        }
    }
    // meanwhile: clear the buckets (unless the caller did, before an earlier barrier) and the piece-start bitmap,
    // fetch the run predecessors
    if (!cs_zeroed) {
        uint4* z = reinterpret_cast<uint4*>(sm.cs);
#pragma unroll
        for (int i = 0; i < kCap / 4 / kMThreads; ++i) z[tid + i * kMThreads] = make_uint4(0, 0, 0, 0);
    }
    if (check_runs && tid < (uint32_t)kCap / 32) sm.pstart[tid] = 0;
    uint64_t prev_key = 0;
    bool has_prev = false;
    if (check_runs && my_len && sm.cur[tid] > run_begin[tid]) { prev_key = prev_pre ? *prev_pre : key_at(in, sm.cur[tid] - 1); has_prev = true; }
    if (check_runs || !cs_zeroed) __syncthreads();
    if (check_runs && my_len) atomicOr(&sm.pstart[my_s0 >> 5], 1u << (my_s0 & 31));
    mbar_wait(&sm.mbar, phase);  // every thread waits itself: the staged data is visible to it
    phase ^= 1u;
    if (check_runs) __syncthreads();  // the piece-start bitmap
    const bool direct = width <= (uint32_t)kCap;
    const uint32_t scale = direct ? 0u : (uint32_t)(((uint64_t)kCap << 32) / width);
    const uint32_t Ta_lo = (uint32_t)Ta, Ta_hi = (uint32_t)(Ta >> 32);
    uint32_t fb[kMItems];    // composite high part (20 bits) << 12 | bucket
    uint32_t slot[kMItems];  // arrival position in the bucket, later start << 16 | count of the bucket
    bool unsorted = false;
    if (check_runs && has_prev && prev_key > tile_key(sm, my_s0)) unsorted = true;
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t e = tid + i * kMThreads;
        fb[i] = 0; slot[i] = 0;
        uint32_t d = 0;
        bool oob = false;
        uint2 kv = make_uint2(0u, 0u);
        if (e < count) {
            const uint2 v = *reinterpret_cast<const uint2*>(&sm.tile[e]);
            kv = v;
            const uint32_t hi = (v.y ^ 0x80000000u) - Ta_hi - (v.x < Ta_lo ? 1u : 0u);  // high word of key - Ta
            d = v.x - Ta_lo;
            oob = hi != 0u || d >= width;          // only with unsorted runs (the splits assume sorted runs)
            if (oob) d = (hi & 0x80000000u) ? 0u : width - 1u;
        }
        if (check_runs) {
            // order inside a run piece: the staged predecessor's key, compared as (high, low) words -- the same for
            // every lane (no shuffle, no lane-0 special case); piece starts are checked against prev_key above
            if (e < count && e > 0 && !((sm.pstart[e >> 5] >> (e & 31)) & 1u)) {
                const uint2 u = *reinterpret_cast<const uint2*>(&sm.tile[e - 1]);
                const uint32_t uy = u.y ^ 0x80000000u, vy = kv.y ^ 0x80000000u;
                if (uy > vy || (uy == vy && u.x > kv.x)) unsorted = true;
            }
            if (oob) unsorted = true;
        }
        if (e < count) {
            uint32_t b, fr;
            if (direct) { b = d; fr = 0; }
            else { const uint64_t pr = (uint64_t)d * scale; b = (uint32_t)(pr >> 32); fr = (uint32_t)pr & 0xFFFFF000u; }
            slot[i] = atomicAdd(&sm.cs[b], 1u) & 0xFFFFu;
            fb[i] = fr | b;
        }
    }
    if (check_runs) {
        if (__syncthreads_or(unsorted) && tid == 0) atomicOr(status, TT_S_RUN_UNSORTED);
    } else {
        __syncthreads();
    }
    // exclusive scan of the kCap bucket counts: 8 consecutive buckets per thread -> start << 16 | count
    {
        uint4* c4 = reinterpret_cast<uint4*>(sm.cs);
        uint4 w0 = c4[2 * tid], w1 = c4[2 * tid + 1];
        uint32_t c[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
        uint32_t sum = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) sum += c[i];
        uint32_t tot;
        uint32_t ex = block_scan1(sum, sm.scan + 16, &tot);
#pragma unroll
        for (int i = 0; i < 8; ++i) { const uint32_t t = c[i]; c[i] = (ex << 16) | t; ex += t; }
        c4[2 * tid] = make_uint4(c[0], c[1], c[2], c[3]);
        c4[2 * tid + 1] = make_uint4(c[4], c[5], c[6], c[7]);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t e = tid + i * kMThreads;
        if (e < count) {
            const uint32_t w = sm.cs[fb[i] & 0xFFFu];
            sm.list[(w >> 16) + slot[i]] = (fb[i] & 0xFFFFF000u) | e;
            slot[i] = w;
        }
    }
    __syncthreads();
    // exact rank inside the bucket; inv[] reuses the bucket array (its contents now live in slot[])
    uint16_t* const inv16 = reinterpret_cast<uint16_t*>(sm.cs);
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t e = tid + i * kMThreads;
        if (e < count) {
            const uint32_t s0 = slot[i] >> 16, cb = slot[i] & 0xFFFFu;
            uint32_t r = s0;
            if (cb > 1u) {
                const uint32_t c = (fb[i] & 0xFFFFF000u) | e;
                // four independent loads cover 99 % of the hits (bucket load 0.875: P(more than 4 in a bucket) = 1.2 %);
                // the tail loop runs for the rare larger buckets only
#pragma unroll
                for (uint32_t q = 0; q < 4u; ++q) {
                    const uint32_t o = q < cb ? sm.list[s0 + q] : 0xFFFFFFFFu;
                    r += o < c ? 1u : 0u;
                }
                for (uint32_t q = 4u; q < cb; ++q) r += sm.list[s0 + q] < c ? 1u : 0u;
            }
            inv16[r] = (uint16_t)e;  // cs[] was last read before the barrier above
        }
    }
    __syncthreads();
    // coalesced output
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t r = tid + i * kMThreads;
        if (r < count && out_base + r < out_end) {
            const uint32_t e = inv16[r];
            out[out_base + r] = sm.tile[e];
            if (kPerm) {
                uint32_t lo = 0, hi = K;  // piece j with segstart[j] <= e < segstart[j+1]
                while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (sm.segstart[mid] <= e) lo = mid; else hi = mid; }
                const uint32_t src = sm.cur[lo] + (e - sm.segstart[lo]);
                perm_out[out_base + r] = perm_in ? perm_in[src] : src;
            }
        }
    }
    return count;  // the caller puts a barrier before the shared memory is used again
}

// Sort the chunk [cur_j, chunk_end_j) over the runs j < K (<= kCap hits in total) and write it at out_base.
// Keys of the chunk lie in [Ta, Ta + width).  Returns the chunk size (uniform over the block).
// `phase` is the parity of the TMA barrier for this use (flips every call).
template <bool kPerm>
__device__ uint32_t sort_chunk(MergeSmem& sm, const uint4* __restrict__ in, uint4* __restrict__ out, uint32_t K,
                               const uint32_t* chunk_end, uint64_t Ta, uint64_t width, uint32_t out_base, uint32_t out_end,
                               const uint32_t* __restrict__ perm_in, uint32_t* __restrict__ perm_out, bool check_runs,
                               const uint32_t* __restrict__ run_begin, const uint64_t* prev_pre,
                               int32_t* __restrict__ status, uint32_t& phase) {
    const uint32_t tid = threadIdx.x;
    // tile-local piece starts
    uint32_t my_len = 0, my_s0 = 0;
    {
        my_len = tid < K ? chunk_end[tid] - sm.cur[tid] : 0u;
        uint32_t total;
        my_s0 = block_exclusive_scan(my_len, sm.scan, &total);
        if (total > (uint32_t)kCap) {  // the split table and the pieces disagree: only with unsorted runs
            if (tid == 0) atomicOr(status, TT_S_RUN_UNSORTED);
            return total;
        }
        if (tid < K) sm.segstart[tid] = my_s0;
        if (tid == 0) {
            sm.segstart[K] = total;
            if (total) mbar_expect_tx(&sm.mbar, total * 16u);
        }
    }
    fence_proxy_async();  // earlier generic-proxy accesses of the tile buffer are ordered before the bulk copies
    __syncthreads();
    const uint32_t count = sm.segstart[K];
    // stage the pieces: one TMA bulk copy per run piece, all in flight at once
    if (my_len) bulk_g2s(&sm.tile[my_s0], in + sm.cur[tid], my_len * 16u, &sm.mbar);
    // meanwhile: clear the counters and the piece-start bitmap, fetch the run predecessors
    uint16_t* const list16 = reinterpret_cast<uint16_t*>(sm.list);
    uint16_t* const inv16 = reinterpret_cast<uint16_t*>(sm.cs + kCap / 2);
    for (uint32_t b = tid; b < (uint32_t)kCap / 2; b += kMThreads) sm.cs[b] = 0;
    if (check_runs && tid < (uint32_t)kCap / 32) sm.pstart[tid] = 0;
    uint64_t prev_key = 0;
    bool has_prev = false;
    if (check_runs && my_len && sm.cur[tid] > run_begin[tid]) { prev_key = prev_pre ? *prev_pre : key_at(in, sm.cur[tid] - 1); has_prev = true; }
    __syncthreads();
    if (check_runs && my_len) atomicOr(&sm.pstart[my_s0 >> 5], 1u << (my_s0 & 31));
    mbar_wait(&sm.mbar, phase);
    phase ^= 1u;
    __syncthreads();
    // bucket function: monotone map of (key - Ta) in [0, width) onto [0, kCap)
    int pre = 0;
    while ((width >> pre) > 0xFFFFFFFFull) ++pre;
    const uint32_t wp = (uint32_t)(width >> pre);
    const bool direct = wp <= (uint32_t)kCap;
    const uint32_t scale = direct ? 0u : (uint32_t)(((uint64_t)kCap << 32) / wp);
    uint32_t bs[kMItems];  // bucket << 16 | slot
    bool unsorted = false;
    if (check_runs && has_prev && prev_key > tile_key(sm, my_s0)) unsorted = true;
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t e = tid + i * kMThreads;
        bs[i] = 0;
        if (e < count) {
            const uint64_t key = tile_key(sm, e);
            if (check_runs && e > 0 && !((sm.pstart[e >> 5] >> (e & 31)) & 1u) && tile_key(sm, e - 1) > key) unsorted = true;
            uint64_t dt = key - Ta;
            if (key < Ta) dt = 0;
            if (dt >= width) dt = width - 1;
            const uint32_t d = (uint32_t)(dt >> pre);
            uint32_t b = direct ? d : __umulhi(d, scale);
            if (b >= (uint32_t)kCap) b = kCap - 1;
            const uint32_t sh = (b & 1) * 16;
            const uint32_t old = atomicAdd(&sm.cs[b >> 1], 1u << sh);
            bs[i] = (b << 16) | ((old >> sh) & 0xFFFFu);
        }
    }
    if (check_runs) {
        if (__syncthreads_or(unsorted) && tid == 0) atomicOr(status, TT_S_RUN_UNSORTED);
    } else {
        __syncthreads();
    }
    // exclusive scan of the kCap packed counters: 8 consecutive counters (one 16-byte word) per thread
    {
        uint4 w = reinterpret_cast<uint4*>(sm.cs)[tid];
        uint32_t c[8] = {w.x & 0xFFFFu, w.x >> 16, w.y & 0xFFFFu, w.y >> 16, w.z & 0xFFFFu, w.z >> 16, w.w & 0xFFFFu, w.w >> 16};
        uint32_t s = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += c[i];
        uint32_t total;
        uint32_t ex = block_exclusive_scan(s, sm.scan, &total);
#pragma unroll
        for (int i = 0; i < 8; ++i) { const uint32_t t = c[i]; c[i] = ex; ex += t; }
        w.x = c[0] | (c[1] << 16); w.y = c[2] | (c[3] << 16); w.z = c[4] | (c[5] << 16); w.w = c[6] | (c[7] << 16);
        reinterpret_cast<uint4*>(sm.cs)[tid] = w;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t e = tid + i * kMThreads;
        if (e < count) list16[bucket_start(sm, bs[i] >> 16) + (bs[i] & 0xFFFFu)] = (uint16_t)e;
    }
    __syncthreads();
    // exact rank inside the bucket: order by (key, element id) = (time, input order)
#pragma unroll
    for (int i = 0; i < kMItems; ++i) {
        const uint32_t e = tid + i * kMThreads;
        if (e < count) {
            const uint32_t b = bs[i] >> 16;
            const uint32_t s0 = bucket_start(sm, b);
            const uint32_t s1 = b + 1 < (uint32_t)kCap ? bucket_start(sm, b + 1) : count;
            uint32_t r = s0;
            if (s1 - s0 > 1) {
                const uint64_t key = tile_key(sm, e);
                for (uint32_t m = s0; m < s1; ++m) {
                    const uint32_t o = list16[m];
                    const uint64_t ko = tile_key(sm, o);
                    r += (ko < key || (ko == key && o < e)) ? 1u : 0u;
                }
            }
            inv16[r] = (uint16_t)e;
        }
    }
    __syncthreads();
    // coalesced output
    for (uint32_t r = tid; r < count && out_base + r < out_end; r += kMThreads) {
        const uint32_t e = inv16[r];
        out[out_base + r] = sm.tile[e];
        if (kPerm) {
            uint32_t lo = 0, hi = K;  // piece j with segstart[j] <= e < segstart[j+1]
            while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (sm.segstart[mid] <= e) lo = mid; else hi = mid; }
            const uint32_t src = sm.cur[lo] + (e - sm.segstart[lo]);
            perm_out[out_base + r] = perm_in ? perm_in[src] : src;
        }
    }
    __syncthreads();
    return count;
}

// 32-bit keys when the chunk spans < 2^32 key units (block-uniform), else the general 64-bit path
template <bool kPerm>
__device__ __forceinline__ uint32_t sort_any(MergeSmem& sm, const uint4* __restrict__ in, uint4* __restrict__ out, uint32_t K,
                                             const uint32_t* chunk_end, uint64_t Ta, uint64_t width, uint32_t out_base,
                                             uint32_t out_end, const uint32_t* __restrict__ perm_in,
                                             uint32_t* __restrict__ perm_out, bool check_runs,
                                             const uint32_t* __restrict__ run_begin, const uint64_t* prev_pre,
                                             int32_t* __restrict__ status, uint32_t& phase, bool cs_zeroed = false) {
    if (width <= 0xFFFFFFFFull)
        return sort_chunk32<kPerm>(sm, in, out, K, chunk_end, Ta, (uint32_t)width, out_base, out_end, perm_in, perm_out,
                                   check_runs, run_begin, prev_pre, status, phase, cs_zeroed);
    return sort_chunk<kPerm>(sm, in, out, K, chunk_end, Ta, width, out_base, out_end, perm_in, perm_out, check_runs, run_begin,
                             prev_pre, status, phase);
}

// The general tile: any density, any key span, tie blocks (see the file header).  `tile` indexes tile_desc.
template <bool kPerm>
__device__ void merge_tile_general(MergeSmem& sm, const LevelDev& lv, uint32_t tile, const uint4* __restrict__ in,
                                   uint4* __restrict__ out, const uint32_t* __restrict__ perm_in,
                                   uint32_t* __restrict__ perm_out, int check_runs, int32_t* __restrict__ status,
                                   uint32_t& phase) {
    const uint32_t tid = threadIdx.x;
    {   // the bucket array is cleared while the tile's description is on its way; the barrier below orders it
        uint4* z = reinterpret_cast<uint4*>(sm.cs);
#pragma unroll
        for (int i = 0; i < kCap / 4 / kMThreads; ++i) z[tid + i * kMThreads] = make_uint4(0, 0, 0, 0);
    }
    const uint4 td = lv.tile_desc[tile];
    const uint2 td2 = lv.tile_desc2[tile];
    const uint32_t g = td.x, r0 = td.y, K = td.z, k = td.w;
    const uint32_t* row0 = lv.splits + td2.x;
    const uint32_t* row1 = row0 + K;
    const uint32_t* run_begin = lv.roff + r0;
    uint64_t prev0 = 0;  // key of the hit before the piece of run tid (run check), fetched early
    if (tid < K) {
        const uint32_t a = row0[tid];
        uint32_t b = row1[tid];
        if (b < a) b = a;  // only with unsorted runs (flagged by the run check)
        sm.cur[tid] = a;
        sm.end[tid] = b;
        if (check_runs && b > a && a > run_begin[tid]) prev0 = key_at(in, a - 1);
    }
    // hits of the group before this tile / in it: summed by the partition kernel
    const uint32_t tb0 = lv.tile_base[td2.y];
    uint32_t out_base = lv.roff[r0] + tb0;
    uint32_t remaining = lv.tile_base[td2.y + 1] - tb0;
    const uint32_t out_end = lv.roff[r0 + K];  // end of the group's output range
    const uint64_t T0 = lv.gT0[g], DT = lv.gDT[g];  // in flight together with the split rows, not after the barrier
    __syncthreads();
    uint64_t Ta = T0 + (uint64_t)k * DT;
    if (Ta < T0) Ta = ~0ull;
    if (remaining > (uint32_t)kCap) remaining = block_sum(tid < K ? sm.end[tid] - sm.cur[tid] : 0u, sm.scan);  // from the pieces
    if (remaining <= (uint32_t)kCap) {  // the common case: the whole tile in one chunk
        if (remaining)
            sort_any<kPerm>(sm, in, out, K, sm.end, Ta, DT, out_base, out_end, perm_in, perm_out, check_runs != 0, run_begin,
                            &prev0, status, phase, true);
        return;
    }
    // ---- overflow sweep: chunks of <= kCap hits in key order ------------------------------------------
    while (remaining) {
        // key range of what is left
        uint64_t kmin = ~0ull, kmax = 0;
        if (tid < K && sm.end[tid] > sm.cur[tid]) { kmin = key_at(in, sm.cur[tid]); kmax = key_at(in, sm.end[tid] - 1); }
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            const uint64_t o0 = __shfl_xor_sync(0xffffffffu, kmin, d), o1 = __shfl_xor_sync(0xffffffffu, kmax, d);
            kmin = o0 < kmin ? o0 : kmin;
            kmax = o1 > kmax ? o1 : kmax;
        }
        if ((tid & 31) == 0) { sm.red64[2 * (tid >> 5)] = kmin; sm.red64[2 * (tid >> 5) + 1] = kmax; }
        __syncthreads();
        kmin = ~0ull; kmax = 0;
        for (int w = 0; w < kMThreads / 32; ++w) {
            kmin = sm.red64[2 * w] < kmin ? sm.red64[2 * w] : kmin;
            kmax = sm.red64[2 * w + 1] > kmax ? sm.red64[2 * w + 1] : kmax;
        }
        __syncthreads();
        if (remaining <= (uint32_t)kCap) {
            const uint32_t c = sort_any<kPerm>(sm, in, out, K, sm.end, kmin, kmax - kmin + 1 ? kmax - kmin + 1 : ~0ull,
                                               out_base, out_end, perm_in, perm_out, check_runs != 0, run_begin, nullptr, status,
                                               phase);
            out_base += c;
            break;
        }
        // largest x in [kmin, kmax) with C(x) = #{key <= x} <= kCap; C(kmax) = remaining > kCap.
        // have_lo == false stands for x = kmin - 1 (C = 0).
        bool have_lo = false;
        uint64_t xlo = kmin, xhi = kmax;  // invariant: C(xlo) <= kCap (if have_lo) < C(xhi)
        while (true) {
            uint64_t xm;
            if (!have_lo) {
                if (xhi == kmin) break;  // even the single smallest key overflows: tie block
                xm = kmin + ((xhi - kmin) >> 1);
            } else {
                if (xhi - xlo <= 1) break;
                xm = xlo + ((xhi - xlo) >> 1);
            }
            uint32_t c = 0;
            if (tid < K) {
                uint32_t a = sm.cur[tid], b = sm.end[tid];
                while (a < b) { const uint32_t mid = a + ((b - a) >> 1); if (key_at(in, mid) <= xm) a = mid + 1; else b = mid; }
                sm.mid[tid] = a;
                c = a - sm.cur[tid];
            }
            const uint32_t C = block_sum(c, sm.scan);
            if (C <= (uint32_t)kCap) { have_lo = true; xlo = xm; } else xhi = xm;
        }
        // chunk end per run: keys <= xlo (or the tie block keys == kmin)
        const uint64_t xcut = have_lo ? xlo : kmin;
        uint32_t c = 0;
        if (tid < K) {
            uint32_t a = sm.cur[tid], b = sm.end[tid];
            while (a < b) { const uint32_t mid = a + ((b - a) >> 1); if (key_at(in, mid) <= xcut) a = mid + 1; else b = mid; }
            sm.mid[tid] = a;
            c = a - sm.cur[tid];
        }
        uint32_t total;
        const uint32_t ex = block_exclusive_scan(c, sm.scan, &total);
        if (have_lo && total) {
            sort_any<kPerm>(sm, in, out, K, sm.mid, kmin, xlo - kmin + 1, out_base, out_end, perm_in, perm_out, check_runs != 0,
                            run_begin, nullptr, status, phase);
            __syncthreads();
        } else {
            // tie block: every hit has key == kmin; the stable order is the run-major concatenation
            if (tid < K) sm.segstart[tid] = ex;
            if (tid == 0) sm.segstart[K] = total;
            __syncthreads();
            for (uint32_t e = tid; e < total; e += kMThreads) {
                uint32_t lo2 = 0, hi2 = K;
                while (hi2 - lo2 > 1) { const uint32_t mid = (lo2 + hi2) >> 1; if (sm.segstart[mid] <= e) lo2 = mid; else hi2 = mid; }
                const uint32_t src = sm.cur[lo2] + (e - sm.segstart[lo2]);
                if (out_base + e < out_end) {
                    out[out_base + e] = __ldg(in + src);
                    if (kPerm) perm_out[out_base + e] = perm_in ? perm_in[src] : src;
                }
            }
            __syncthreads();
        }
        if (tid < K) sm.cur[tid] = sm.mid[tid];
        out_base += total;
        remaining -= total;
        __syncthreads();
    }
}

// The tiles the fast kernel (tt_merge_fast.cuh) left over: a fixed grid walks the list.
template <bool kPerm>
__global__ void __launch_bounds__(kMThreads, 2) merge_slow_kernel(LevelDev lv, LevelDev nx, int has_next,
                                                                  const uint4* __restrict__ in, uint4* __restrict__ out,
                                                                  const uint32_t* __restrict__ perm_in,
                                                                  uint32_t* __restrict__ perm_out, int check_runs,
                                                                  int32_t* __restrict__ status) {
    const uint32_t n_slow = *lv.slow_cnt;
    if (blockIdx.x >= n_slow) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    MergeSmem& sm = *reinterpret_cast<MergeSmem*>(smem_raw);
    if (threadIdx.x == 0) mbar_init(&sm.mbar, 1);
    uint32_t phase = 0;
    for (uint32_t i = blockIdx.x; i < n_slow; i += gridDim.x) {
        const uint32_t tile = lv.slow_list[i];
        merge_tile_general<kPerm>(sm, lv, tile, in, out, perm_in, perm_out, check_runs, status, phase);
        __syncthreads();  // the tile is in global memory, visible to this block
        if (has_next) {
            const uint4 td = lv.tile_desc[tile];
            const uint2 td2 = lv.tile_desc2[tile];
            const uint32_t gs = lv.roff[td.y], ge = lv.roff[td.y + td.z];
            uint32_t b0 = gs + lv.tile_base[td2.y], b1 = gs + lv.tile_base[td2.y + 1];
            b0 = b0 > ge ? ge : b0;
            b1 = b1 > ge ? ge : (b1 < b0 ? b0 : b1);
            const uint4* o = out;
            const EmitRange er = emit_range(lv, nx, td.x, td.w);  // (every thread: the general path is rare)
            emit_next_splits(nx, er, gs, ge, b0, b1 - b0, [&](uint32_t q) { return key_of(hit_time(__ldcg(o + b0 + q))); });
        }
    }
}

#include "tt_merge_fast.cuh"
static_assert(kFCap == kFastCap, "plan and fast kernel agree on the bucket count");

// ---- host side: plan mirror -----------------------------------------------------------------------------
// Only counts: the host never needs the per-level offset arrays after sizing, so the plan of the last call is kept
// per host thread and reused while the offsets are unchanged (a hot call then allocates nothing).
struct LevelHost {
    uint32_t R, G, F, tiles, split_entries;
    uint32_t kmax;               // most runs in one group of this level
};

struct PlanCache {
    std::vector<uint32_t> seg, runs;  // the offsets the plan was made for
    uint32_t n = 0;
    bool valid = false;
    std::vector<LevelHost> levels;
    std::vector<uint32_t> roff, next;  // scratch of build_plan
};

static uint32_t lower_bound_u32(const std::vector<uint32_t>& v, uint32_t R, uint32_t x) {
    uint32_t lo = 0, hi = R;
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (v[mid] < x) lo = mid + 1; else hi = mid; }
    return lo;
}

static void build_plan(PlanCache& pc, uint32_t n, const uint32_t* h_seg, uint32_t n_seg, const uint32_t* h_runs,
                       uint32_t n_runs) {
    // largest number of runs in one segment decides the number of levels and the fan-in
    pc.roff.assign(h_runs, h_runs + n_runs + 1);
    uint32_t pmax = 1;
    for (uint32_t s = 0; s < n_seg; ++s) {
        const uint32_t r0 = lower_bound_u32(pc.roff, n_runs, h_seg[s]);
        const uint32_t r1 = s + 1 == n_seg ? n_runs : lower_bound_u32(pc.roff, n_runs, h_seg[s + 1]);
        if (r1 - r0 > pmax) pmax = r1 - r0;
    }
    uint32_t nlev = 1;
    for (uint64_t cap = kMaxFan; cap < pmax; cap *= kMaxFan) ++nlev;
    uint32_t F = kMaxFan;
    if (nlev > 1) {  // smallest F with F^nlev >= pmax
        F = 2;
        while (true) {
            uint64_t c = 1;
            for (uint32_t l = 0; l < nlev; ++l) c *= F;
            if (c >= pmax) break;
            ++F;
        }
    }
    pc.levels.clear();
    uint32_t R = n_runs;
    uint32_t pm = pmax;  // most runs of one segment at this level
    for (uint32_t l = 0; l < nlev; ++l) {
        LevelHost L;
        L.R = R; L.F = F; L.tiles = 0; L.split_entries = 0; L.G = 0;
        pc.next.clear();
        for (uint32_t s = 0; s < n_seg; ++s) {
            const uint32_t r0 = lower_bound_u32(pc.roff, R, h_seg[s]);
            const uint32_t r1 = s + 1 == n_seg ? R : lower_bound_u32(pc.roff, R, h_seg[s + 1]);
            for (uint32_t r = r0; r < r1; r += F) {
                const uint32_t re = r + F < r1 ? r + F : r1;
                const uint32_t nt = tiles_for(pc.roff[re] - pc.roff[r]);
                L.tiles += nt;
                L.split_entries += nt ? (nt + 1) * (re - r) : 0;
                pc.next.push_back(pc.roff[r]);
                ++L.G;
            }
        }
        pc.next.push_back(n);
        L.kmax = pm < F ? pm : F;
        pm = (pm + F - 1) / F;
        pc.levels.push_back(L);
        pc.roff.swap(pc.next);
        R = L.G;
    }
}

static const std::vector<LevelHost>& plan_for(uint32_t n, const uint32_t* h_seg, uint32_t n_seg, const uint32_t* h_runs,
                                              uint32_t n_runs) {
    thread_local PlanCache pc;
    if (pc.valid && pc.n == n && pc.seg.size() == (size_t)n_seg + 1 && pc.runs.size() == (size_t)n_runs + 1 &&
        std::memcmp(pc.seg.data(), h_seg, ((size_t)n_seg + 1) * 4) == 0 &&
        std::memcmp(pc.runs.data(), h_runs, ((size_t)n_runs + 1) * 4) == 0)
        return pc.levels;
    pc.valid = false;
    pc.seg.assign(h_seg, h_seg + n_seg + 1);
    pc.runs.assign(h_runs, h_runs + n_runs + 1);
    pc.n = n;
    build_plan(pc, n, h_seg, n_seg, h_runs, n_runs);
    pc.valid = true;
    return pc.levels;
}

constexpr int kMaxLevels = 4;  // 512^4 runs

struct MergeWs {
    LevelDev dev[kMaxLevels];
    uint4* tmp[2];
    uint32_t* ptmp[2];
};

static void carve(Arena& a, const std::vector<LevelHost>& levels, uint32_t n, bool perm, MergeWs& w) {
    for (size_t l = 0; l < levels.size(); ++l) {
        const LevelHost& L = levels[l];
        LevelDev& d = w.dev[l];
        d.R = L.R; d.G = L.G; d.F = L.F;
        d.gfirst = a.take<uint32_t>(L.G + 1);
        d.tbase = a.take<uint32_t>(L.G + 1);
        d.sbase = a.take<uint32_t>(L.G + 1);
        d.gT0 = a.take<uint64_t>(L.G + 1);
        d.gDT = a.take<uint64_t>(L.G + 1);
        d.gKmax = a.take<uint64_t>(L.G + 1);
        d.run_group = a.take<uint32_t>((size_t)L.R + 1);
        d.gScale = a.take<uint32_t>(L.G + 1);
        d.splits = a.take<uint32_t>((size_t)L.split_entries + 1);
        d.roff_next = a.take<uint32_t>(L.G + 1);
        d.tile_desc = a.take<uint4>((size_t)L.tiles + 1);
        d.tile_desc2 = a.take<uint2>((size_t)L.tiles + 1);
        d.tile_base = a.take<uint32_t>((size_t)L.tiles + L.G + 2);  // + the slow-tile counter: one memset clears both
        d.slow_cnt = d.tile_base ? d.tile_base + ((size_t)L.tiles + L.G + 1) : nullptr;
        d.slow_list = a.take<uint32_t>((size_t)L.tiles + 1);
        d.tile_open = a.take<uint8_t>((size_t)L.tiles + 1);
    }
    const size_t nlev = levels.size();
    w.tmp[0] = nlev > 1 ? a.take<uint4>(n) : nullptr;
    w.tmp[1] = nlev > 2 ? a.take<uint4>(n) : nullptr;
    w.ptmp[0] = (perm && nlev > 1) ? a.take<uint32_t>(n) : nullptr;
    w.ptmp[1] = (perm && nlev > 2) ? a.take<uint32_t>(n) : nullptr;
}

size_t merge_ws_bytes(uint32_t n, const uint32_t* h_seg, uint32_t n_seg, const uint32_t* h_runs, uint32_t n_runs) {
    const std::vector<LevelHost>& levels = plan_for(n, h_seg, n_seg, h_runs, n_runs);
    if (levels.size() > (size_t)kMaxLevels) return ~size_t(0);
    Arena a(nullptr);
    MergeWs w;
    carve(a, levels, n, true, w);
    return a.off;
}

static int merge_attrs() {
    TT_CUDA_OK(cudaFuncSetAttribute(merge_slow_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MergeSmem)));
    TT_CUDA_OK(cudaFuncSetAttribute(merge_slow_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MergeSmem)));
    TT_CUDA_OK(cudaFuncSetAttribute(merge_fast_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem)));
    TT_CUDA_OK(cudaFuncSetAttribute(merge_fast_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem)));
    TT_CUDA_OK(cudaFuncSetAttribute(merge_fast_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem)));
    TT_CUDA_OK(cudaFuncSetAttribute(merge_fast_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem)));
    return TT_OK;
}

int merge_sort_runs(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
                    const uint32_t* h_seg, uint32_t n_seg, const uint32_t* d_run_offsets, const uint32_t* h_runs,
                    uint32_t n_runs, void* d_ws, int32_t* d_status, cudaStream_t s, const FuseL1* fuse, MergeLast* last) {
    const std::vector<LevelHost>& levels = plan_for(n, h_seg, n_seg, h_runs, n_runs);
    const size_t nlev = levels.size();
    if (nlev > (size_t)kMaxLevels) return TT_E_INVAL;
    Arena a(d_ws);
    MergeWs w;
    carve(a, levels, n, true, w);
    int rc = once_per_device(kSlotMerge, merge_attrs);
    if (rc != TT_OK) return rc;
    const uint32_t slow_grid = 2u * (uint32_t)sm_count();
    const uint4* src = (const uint4*)d_in;
    const uint32_t* psrc = nullptr;
    FuseL1 none;
    none.flags = nullptr; none.lc = 0; none.q_thresh = 0;
    bool planned = false;  // this level's plan and split table were made by the previous level (emit_next_splits)
    for (size_t l = 0; l < nlev; ++l) {
        LevelDev& d = w.dev[l];
        d.roff = l == 0 ? d_run_offsets : w.dev[l - 1].roff_next;
        const bool is_last = l + 1 == nlev;
        const bool fused = is_last && fuse && fuse->flags;
        uint4* dst = is_last ? (uint4*)d_out : w.tmp[l & 1];
        uint32_t* pdst = d_perm ? (is_last ? d_perm : w.ptmp[l & 1]) : nullptr;
        if (!planned) {
            prof_mark(s, l == 0 ? "sort.merge_plan0" : "sort.merge_plan1");
            TT_K(merge_plan_kernel)<<<1, 1024, 0, s>>>(d, d_seg_offsets, n_seg, src, n, nullptr, nullptr);
            TT_CUDA_OK(cudaMemsetAsync(d.tile_base, 0, ((size_t)levels[l].tiles + levels[l].G + 2) * sizeof(uint32_t), s));
            if (levels[l].split_entries) {
                prof_mark(s, l == 0 ? "sort.merge_partition0" : "sort.merge_partition1");
                if (levels[l].kmax >= kInterpFan)
                    TT_K(merge_partition_kernel<true>)<<<div_up(levels[l].split_entries, 256), 256, 0, s>>>(d, src, levels[l].split_entries);
                else
                    TT_K(merge_partition_kernel<false>)<<<div_up(levels[l].split_entries, 256), 256, 0, s>>>(d, src, levels[l].split_entries);
            }
        }
        // the next level's plan, from this level's group key ranges, BEFORE this level's tiles run: they fill its split table
        const bool emit = !is_last && levels[l].tiles && levels[l + 1].split_entries;
        LevelDev nx = d;
        if (emit) {
            LevelDev& e = w.dev[l + 1];
            e.roff = d.roff_next;
            prof_mark(s, "sort.merge_plan1");
            TT_K(merge_plan_kernel)<<<1, 1024, 0, s>>>(e, d_seg_offsets, n_seg, nullptr, n, d.gT0, d.gKmax);
            TT_CUDA_OK(cudaMemsetAsync(e.tile_base, 0, ((size_t)levels[l + 1].tiles + levels[l + 1].G + 2) * sizeof(uint32_t), s));
            TT_K(merge_init_next_kernel)<<<div_up(levels[l + 1].split_entries, 256), 256, 0, s>>>(e, levels[l + 1].split_entries);
            nx = e;
        }
        planned = emit;
        if (levels[l].tiles) {
            prof_mark(s, l == 0 ? "sort.merge_tile0" : "sort.merge_tile1");
            const uint32_t nt = levels[l].tiles;
            const int chk = l == 0, hn = emit ? 1 : 0;
            if (d_perm) {
                if (fused) TT_K((merge_fast_kernel<true, true>))<<<nt, kFThreads, sizeof(FastSmem), s>>>(d, nx, hn, src, dst, psrc, pdst, chk, *fuse, d_status);
                else TT_K((merge_fast_kernel<true, false>))<<<nt, kFThreads, sizeof(FastSmem), s>>>(d, nx, hn, src, dst, psrc, pdst, chk, none, d_status);
                TT_K(merge_slow_kernel<true>)<<<slow_grid, kMThreads, sizeof(MergeSmem), s>>>(d, nx, hn, src, dst, psrc, pdst, chk, d_status);
            } else {
                if (fused) TT_K((merge_fast_kernel<false, true>))<<<nt, kFThreads, sizeof(FastSmem), s>>>(d, nx, hn, src, dst, nullptr, nullptr, chk, *fuse, d_status);
                else TT_K((merge_fast_kernel<false, false>))<<<nt, kFThreads, sizeof(FastSmem), s>>>(d, nx, hn, src, dst, nullptr, nullptr, chk, none, d_status);
                TT_K(merge_slow_kernel<false>)<<<slow_grid, kMThreads, sizeof(MergeSmem), s>>>(d, nx, hn, src, dst, nullptr, nullptr, chk, d_status);
            }
        }
        if (is_last && last) { last->lv = d; last->tiles = levels[l].tiles; }
        src = dst;
        psrc = pdst;
    }
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

}  // namespace tt
