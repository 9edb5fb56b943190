// tt_pairs.cu -- the paper's pair-coincidence seeds and its combined trigger.
//
//   PAPER.md:61  SC  "a coincidence between two hits occurred in two adjacent PMTs within 20 ns"
//   PAPER.md:62  FC  "a coincidence between two hits occurred in two PMTs in the same floor within 100 ns"
//   PAPER.md:63  AFC "... in two PMTs located at two consecutive floors within 250 ns"
//   PAPER.md:65, 73  "applying N7TW1000, and if it is satisfied, we apply [SC and AFC] or [FC and AFC]"
//   DESIGN.md readings R21 (adjacent = caller's table over the PMTs of one tower), R22 (the combination is
//   evaluated over the N hits of each firing level-0 window), R4 (inclusive windows), R5 (two different PMTs).
//
// pair_seeds_kernel: one CTA per tile of kPTile sorted hits, staged with kPHalo hits on both sides as (32-bit time
// relative to the first staged hit, floor << 16 | local pmt, tower).  Every staged hit scans FORWARD while
// t_j - t_i <= the largest window and ORs the rule bits into both partners, so each pair is tested once.  What the
// staged window cannot decide (a window reaching past the halo, >= 2^32 ps across the staged hits, segment ends) is
// finished by exact scans of global memory: the result is the plain definition for any input.
#include "tt_common.cuh"

namespace tt {

constexpr int kPThreads = 256;
constexpr int kPPer = 8;
constexpr int kPTile = kPThreads * kPPer;     // 2048
constexpr int kPHalo = 256;
constexpr int kPStage = kPTile + 2 * kPHalo;  // 2560
constexpr int kPPad = 64;                     // readable slack behind the staged arrays (speculative lockstep reads)
constexpr uint32_t kPAdjSmem = 128;           // adjacency table in shared memory up to 128 PMTs per tower (16 KB)

struct PairWin {
    uint64_t sc, fc, afc, wmax;
    uint64_t rcp;  // ceil(2^32 / pmts_per_tower)
};

// rule bits of the ordered pair (i, j), dt = |t_j - t_i|; a = floor << 16 | local pmt, tw = tower
template <typename DT, typename Adj>
__device__ __forceinline__ uint32_t pair_rules(uint32_t ai, uint32_t twi, uint32_t aj, uint32_t twj, DT dt, DT w_sc,
                                               DT w_fc, DT w_afc, uint32_t ppt, Adj adj) {
    const bool same_tower = twi == twj;
    if (same_tower && ((ai ^ aj) & 0xFFFFu) == 0u) return 0u;  // the same PMT: "two PMTs" (R5)
    uint32_t m = 0;
    const uint32_t fi = ai >> 16, fj = aj >> 16;
    if (dt <= w_fc && fi == fj) m |= TT_P_FC;
    if (same_tower) {
        if (dt <= w_afc && (fi + 1u == fj || fj + 1u == fi)) m |= TT_P_AFC;
        if (dt <= w_sc && adj((ai & 0xFFFFu) * ppt + (aj & 0xFFFFu))) m |= TT_P_SC;
    }
    return m;
}

// tower = pmt / ppt through the host's reciprocal rcp = ceil(2^32 / ppt): exact for pmt < 2^16 and ppt <= 2^16
// (the error pmt * (rcp - 2^32 / ppt) < 2^16 <= 2^32 / ppt never reaches the next integer)
__device__ __forceinline__ void split_pmt(uint32_t z, uint32_t ppt, uint64_t rcp, uint32_t& a, uint32_t& tw) {
    const uint32_t pmt = z & 0xFFFFu;
    tw = (uint32_t)(((uint64_t)pmt * rcp) >> 32);
    a = (z & 0xFFFF0000u) | (pmt - tw * ppt);
}

// exact rule bits of hit i from partners j < below and j >= above inside [a, b), by global memory
__device__ uint32_t pair_scan_global(const uint4* __restrict__ hits, int64_t t, uint32_t ai, uint32_t twi,
                                     uint32_t below, uint32_t above, uint32_t a, uint32_t b, const PairWin& w,
                                     uint32_t ppt, const uint8_t* __restrict__ adj) {
    uint32_t m = 0;
    auto ga = [&](uint32_t k) { return __ldg(adj + k) != 0; };
    for (uint32_t j = below; j > a;) {
        --j;
        const uint4 v = __ldg(hits + j);
        const uint64_t dt = udiff(t, hit_time(v));
        if (dt > w.wmax) break;
        uint32_t aj, twj;
        split_pmt(v.z, ppt, w.rcp, aj, twj);
        m |= pair_rules<uint64_t>(ai, twi, aj, twj, dt, w.sc, w.fc, w.afc, ppt, ga);
    }
    for (uint32_t j = above; j < b; ++j) {
        const uint4 v = __ldg(hits + j);
        const uint64_t dt = udiff(hit_time(v), t);
        if (dt > w.wmax) break;
        uint32_t aj, twj;
        split_pmt(v.z, ppt, w.rcp, aj, twj);
        m |= pair_rules<uint64_t>(ai, twi, aj, twj, dt, w.sc, w.fc, w.afc, ppt, ga);
    }
    return m;
}

struct PairSmem {
    uint32_t t[kPStage + kPPad];    // time relative to the first staged hit
    uint32_t a[kPStage + kPPad];    // floor << 16 | local pmt
    uint32_t tw[kPStage + kPPad];   // tower
    uint32_t f[kPTile / 4]; // rule bytes of the in-tile hits
};

__global__ void __launch_bounds__(kPThreads) pair_seeds_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                               const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                               const uint8_t* __restrict__ adj, uint32_t ppt, PairWin w,
                                                               uint8_t* __restrict__ bits) {
    extern __shared__ __align__(16) unsigned char pair_smem_raw[];
    PairSmem& sm = *reinterpret_cast<PairSmem*>(pair_smem_raw);
    uint8_t* const s_adj = pair_smem_raw + sizeof(PairSmem);  // [ppt * ppt] when ppt <= kPAdjSmem
    const bool adj_smem = ppt <= kPAdjSmem;
    const uint32_t tid = threadIdx.x;
    const uint32_t tb = blockIdx.x * (uint32_t)kPTile;
    const uint32_t te = min(n, tb + (uint32_t)kPTile);
    // Staged halo: 32 hits when the 32nd hit before and after the tile already lies outside the largest window (the
    // usual case: a tower has a hit or two inside 250 ns), else kPHalo.  Purely a cost choice: whatever the staged
    // range cannot decide goes to the exact global scans below, so the result does not depend on it.
    uint32_t halo = kPHalo;
    if (tb >= 32u && te + 32u <= n) {
        const int64_t f0 = hit_time(__ldg(hits + (tb - 32u))), f1 = hit_time(__ldg(hits + tb));
        const int64_t b0 = hit_time(__ldg(hits + (te - 1u))), b1 = hit_time(__ldg(hits + (te + 31u)));
        if (f1 >= f0 && b1 >= b0 && udiff(f1, f0) > w.wmax && udiff(b1, b0) > w.wmax) halo = 32u;
    }
    const uint32_t glo = tb >= halo ? tb - halo : 0u;
    const uint32_t ghi = min(n, te + halo);
    const uint32_t g0 = tb - (uint32_t)kPHalo;  // staged slot e <-> global index g0 + e (modulo 2^32), whatever the halo
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
    bool wide = false;
#pragma unroll
    for (int r = 0; r < kPStage / kPThreads; ++r) {
        const uint32_t e = tid + r * kPThreads;
        uint32_t tr = 0xFFFFFFFFu, a = 0xFFFFFFFFu, tw = 0xFFFFFFFFu;
        if (e >= e_lo && e < e_hi) {
            const uint4 v = __ldg(hits + (g0 + e));
            const uint64_t d64 = udiff(hit_time(v), t0);
            wide |= d64 >= 0xFFFFFFFFull;
            tr = (uint32_t)d64;
            split_pmt(v.z, ppt, w.rcp, a, tw);
        }
        sm.t[e] = tr; sm.a[e] = a; sm.tw[e] = tw;
    }
    for (uint32_t i = tid; i < (uint32_t)kPTile / 4; i += kPThreads) sm.f[i] = 0;
    if (tid < (uint32_t)kPPad) { sm.t[kPStage + tid] = 0xFFFFFFFFu; sm.a[kPStage + tid] = 0xFFFFFFFFu; sm.tw[kPStage + tid] = 0xFFFFFFFFu; }
    if (adj_smem)
        for (uint32_t i = tid; i < ppt * ppt; i += kPThreads) s_adj[i] = __ldg(adj + i);
    const bool fits32 = !__syncthreads_or(wide);
    auto clamp32 = [](uint64_t x) { return x > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)x; };
    const uint32_t w_sc = clamp32(w.sc), w_fc = clamp32(w.fc), w_afc = clamp32(w.afc), w_max = clamp32(w.wmax);
    auto sa_ = [&](uint32_t k) { return adj_smem ? s_adj[k] != 0 : __ldg(adj + k) != 0; };
    if (fits32) {
        // round 0: the halo before the tile (marks its in-tile partners only); rounds 1..: the tile.  A warp walks its 32
        // hits in lockstep, four offsets per step, and leaves when no lane has an offset inside its window any more.
        // Prefilter per offset: a rule needs floors within one of each other (FC, AFC) or dt inside the SC window.
        const uint32_t lane = tid & 31u;
#pragma unroll 1
        for (int r = 0; r < (kPTile + kPHalo) / kPThreads; ++r) {
            const uint32_t e = tid + r * kPThreads;
            const uint32_t w0 = e - lane;
            if (w0 >= e_te) break;                 // warp-uniform
            if (w0 + 32u <= e_lo) continue;        // warp-uniform: nothing staged here
            const bool valid = e >= e_lo && e < e_te;
            const uint32_t ti = sm.t[e], ai = sm.a[e], twi = sm.tw[e];
            uint32_t jmax = e_hi, sa = seg_a, sb = seg_b;
            if (!one_seg && valid) {
                const uint32_t s = find_segment(seg_off, n_seg, g0 + e);
                sa = __ldg(seg_off + s);
                sb = __ldg(seg_off + s + 1);
                if (sb < ghi) jmax = sb - g0;
            }
            uint32_t mine = 0;
            const uint32_t fi1 = (ai >> 16) - 1u;  // floor - 1: (floor_j - fi1) <= 2 <=> floors within one of each other
            for (uint32_t d0 = 1;; d0 += 4) {
                const uint32_t j0 = e + d0;
                const uint32_t dt0 = sm.t[j0] - ti;
                if (!__any_sync(0xffffffffu, valid && j0 < jmax && dt0 <= w_max)) break;
                const uint32_t dt1 = sm.t[j0 + 1] - ti, dt2 = sm.t[j0 + 2] - ti, dt3 = sm.t[j0 + 3] - ti;
                const uint32_t a0 = sm.a[j0], a1 = sm.a[j0 + 1], a2 = sm.a[j0 + 2], a3 = sm.a[j0 + 3];
                const bool p0 = valid && j0 < jmax && dt0 <= w_max && ((a0 >> 16) - fi1 <= 2u || dt0 <= w_sc);
                const bool p1 = valid && j0 + 1 < jmax && dt1 <= w_max && ((a1 >> 16) - fi1 <= 2u || dt1 <= w_sc);
                const bool p2 = valid && j0 + 2 < jmax && dt2 <= w_max && ((a2 >> 16) - fi1 <= 2u || dt2 <= w_sc);
                const bool p3 = valid && j0 + 3 < jmax && dt3 <= w_max && ((a3 >> 16) - fi1 <= 2u || dt3 <= w_sc);
                if (p0 | p1 | p2 | p3) {
                    const uint32_t pm = (p0 ? 1u : 0u) | (p1 ? 2u : 0u) | (p2 ? 4u : 0u) | (p3 ? 8u : 0u);
#pragma unroll
                    for (uint32_t q = 0; q < 4; ++q) {
                        if (!((pm >> q) & 1u)) continue;
                        const uint32_t j = j0 + q;
                        const uint32_t m = pair_rules<uint32_t>(ai, twi, sm.a[j], sm.tw[j], sm.t[j] - ti, w_sc, w_fc, w_afc, ppt, sa_);
                        if (m) {
                            mine |= m;
                            if (j >= (uint32_t)kPHalo && j < e_te)
                                atomicOr(&sm.f[(j - kPHalo) >> 2], m << (8 * ((j - kPHalo) & 3)));
                        }
                    }
                }
            }
            if (!valid) continue;
            // the staged hits of this hit's segment end inside its window <=> the last of them is still inside
            const uint32_t j = (jmax - 1u > e && sm.t[jmax - 1u] - ti > w_max) ? 0u : jmax;  // == jmax: not closed
            if (e < (uint32_t)kPHalo) continue;  // a halo hit: its own bits belong to another tile
            // what the staged window leaves open: partners beyond its end / before its start
            const bool open_fwd = j == jmax && jmax == e_hi && ghi < sb;
            const uint32_t first = max(glo, sa);  // first staged hit of this hit's segment
            const bool open_bwd = first > sa && (uint64_t)(ti - sm.t[first - g0]) <= w.wmax;
            if (open_fwd || open_bwd) {
                const int64_t t = (int64_t)((uint64_t)t0 + ti);
                mine |= pair_scan_global(hits, t, ai, twi, open_bwd ? glo : sa, open_fwd ? ghi : sb, sa, sb, w, ppt, adj);
            }
            if (mine) atomicOr(&sm.f[(e - kPHalo) >> 2], mine << (8 * ((e - kPHalo) & 3)));
        }
    } else {
        // sparse tile (>= 2^32 ps across the staged hits): exact scans of global memory
#pragma unroll 1
        for (int r = 1; r < (kPTile + kPHalo) / kPThreads; ++r) {
            const uint32_t e = tid + r * kPThreads;
            if (e >= e_te) break;
            const uint32_t g = g0 + e;
            uint32_t sa = seg_a, sb = seg_b;
            if (!one_seg) {
                const uint32_t s = find_segment(seg_off, n_seg, g);
                sa = __ldg(seg_off + s);
                sb = __ldg(seg_off + s + 1);
            }
            const uint4 v = __ldg(hits + g);
            uint32_t ai, twi;
            split_pmt(v.z, ppt, w.rcp, ai, twi);
            const uint32_t mine = pair_scan_global(hits, hit_time(v), ai, twi, g, g + 1, sa, sb, w, ppt, adj);
            if (mine) atomicOr(&sm.f[(e - kPHalo) >> 2], mine << (8 * ((e - kPHalo) & 3)));
        }
    }
    __syncthreads();
    // thread t writes the kPPer bytes [kPPer t, kPPer t + kPPer) of the tile
    const uint32_t i0 = tb + tid * kPPer;
    const uint32_t w0 = sm.f[2 * tid], w1 = sm.f[2 * tid + 1];
    if (i0 + kPPer <= te && (((uintptr_t)(bits + i0)) & 7) == 0) {
        *reinterpret_cast<uint2*>(bits + i0) = make_uint2(w0, w1);
    } else {
        for (uint32_t b8 = 0; b8 < (uint32_t)kPPer && i0 + b8 < te; ++b8)
            bits[i0 + b8] = (uint8_t)(((b8 < 4 ? w0 : w1) >> (8 * (b8 & 3))) & 0xFFu);
    }
}

// The combined trigger on firing level-0 window starts (reading R22): OR of the pair bits of the N hits k..k+N-1.
// One CTA per tile of kCTile hits: the tile's pair bytes and the N - 1 bytes behind it are staged in shared memory,
// lanes take consecutive hits (their window bytes are consecutive: conflict-free reads), the result bytes go back
// through shared memory so that every thread writes 16 of them at once; one pair of atomics per CTA for the counts.
constexpr int kCThreads = 256;
constexpr int kCPer = 16;
constexpr int kCTile = kCThreads * kCPer;  // 4096
__global__ void __launch_bounds__(kCThreads) l0_combine_kernel(const uint8_t* __restrict__ l0,
                                                               const uint8_t* __restrict__ pair_bits, uint32_t n,
                                                               uint32_t N, uint8_t* __restrict__ cand,
                                                               uint32_t* __restrict__ n_cand) {
    __shared__ __align__(16) uint8_t s_pb[kCTile + TT_MAX_L0_MULTIPLICITY];
    __shared__ __align__(16) uint8_t s_l0[kCTile];
    __shared__ __align__(16) uint8_t s_out[kCTile];
    __shared__ uint32_t s_cnt[2];
    const uint32_t tid = threadIdx.x;
    const uint32_t tb = blockIdx.x * (uint32_t)kCTile;
    const uint32_t te = min(n, tb + (uint32_t)kCTile);
    const uint32_t i0 = tb + tid * kCPer;
    if (tid < 2) s_cnt[tid] = 0;
    // stage: 16 bytes per thread of both arrays (vector loads when the pointers allow), then the halo of pair bytes
    const bool full = i0 + kCPer <= te;
    if (full && ((((uintptr_t)(pair_bits + i0)) | ((uintptr_t)(l0 + i0))) & 15) == 0) {
        reinterpret_cast<uint4*>(s_pb)[tid] = __ldg(reinterpret_cast<const uint4*>(pair_bits + i0));
        reinterpret_cast<uint4*>(s_l0)[tid] = __ldg(reinterpret_cast<const uint4*>(l0 + i0));
    } else {
        for (uint32_t b8 = 0; b8 < (uint32_t)kCPer; ++b8) {
            const uint32_t i = i0 + b8;
            s_pb[tid * kCPer + b8] = i < te ? pair_bits[i] : (uint8_t)0;
            s_l0[tid * kCPer + b8] = i < te ? l0[i] : (uint8_t)0;
        }
    }
    for (uint32_t h = tid; h + 1 < N; h += kCThreads) {  // N - 1 bytes behind the tile
        const uint32_t i = tb + (uint32_t)kCTile + h;
        s_pb[kCTile + h] = i < n ? pair_bits[i] : (uint8_t)0;
    }
    __syncthreads();
    uint32_t ca = 0, cb = 0;
#pragma unroll 4
    for (int r = 0; r < kCPer; ++r) {
        const uint32_t q = tid + r * kCThreads;  // lanes on consecutive hits
        uint32_t out = 0;
        if (tb + q < te && (s_l0[q] & TT_L0_START)) {
            uint32_t m = 0;
            for (uint32_t j = 0; j < N; ++j) m |= s_pb[q + j];  // bytes past n are 0: a start from tt_l0_ntw never needs them
            if ((m & TT_P_SC) && (m & TT_P_AFC)) { out |= TT_P_CAND_A; ++ca; }
            if ((m & TT_P_FC) && (m & TT_P_AFC)) { out |= TT_P_CAND_B; ++cb; }
        }
        s_out[q] = (uint8_t)out;
    }
    __syncthreads();
    if (full && (((uintptr_t)(cand + i0)) & 15) == 0) {
        *reinterpret_cast<uint4*>(cand + i0) = reinterpret_cast<const uint4*>(s_out)[tid];
    } else {
        for (uint32_t b8 = 0; b8 < (uint32_t)kCPer && i0 + b8 < te; ++b8) cand[i0 + b8] = s_out[tid * kCPer + b8];
    }
    if (n_cand) {
        ca = __reduce_add_sync(0xffffffffu, ca);
        cb = __reduce_add_sync(0xffffffffu, cb);
        if ((tid & 31) == 0) {
            if (ca) atomicAdd(&s_cnt[0], ca);
            if (cb) atomicAdd(&s_cnt[1], cb);
        }
        __syncthreads();
        if (tid < 2 && s_cnt[tid]) atomicAdd(n_cand + tid, s_cnt[tid]);
    }
}

}  // namespace tt

static int pairs_attrs() {
    TT_CUDA_OK(cudaFuncSetAttribute(tt::pair_seeds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(sizeof(tt::PairSmem) + tt::kPAdjSmem * tt::kPAdjSmem)));
    return TT_OK;
}

extern "C" int tt_pair_seeds(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                             const uint8_t* d_adj, uint32_t pmts_per_tower, int64_t sc_window_ps, int64_t fc_window_ps,
                             int64_t afc_window_ps, uint8_t* d_bits, void* stream) {
    using namespace tt;
    cudaStream_t s = (cudaStream_t)stream;
    if (pmts_per_tower < 1 || pmts_per_tower > 65535u) return TT_E_INVAL;
    if (sc_window_ps < 0 || fc_window_ps < 0 || afc_window_ps < 0) return TT_E_INVAL;
    if (n && (!d_sorted || !d_bits || !d_seg_offsets || !d_adj || n_seg < 1)) return TT_E_INVAL;
    if (n >= 0xFFF00000u) return TT_E_INVAL;
    if (n == 0) return TT_OK;
    PairWin w;
    w.sc = (uint64_t)sc_window_ps; w.fc = (uint64_t)fc_window_ps; w.afc = (uint64_t)afc_window_ps;
    w.wmax = w.sc > w.fc ? w.sc : w.fc;
    w.wmax = w.afc > w.wmax ? w.afc : w.wmax;
    w.rcp = ((1ull << 32) + pmts_per_tower - 1) / pmts_per_tower;
    const size_t smem = sizeof(PairSmem) + (pmts_per_tower <= kPAdjSmem ? (size_t)pmts_per_tower * pmts_per_tower : 0);
    {
        const int rc = once_per_device(kSlotPairs, pairs_attrs);
        if (rc != TT_OK) return rc;
    }
    prof_mark(s, "pairs.seeds");
    TT_K(pair_seeds_kernel)<<<div_up(n, kPTile), kPThreads, smem, s>>>((const uint4*)d_sorted, n, d_seg_offsets, n_seg,
                                                                        d_adj, pmts_per_tower, w, d_bits);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}

extern "C" int tt_l0_combine(const uint8_t* d_l0, const uint8_t* d_pair_bits, uint32_t n, uint32_t multiplicity,
                             uint8_t* d_cand, uint32_t* d_n_cand, void* stream) {
    using namespace tt;
    cudaStream_t s = (cudaStream_t)stream;
    if (multiplicity < 1 || multiplicity > TT_MAX_L0_MULTIPLICITY) return TT_E_INVAL;
    if (n && (!d_l0 || !d_pair_bits || !d_cand)) return TT_E_INVAL;
    if (d_n_cand) TT_CUDA_OK(cudaMemsetAsync(d_n_cand, 0, 2 * sizeof(uint32_t), s));
    if (n == 0) return TT_OK;
    prof_mark(s, "pairs.combine");
    TT_K(l0_combine_kernel)<<<div_up(n, kCTile), kCThreads, 0, s>>>(d_l0, d_pair_bits, n, multiplicity, d_cand, d_n_cand);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}
