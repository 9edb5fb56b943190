// tt_dn.cu -- distinct-PMT level-0 trigger DNnTW on time-sorted hits (second half).
//
//   PAPER.md:60  "DN7TW1000: looking for 7 hits from different PMTs within TW = 1000 ns"
//   PAPER.md:67  "more efficient in the presence of bioluminescence ... time consuming" (the paper ran N7TW instead)
//   DESIGN.md reading R23: window start k fires <=> the hits j >= k of k's segment with t_j - t_k < TW (strict, as for
//   N-in-TW) carry at least N different pmt_id values; its members are k..e_k, e_k = the first hit at which the N-th
//   different PMT appears.
//
// One CTA per tile of kDTile sorted hits; the tile and kDHalo hits behind it are staged as (64-bit key, pmt).  Every
// in-tile hit scans forward, keeping the different PMTs seen so far (N <= 16) behind a Bloom mask; a window still open at the
// staged end goes on in global memory, so the result is the plain definition for any density.  Members can lie in later
// tiles: the output is zeroed by the call and every byte reaches it through atomicOr.
#include "tt_common.cuh"

namespace tt {

constexpr int kDThreads = 256;
constexpr int kDPer = 4;
constexpr int kDTile = kDThreads * kDPer;  // 1024
constexpr int kDHalo = 256;
constexpr int kDStage = kDTile + kDHalo;

struct DnSmem {
    uint64_t key[kDStage];
    uint16_t pmt[kDStage];
    uint32_t f[kDTile / 4];  // result bytes of the tile
    uint16_t seen[TT_MAX_DN_MULTIPLICITY][kDThreads];  // the different PMTs of the running window, one column per thread
    uint32_t red[kDThreads / 32];
    uint32_t n_cand;                // starts that passed the plain N-in-TW pre-test
    uint16_t cand[kDTile];          // their tile positions
};

// OR `bits` into byte i of a byte array of any alignment (the aligned 32-bit word around it lies inside the same
// allocation granule)
__device__ __forceinline__ void or_byte(uint8_t* base, uint32_t i, uint32_t bits) {
    const uintptr_t a = (uintptr_t)(base + i);
    atomicOr(reinterpret_cast<uint32_t*>(a & ~(uintptr_t)3), bits << (8 * (uint32_t)(a & 3)));
}

__global__ void __launch_bounds__(kDThreads) l0_dntw_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                            const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                            uint32_t N, uint64_t tw, uint8_t* __restrict__ l0,
                                                            uint32_t* __restrict__ n_start) {
    __shared__ DnSmem sm;
    const uint32_t tid = threadIdx.x;
    const uint32_t tb = blockIdx.x * (uint32_t)kDTile;
    const uint32_t te = min(n, tb + (uint32_t)kDTile);
    const uint32_t ghi = min(n, te + (uint32_t)kDHalo);
    uint32_t seg_b = n;
    bool one_seg = true;
    if (n_seg > 1) {
        const uint32_t s = find_segment(seg_off, n_seg, tb);
        seg_b = __ldg(seg_off + s + 1);
        one_seg = seg_b >= ghi;
    }
#pragma unroll
    for (int r = 0; r < kDStage / kDThreads; ++r) {
        const uint32_t q = tid + r * kDThreads;
        uint64_t key = ~0ull;
        uint32_t p = 0;
        if (tb + q < ghi) {
            const uint4 v = __ldg(hits + (tb + q));
            key = key_of(hit_time(v));
            p = v.z & 0xFFFFu;
        }
        sm.key[q] = key;
        sm.pmt[q] = (uint16_t)p;
    }
    sm.f[tid] = 0;
    if (tid == 0) sm.n_cand = 0;
    __syncthreads();
    // N different PMTs need N hits: the plain N-in-TW test on hit k + N - 1 (staged: N - 1 < kDHalo) rules out most
    // starts of a quiet tower before any scan (one tower at 55 kHz per PMT: 97 %).  The survivors go to a list and are
    // scanned one per thread afterwards, so a warp is not held by the one lane in thirty that has a window to walk.
#pragma unroll
    for (int r = 0; r < kDPer; ++r) {
        const uint32_t q = tid + r * kDThreads;
        const uint32_t k = tb + q;
        bool pass = false;
        if (k < te) {
            uint32_t sb = seg_b;
            if (!one_seg) sb = __ldg(seg_off + find_segment(seg_off, n_seg, k) + 1);
            pass = (uint64_t)k + N - 1 < sb && sm.key[q + N - 1] - sm.key[q] < tw;
        }
        const uint32_t mk = __ballot_sync(0xffffffffu, pass);
        if (mk) {
            uint32_t base = 0;
            if ((tid & 31u) == 0) base = atomicAdd(&sm.n_cand, (uint32_t)__popc(mk));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (pass) sm.cand[base + (uint32_t)__popc(mk & lanemask_lt())] = (uint16_t)q;
        }
    }
    __syncthreads();
    const uint32_t n_cand = sm.n_cand;
    uint32_t my_starts = 0;
#pragma unroll 1
    for (uint32_t c = tid; c < n_cand; c += kDThreads) {
        const uint32_t q = sm.cand[c];
        const uint32_t k = tb + q;
        uint32_t sb = seg_b;
        if (!one_seg) sb = __ldg(seg_off + find_segment(seg_off, n_seg, k) + 1);
        const uint64_t tk = sm.key[q];
        // the different PMTs seen so far: a 64-bit Bloom mask in a register decides "new" in the common case, the exact
        // list (a column of shared memory) is only read when the mask bit is already set
        uint64_t mask = 0;
        uint32_t cnt = 0;
        auto add = [&](uint32_t p) -> bool {
            const uint64_t bit = 1ull << (p & 63u);
            if (mask & bit)
                for (uint32_t c = 0; c < cnt; ++c)
                    if (sm.seen[c][tid] == (uint16_t)p) return false;
            mask |= bit;
            sm.seen[cnt][tid] = (uint16_t)p;
            ++cnt;
            return true;
        };
        bool fire = false, closed = false;
        uint32_t j = k;
        const uint32_t stage_end = min(sb, ghi);
        for (; j < stage_end; ++j) {  // the staged part of the window
            if (sm.key[j - tb] - tk >= tw) { closed = true; break; }
            if (add(sm.pmt[j - tb]) && cnt == N) { fire = true; break; }
        }
        if (!fire && !closed) {       // still open at the staged end: on in global memory
            for (; j < sb; ++j) {
                const uint4 v = __ldg(hits + j);
                if (key_of(hit_time(v)) - tk >= tw) break;
                if (add(v.z & 0xFFFFu) && cnt == N) { fire = true; break; }
            }
        }
        if (!fire) continue;
        ++my_starts;
        atomicOr(&sm.f[q >> 2], (uint32_t)(TT_L0_START | TT_L0_MEMBER) << (8 * (q & 3)));
        for (uint32_t m = k + 1; m <= j; ++m) {  // members k..j (j = e_k)
            if (m < te) {
                const uint32_t qm = m - tb;
                atomicOr(&sm.f[qm >> 2], (uint32_t)TT_L0_MEMBER << (8 * (qm & 3)));
            } else {
                or_byte(l0, m, TT_L0_MEMBER);
            }
        }
    }
    __syncthreads();
    // the tile's bytes: OR-ed in (later tiles' members may already be there, earlier tiles may still add theirs)
    {
        const uint32_t w = sm.f[tid];
        const uint32_t i0 = tb + 4 * tid;
        if (w) {
            if (i0 + 4 <= te && (((uintptr_t)(l0 + i0)) & 3) == 0) {
                atomicOr(reinterpret_cast<uint32_t*>(l0 + i0), w);
            } else {
                for (uint32_t b8 = 0; b8 < 4u && i0 + b8 < te; ++b8) {
                    const uint32_t f = (w >> (8 * b8)) & 0xFFu;
                    if (f) or_byte(l0, i0 + b8, f);
                }
            }
        }
    }
    if (n_start) {
        my_starts = __reduce_add_sync(0xffffffffu, my_starts);
        if ((tid & 31) == 0) sm.red[tid >> 5] = my_starts;
        __syncthreads();
        if (tid == 0) {
            uint32_t c = 0;
#pragma unroll
            for (int w = 0; w < kDThreads / 32; ++w) c += sm.red[w];
            if (c) atomicAdd(n_start, c);
        }
    }
}

}  // namespace tt

extern "C" int tt_l0_dntw(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                          uint32_t multiplicity, int64_t window_ps, uint8_t* d_l0, uint32_t* d_n_start, void* stream) {
    using namespace tt;
    cudaStream_t s = (cudaStream_t)stream;
    if (multiplicity < 1 || multiplicity > TT_MAX_DN_MULTIPLICITY) return TT_E_INVAL;
    if (n && (!d_sorted || !d_l0 || !d_seg_offsets || n_seg < 1)) return TT_E_INVAL;
    if (n >= 0xFFF00000u) return TT_E_INVAL;
    if (d_n_start) TT_CUDA_OK(cudaMemsetAsync(d_n_start, 0, sizeof(uint32_t), s));
    if (n == 0) return TT_OK;
    TT_CUDA_OK(cudaMemsetAsync(d_l0, 0, n, s));
    const uint64_t tw = window_ps > 0 ? (uint64_t)window_ps : 0ull;  // TW <= 0 never fires
    prof_mark(s, "l0.dntw");
    TT_K(l0_dntw_kernel)<<<div_up(n, kDTile), kDThreads, 0, s>>>((const uint4*)d_sorted, n, d_seg_offsets, n_seg,
                                                                  multiplicity, tw, d_l0, d_n_start);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}
