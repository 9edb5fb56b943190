// tt_l0.cu -- level-0 N-in-TW trigger on time-sorted hits.
//
//   PAPER.md:59  "N7TW1000: looking for 7 hits in TW = 1000 ns: hit[i].time-hit[i+7].time< TW"
//   PAPER.md:73  N7TW500 for the 84-PMT tower (20 m floors)
//   PAPER.md:67  "we have chosen N7TW1000 first (as level 0 trigger)"
//   DESIGN.md reading R14 / R20: the printed formula has the sign reversed and 7 hits span i..i+6, so window start k
//   fires <=> hit k+N-1 exists in k's segment and t[k+N-1] - t[k] < TW (strict, as printed).
//
// One CTA per tile of kL0Tile consecutive sorted hits.  The times of the tile and of kHalo hits on both sides are
// staged in shared memory; every staged position computes its start bit once, the bits are packed with warp ballots
// (a halo that is a multiple of 32 keeps bitmap words aligned with warps), and a hit is a member of a firing window
// <=> one of the N positions ending at it is a firing start (a firing window lies inside its start's segment, so no
// segment test is needed there).  Streaming kernel: reads 16 B/hit (the records are AoS; only the time is used), writes 1 B/hit.
#include "tt_common.cuh"

namespace tt {

constexpr int kL0Threads = 128;
constexpr int kL0Per = 8;
constexpr int kL0Tile = kL0Threads * kL0Per;   // 1024
static_assert(TT_MAX_L0_MULTIPLICITY - 1 <= 256, "the wide halo covers the longest window");

// kHalo staged hits before and after the tile (>= N - 1, multiple of 32): 32 for N <= 33 (N7TW: 6 % of re-reads, 10 KB
// of shared memory per CTA), 256 for the long windows.  Small CTAs on purpose: the kernel is bound by the latency of
// its staging loads, so what counts is how many CTAs are resident per SM (ncu, profiles/r1_v6.md).
template <int kHalo>
struct L0Smem {
    static constexpr int kStage = kL0Tile + 2 * kHalo;
    uint64_t t[kStage];                   // order-preserving keys of the staged times
    uint32_t start[kStage / 32];          // start bits of the staged positions (the last kHalo stay 0)
    uint32_t red[kL0Threads / 32];
};

template <int kHalo>
__global__ void __launch_bounds__(kL0Threads, 16) l0_ntw_kernel(const uint4* __restrict__ hits, uint32_t n,
                                                               const uint32_t* __restrict__ seg_off, uint32_t n_seg,
                                                               uint32_t N, uint64_t tw, uint8_t* __restrict__ l0,
                                                               uint32_t* __restrict__ n_start) {
    constexpr int kL0Halo = kHalo;
    constexpr int kL0Stage = L0Smem<kHalo>::kStage;
    constexpr int kStageRounds = (kL0Stage + kL0Threads - 1) / kL0Threads;
    constexpr int kStartRounds = (kL0Tile + kL0Halo + kL0Threads - 1) / kL0Threads;
    __shared__ L0Smem<kHalo> sm;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tb = blockIdx.x * (uint32_t)kL0Tile;
    const uint32_t te = min(n, tb + (uint32_t)kL0Tile);
    // staged slot q <-> global index tb - kL0Halo + q
    const int64_t g0 = (int64_t)tb - kL0Halo;
    const uint32_t glo = tb >= (uint32_t)kL0Halo ? tb - kL0Halo : 0u;
    const uint32_t ghi = min(n, te + (uint32_t)kL0Halo);
    uint32_t seg_b = n;
    bool one_seg = true;
    if (n_seg > 1) {
        const uint32_t s = find_segment(seg_off, n_seg, glo);
        seg_b = __ldg(seg_off + s + 1);
        one_seg = seg_b >= ghi;
    }
    // ---- stage the times (8-byte loads of the first half of each record) ---------------------------------
    const uint2* __restrict__ h2 = reinterpret_cast<const uint2*>(hits);
#pragma unroll
    for (int r = 0; r < kStageRounds; ++r) {
        const uint32_t q = tid + r * kL0Threads;
        if (kL0Stage % kL0Threads != 0 && q >= (uint32_t)kL0Stage) break;
        const int64_t gp = g0 + q;
        uint64_t key = 0;
        if (gp >= (int64_t)glo && gp < (int64_t)ghi) {
            const uint2 v = __ldg(h2 + 2 * (size_t)gp);
            key = (((uint64_t)v.y << 32) | v.x) ^ 0x8000000000000000ull;
        }
        sm.t[q] = key;
    }
    __syncthreads();
    // ---- start bits of the positions [tb - kL0Halo, te): warp w, round r owns bitmap word w + 8 r -----------
    uint32_t my_starts = 0;
#pragma unroll
    for (int r = 0; r < kStartRounds; ++r) {
        const uint32_t q = tid + r * kL0Threads;
        if ((kL0Tile + kL0Halo) % kL0Threads != 0 && q - lane >= (uint32_t)(kL0Tile + kL0Halo)) break;  // warp-uniform
        const int64_t gp = g0 + q;
        bool fire = false;
        if (gp >= (int64_t)glo && gp < (int64_t)te) {
            uint32_t sb = seg_b;
            if (!one_seg) sb = __ldg(seg_off + find_segment(seg_off, n_seg, (uint32_t)gp) + 1);
            const uint64_t last = (uint64_t)gp + N - 1;
            if (last < sb) fire = sm.t[q + N - 1] - sm.t[q] < tw;  // sorted: the difference is the exact span
        }
        const uint32_t word = __ballot_sync(0xffffffffu, fire);
        if (lane == 0) sm.start[warp + r * (kL0Threads / 32)] = word;
        if (fire && gp >= (int64_t)tb) ++my_starts;
    }
    if (tid < kL0Halo / 32) sm.start[(kL0Tile + kL0Halo) / 32 + tid] = 0;
    __syncthreads();
    // ---- member bits + output: thread t owns the kL0Per consecutive hits from tb + kL0Per * t -----------------
    uint32_t out[kL0Per / 4] = {};
#pragma unroll
    for (int j = 0; j < kL0Per; ++j) {
        const uint32_t q = (uint32_t)kL0Halo + tid * kL0Per + j;  // staged slot of the hit
        uint32_t f = (sm.start[q >> 5] >> (q & 31)) & 1u;
        // any start bit among the N positions ending at q: 32 positions at a time, going back
        bool member = false;
        uint32_t left = N, qe = q;  // window of positions (qe - 31 .. qe], `left` of them still to be looked at
        while (left) {
            const uint32_t w = qe >> 5, sh = qe & 31u;
            const uint32_t hiw = sm.start[w], low = w ? sm.start[w - 1] : 0u;
            // bit 31 <-> position qe, bit 0 <-> position qe - 31
            const uint32_t v = sh == 31u ? hiw : __funnelshift_r(low, hiw, sh + 1u);
            const uint32_t take = left < 32u ? left : 32u;
            if (v >> (32u - take)) { member = true; break; }
            left -= take;
            if (qe < 32u) break;  // positions before slot 0 do not exist
            qe -= 32u;
        }
        if (member) f |= 2u;
        out[j >> 2] |= f << (8 * (j & 3));
    }
    const uint32_t i0 = tb + tid * kL0Per;
    if (i0 + kL0Per <= te && (((uintptr_t)(l0 + i0)) & 7) == 0) {
        *reinterpret_cast<uint2*>(l0 + i0) = make_uint2(out[0], out[1]);
    } else {
        for (uint32_t b8 = 0; b8 < (uint32_t)kL0Per && i0 + b8 < te; ++b8)
            l0[i0 + b8] = (uint8_t)((out[b8 >> 2] >> (8 * (b8 & 3))) & 0xFFu);
    }
    if (n_start) {
        my_starts = __reduce_add_sync(0xffffffffu, my_starts);
        if (lane == 0) sm.red[warp] = my_starts;
        __syncthreads();
        if (tid == 0) {
            uint32_t c = 0;
#pragma unroll
            for (int w = 0; w < kL0Threads / 32; ++w) c += sm.red[w];
            if (c) atomicAdd(n_start, c);
        }
    }
}

}  // namespace tt

extern "C" int tt_l0_ntw(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                         uint32_t multiplicity, int64_t window_ps, uint8_t* d_l0, uint32_t* d_n_start, void* stream) {
    using namespace tt;
    cudaStream_t s = (cudaStream_t)stream;
    if (multiplicity < 1 || multiplicity > TT_MAX_L0_MULTIPLICITY) return TT_E_INVAL;
    if (n && (!d_sorted || !d_l0 || !d_seg_offsets || n_seg < 1)) return TT_E_INVAL;
    if (n >= 0xFFF00000u) return TT_E_INVAL;
    if (d_n_start) TT_CUDA_OK(cudaMemsetAsync(d_n_start, 0, sizeof(uint32_t), s));
    if (n == 0) return TT_OK;
    const uint64_t tw = window_ps > 0 ? (uint64_t)window_ps : 0ull;  // TW <= 0 never fires
    prof_mark(s, "l0.ntw");
    if (multiplicity <= 33u)
        TT_K(l0_ntw_kernel<32>)<<<div_up(n, kL0Tile), kL0Threads, 0, s>>>((const uint4*)d_sorted, n, d_seg_offsets, n_seg,
                                                                           multiplicity, tw, d_l0, d_n_start);
    else
        TT_K(l0_ntw_kernel<256>)<<<div_up(n, kL0Tile), kL0Threads, 0, s>>>((const uint4*)d_sorted, n, d_seg_offsets, n_seg,
                                                                            multiplicity, tw, d_l0, d_n_start);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}
