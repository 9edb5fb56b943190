// tt_merge.cuh -- what the run-merge sort (tt_merge.cu) shares with its callers (tt_api.cu, tt_trigger.cu).
#pragma once
#include "tt_common.cuh"

namespace tt {

// Device view of one merge level (all arrays live in the caller's sort workspace).
struct LevelDev {
    const uint32_t* roff;    // [R+1] run offsets of this level
    uint32_t* gfirst;        // [G+1] first run of each group
    uint32_t* tbase;         // [G+1] exclusive prefix of tiles per group
    uint32_t* sbase;         // [G+1] exclusive prefix of split-table entries per group ((tiles+1) * K)
    uint64_t* gT0;           // [G] smallest key of the group
    uint64_t* gDT;           // [G] tile width in key units (>= 1)
    uint64_t* gKmax;         // [G] largest key of the group
    uint32_t* run_group;     // [R] group of every run of this level
    uint32_t* gScale;        // [G] floor(kFCap * 2^32 / DT) when kFCap < DT < 2^32 (the fast tile kernel's bucket map), else 0
    uint32_t* splits;        // split table
    uint32_t* roff_next;     // [G+1] run offsets of the next level (= group boundaries)
    uint4* tile_desc;        // [tiles] {group, first run, runs K, tile k of the group}: one load instead of a chain
    uint2* tile_desc2;       // [tiles] {split-table offset of the tile's row, tile_base index}
    uint32_t* tile_base;     // [tiles + G + 1] hits of the group before tile k (nt + 1 entries per group, zeroed, summed by atomics)
    uint32_t* slow_list;     // [tiles] tiles the fast kernel left to the general kernel
    uint32_t* slow_cnt;      // [1]
    uint8_t* tile_open;      // [tiles] fused L1 only: 1 = the tile has no in-tile L1 bits (every hit is finished by l1_boundary_kernel)
    uint32_t R, G, F;
};

// L1 evaluated on the sorted tile of the LAST merge level while it sits in shared memory (tt_sort_trigger_slice).
struct FuseL1 {
    uint8_t* flags;          // [n] flag bytes of the sorted hits; nullptr = no fusion
    uint64_t lc;             // same-floor coincidence window
    uint32_t q_thresh;
};

// What the fused caller needs from the sort to finish the hits near the tile edges.
struct MergeLast {
    LevelDev lv;             // last level
    uint32_t tiles;          // its tile count (host)
};

size_t merge_ws_bytes(uint32_t n, const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* h_run_offsets,
                      uint32_t n_runs);
// fuse / last: both null for the plain sort
int merge_sort_runs(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
                    const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* d_run_offsets,
                    const uint32_t* h_run_offsets, uint32_t n_runs, void* d_ws, int32_t* d_status, cudaStream_t s,
                    const FuseL1* fuse, MergeLast* last);

}  // namespace tt
