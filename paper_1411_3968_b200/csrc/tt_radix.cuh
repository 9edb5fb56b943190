// tt_radix.cuh -- the LSD radix machinery of tt_radix.cu, shared with tt_prepare.cu.
#pragma once
#include "tt_common.cuh"

namespace tt {

struct RadixState {        // device-resident control block
    uint32_t cur;          // which ping-pong buffer holds the current pairs (0/1)
    uint32_t skip;         // set by the scan step of a pass whose digit is constant
};

struct RadixPlan {
    uint64_t *keys0, *keys1;
    uint32_t *idx0, *idx1, *hist, *scan_scratch;
    RadixState* st;
    uint32_t nblocks;
};

void radix_plan(Arena& a, uint32_t n, RadixPlan& p);
// 8-bit LSD passes [pass_begin, pass_end) over the plan's (key, index) pairs (passes >= 8 use the segment id)
int radix_run_passes(const RadixPlan& p, uint32_t n, int pass_begin, int pass_end, const uint32_t* d_seg_offsets,
                     uint32_t n_seg, cudaStream_t s);

}  // namespace tt
