// tt_prepare.cu -- the paper's preparation step on the GPU.
//   PAPER.md:41  "Every PMT hit data point ... contains a header with the GPS time and geometry information, followed
//                by a sampled charge waveform with a variable size. ... the raw hits are converted to a fixed size
//                structure that contains ... charge, time, DU identification"
//   PAPER.md:45  "convert 5 consecutive time slices of 200 ms to a unique time slice of 1 s ... (one fixed-size
//                memory buffer) ... filling the same memory zone but at different offsets"
//   PAPER.md:71  this step costs the paper's CPU 200-300 ms per second of data.
// The raw format is this build's (reading R24): 16-byte headers in arrival order and the waveforms of all
// hits concatenated in the same order.  Steps: (1) key = slice * n_pmt + pmt per hit, waveform lengths to a scan
// (the start of every variable-length waveform), (2) stable LSD radix passes on the key digits that vary (the
// machinery of tt_radix.cu), (3) run offsets = lower bounds of the keys in the sorted key array, (4) one gather that
// sums the waveform and writes the 16-byte record at its PMT-major position.
#include "tt_radix.cuh"

namespace tt {

struct RawView {
    int64_t t;
    uint32_t pmt, floor, ns, pad;
};
__device__ __forceinline__ RawView unpack_raw(const uint4& v) {
    RawView r;
    r.t = (int64_t)(((uint64_t)v.y << 32) | (uint64_t)v.x);
    r.pmt = v.z & 0xFFFFu;
    r.floor = v.z >> 16;
    r.ns = v.w & 0xFFFFu;
    r.pad = v.w >> 16;
    return r;
}

__global__ void __launch_bounds__(256) prep_extract_kernel(const uint4* __restrict__ raw, uint32_t n,
                                                           const uint32_t* __restrict__ slice_off, uint32_t n_slices,
                                                           uint32_t n_pmt, uint64_t* __restrict__ keys,
                                                           uint32_t* __restrict__ idx, uint32_t* __restrict__ nsamp,
                                                           RadixState* st, int32_t* __restrict__ status) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { st->cur = 0; st->skip = 0; }
    bool bad = false;
    if (i < n) {
        const RawView r = unpack_raw(__ldg(raw + i));
        uint32_t p = r.pmt;
        if (p >= n_pmt) { p = n_pmt - 1u; bad = true; }  // filed under the last PMT of its slice, status says so
        const uint32_t sl = n_slices > 1 ? find_segment(slice_off, n_slices, i) : 0u;
        keys[i] = (uint64_t)sl * n_pmt + p;
        idx[i] = i;
        nsamp[i] = r.ns;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(status, TT_S_BAD_PMT);
}

// run_off[k] = first position of the sorted key array with key >= k (k = 0 .. n_keys)
__global__ void __launch_bounds__(256) prep_runoff_kernel(const uint64_t* __restrict__ keys0,
                                                          const uint64_t* __restrict__ keys1,
                                                          const RadixState* __restrict__ st, uint32_t n, uint32_t n_keys,
                                                          uint32_t* __restrict__ run_off) {
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > n_keys) return;
    const uint64_t* keys = st->cur ? keys1 : keys0;
    uint32_t lo = 0, hi = n;
    while (lo < hi) { const uint32_t mid = lo + ((hi - lo) >> 1); if (keys[mid] < (uint64_t)k) lo = mid + 1; else hi = mid; }
    run_off[k] = lo;
}

__global__ void __launch_bounds__(256) prep_gather_kernel(const uint4* __restrict__ raw, const uint16_t* __restrict__ samples,
                                                          uint32_t n_samples_total, const uint32_t* __restrict__ woff,
                                                          const uint32_t* __restrict__ idx0,
                                                          const uint32_t* __restrict__ idx1,
                                                          const RadixState* __restrict__ st, uint32_t n,
                                                          uint4* __restrict__ out, int32_t* __restrict__ status) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    bool cut = false;
    if (i < n) {
        const uint32_t src = (st->cur ? idx1 : idx0)[i];
        const uint4 v = __ldg(raw + src);
        const RawView r = unpack_raw(v);
        const uint32_t w0 = woff[src];
        uint32_t avail = w0 < n_samples_total ? n_samples_total - w0 : 0u;  // samples behind the section count as 0
        uint32_t m = r.ns;
        if (m > avail) { m = avail; cut = true; }
        uint32_t sum = 0;  // <= 65535 * 65535 < 2^32
        for (uint32_t j = 0; j < m; ++j) sum += __ldg(samples + w0 + j);
        const uint32_t charge = sum > 65535u ? 65535u : sum;
        out[i] = make_uint4(v.x, v.y, v.z, charge | (r.pad << 16));
    }
    if (__syncthreads_or(cut) && threadIdx.x == 0) atomicOr(status, TT_S_RAW_TRUNCATED);
}

struct PrepPlan {
    RadixPlan rp;
    uint32_t* nsamp;  // waveform lengths, then (scanned in place) waveform starts
    uint32_t* scan_scratch;
};

static void prep_plan(Arena& a, uint32_t n, PrepPlan& p) {
    radix_plan(a, n, p.rp);
    p.nsamp = a.take<uint32_t>((size_t)n + 1);
    p.scan_scratch = a.take<uint32_t>(scan_ws_count(n + 1));
}

}  // namespace tt
using namespace tt;

extern "C" int tt_prepare_slice(const tt_raw_hit* d_raw, const uint16_t* d_samples, uint32_t n_raw,
                                uint32_t n_samples_total, const uint32_t* d_slice_offsets,
                                const uint32_t* h_slice_offsets, uint32_t n_slices, uint32_t n_pmt, tt_hit* d_out,
                                uint32_t out_cap, uint32_t* d_run_offsets, void* d_ws, size_t* ws_bytes,
                                int32_t* d_status, void* stream) {
    if (!ws_bytes || n_slices < 1 || n_pmt < 1 || n_pmt > 65536 || n_raw >= 0xFFF00000u || !h_slice_offsets) return TT_E_INVAL;
    if ((uint64_t)n_slices * n_pmt >= 0x7FFFFFFFull) return TT_E_INVAL;
    if (h_slice_offsets[0] != 0 || h_slice_offsets[n_slices] != n_raw) return TT_E_INVAL;
    for (uint32_t s = 0; s < n_slices; ++s)
        if (h_slice_offsets[s] > h_slice_offsets[s + 1]) return TT_E_INVAL;
    if (n_raw > out_cap) return TT_E_INVAL;  // the output buffer is sized by the caller (for 5 x the nominal rate)
    Arena sizing(nullptr);
    PrepPlan plan;
    prep_plan(sizing, n_raw, plan);
    if (!d_ws) {
        *ws_bytes = sizing.off;
        return TT_OK;
    }
    if (*ws_bytes < sizing.off) return TT_E_WORKSPACE;
    if (!d_run_offsets || !d_status || (n_raw && (!d_raw || !d_out || !d_slice_offsets)) || (n_samples_total && !d_samples))
        return TT_E_INVAL;
    if (((uintptr_t)d_ws & 255) || ((uintptr_t)d_raw & 15) || ((uintptr_t)d_out & 15) || ((uintptr_t)d_samples & 1)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const uint32_t n_keys = n_slices * n_pmt;
    if (n_raw == 0) {
        TT_CUDA_OK(cudaMemsetAsync(d_run_offsets, 0, ((size_t)n_keys + 1) * sizeof(uint32_t), s));
        return TT_OK;
    }
    Arena a(d_ws);
    prep_plan(a, n_raw, plan);
    const uint32_t nb = div_up(n_raw, 256);
    prof_mark(s, "prep.extract");
    TT_K(prep_extract_kernel)<<<nb, 256, 0, s>>>((const uint4*)d_raw, n_raw, d_slice_offsets, n_slices, n_pmt, plan.rp.keys0,
                                                plan.rp.idx0, plan.nsamp, plan.rp.st, d_status);
    prof_mark(s, "prep.scan");
    int rc = exclusive_scan_u32(plan.nsamp, plan.nsamp, n_raw, plan.scan_scratch, nullptr, s);
    if (rc != TT_OK) return rc;
    int npass = 0;
    for (uint32_t v = n_keys - 1; v; v >>= 8) ++npass;
    rc = radix_run_passes(plan.rp, n_raw, 0, npass, d_slice_offsets, 1, s);
    if (rc != TT_OK) return rc;
    prof_mark(s, "prep.run_offsets");
    TT_K(prep_runoff_kernel)<<<div_up((uint64_t)n_keys + 1, 256), 256, 0, s>>>(plan.rp.keys0, plan.rp.keys1, plan.rp.st, n_raw,
                                                                            n_keys, d_run_offsets);
    prof_mark(s, "prep.gather");
    TT_K(prep_gather_kernel)<<<nb, 256, 0, s>>>((const uint4*)d_raw, d_samples, n_samples_total, plan.nsamp, plan.rp.idx0,
                                               plan.rp.idx1, plan.rp.st, n_raw, (uint4*)d_out, d_status);
    prof_end(s);
    TT_LAUNCH_OK();
    return TT_OK;
}
