// tt_api.cu -- geometry handle, tt_sort_slice dispatch, version.
#include <cstdlib>
#include <cstring>
#include <vector>

#include <mutex>

#include "tt_merge.cuh"

namespace tt {
size_t radix_ws_bytes(uint32_t n);
int radix_sort(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
               uint32_t n_seg, void* d_ws, cudaStream_t s);

constexpr int kMaxDev = 64;
static std::mutex g_dev_mu;
static uint32_t g_done[kMaxDev];
static int g_sms[kMaxDev];

int once_per_device(int slot, int (*fn)()) {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess) return TT_E_CUDA;
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (d >= 0 && d < kMaxDev && ((g_done[d] >> slot) & 1u)) return TT_OK;
    const int rc = fn();
    if (rc == TT_OK && d >= 0 && d < kMaxDev) g_done[d] |= 1u << slot;
    return rc;
}

int sm_count() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess) return 148;
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (d >= 0 && d < kMaxDev && g_sms[d] > 0) return g_sms[d];
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, d) != cudaSuccess || v <= 0) v = 148;
    if (d >= 0 && d < kMaxDev) g_sms[d] = v;
    return v;
}
}  // namespace tt
using namespace tt;

extern "C" const char* tt_version(void) { return "libtt 0.1 (sm_100a) " __DATE__; }

extern "C" int tt_geometry_create(tt_geometry** out, uint32_t n_pmt, uint32_t n_tower, uint32_t ppt,
                                  const int32_t* h_pair_block, const int32_t* h_blocks, uint32_t n_blocks) {
    if (!out || !h_pair_block || !h_blocks || n_tower == 0 || ppt == 0 || n_blocks == 0) return TT_E_INVAL;
    if ((uint64_t)n_tower * ppt != n_pmt || n_pmt > 65536) return TT_E_INVAL;
    const size_t bs = (size_t)ppt * ppt;
    int32_t max_dt = -1;
    for (size_t ta = 0; ta < n_tower; ++ta)
        for (size_t tb = 0; tb < n_tower; ++tb) {
            const int32_t ab = h_pair_block[ta * n_tower + tb], ba = h_pair_block[tb * n_tower + ta];
            if (ab >= (int32_t)n_blocks || ba >= (int32_t)n_blocks) return TT_E_INVAL;
            if ((ab < 0) != (ba < 0)) return TT_E_INVAL;
            if (ab < 0 || tb < ta) continue;
            // symmetry: block(ta,tb)[i][j] == block(tb,ta)[j][i]
            const int32_t* A = h_blocks + (size_t)ab * bs;
            const int32_t* B = h_blocks + (size_t)ba * bs;
            for (uint32_t i = 0; i < ppt; ++i)
                for (uint32_t j = 0; j < ppt; ++j) {
                    const int32_t v = A[(size_t)i * ppt + j];
                    if (v != B[(size_t)j * ppt + i] || v < -1) return TT_E_INVAL;
                    if (v > max_dt) max_dt = v;
                }
        }
    tt_geometry* g = (tt_geometry*)std::calloc(1, sizeof(tt_geometry));
    if (!g) return TT_E_INVAL;
    const size_t pb_bytes = (size_t)n_tower * n_tower * sizeof(int32_t), bl_bytes = (size_t)n_blocks * bs * sizeof(int32_t);
    if (cudaMalloc(&g->d_pair_block, pb_bytes) != cudaSuccess || cudaMalloc(&g->d_blocks, bl_bytes) != cudaSuccess ||
        cudaMemcpy(g->d_pair_block, h_pair_block, pb_bytes, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(g->d_blocks, h_blocks, bl_bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaFree(g->d_pair_block);
        cudaFree(g->d_blocks);
        std::free(g);
        (void)cudaGetLastError();
        return TT_E_CUDA;
    }
    g->dev.pair_block = g->d_pair_block;
    g->dev.blocks = g->d_blocks;
    g->dev.n_pmt = n_pmt;
    g->dev.n_tower = n_tower;
    g->dev.ppt = ppt;
    g->dev.n_blocks = n_blocks;
    g->dev.max_dt = max_dt;
    *out = g;
    return TT_OK;
}

extern "C" int tt_geometry_destroy(tt_geometry* g) {
    if (!g) return TT_OK;
    cudaFree(g->d_pair_block);
    cudaFree(g->d_blocks);
    std::free(g);
    return TT_OK;
}

static int check_offsets(const uint32_t* h, uint32_t cnt, uint32_t n) {
    if (!h || h[0] != 0 || h[cnt] != n) return TT_E_INVAL;
    for (uint32_t k = 0; k < cnt; ++k)
        if (h[k] > h[k + 1]) return TT_E_INVAL;
    return TT_OK;
}

extern "C" int tt_sort_slice(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n,
                             const uint32_t* d_seg_offsets, const uint32_t* h_seg_offsets, uint32_t n_seg,
                             const uint32_t* d_run_offsets, const uint32_t* h_run_offsets, uint32_t n_runs,
                             void* d_ws, size_t* ws_bytes, int32_t* d_status, void* stream) {
    if (!ws_bytes || n_seg < 1 || n >= 0xFFF00000u) return TT_E_INVAL;
    if (check_offsets(h_seg_offsets, n_seg, n) != TT_OK) return TT_E_INVAL;
    const bool runs = n > 0 && (d_run_offsets != nullptr || h_run_offsets != nullptr);
    if (runs) {
        if (!d_run_offsets || !h_run_offsets || n_runs < 1) return TT_E_INVAL;
        if (check_offsets(h_run_offsets, n_runs, n) != TT_OK) return TT_E_INVAL;
        // runs never straddle a segment: every segment boundary is a run boundary
        uint32_t r = 0;
        for (uint32_t s = 0; s <= n_seg; ++s) {
            while (r < n_runs && h_run_offsets[r] < h_seg_offsets[s]) ++r;
            if (h_run_offsets[r] != h_seg_offsets[s]) return TT_E_INVAL;
        }
    }
    const size_t need = runs ? merge_ws_bytes(n, h_seg_offsets, n_seg, h_run_offsets, n_runs) : radix_ws_bytes(n);
    if (!d_ws) {
        *ws_bytes = need;
        return TT_OK;
    }
    if (*ws_bytes < need) return TT_E_WORKSPACE;
    if (n == 0) return TT_OK;
    if (!d_in || !d_out || !d_seg_offsets || !d_status || d_in == d_out) return TT_E_INVAL;
    if (((uintptr_t)d_ws & 255) || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return TT_E_INVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (runs)
        return merge_sort_runs(d_in, d_out, d_perm, n, d_seg_offsets, h_seg_offsets, n_seg, d_run_offsets, h_run_offsets,
                               n_runs, d_ws, d_status, s, nullptr, nullptr);
    return radix_sort(d_in, d_out, d_perm, n, d_seg_offsets, n_seg, d_ws, s);
}
