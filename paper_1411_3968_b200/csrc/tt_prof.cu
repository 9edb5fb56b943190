// tt_prof.cu -- kernel-launch counter and an optional per-stage CUDA-event profiler.
// Off by default (one branch per mark).  When enabled, every stage boundary inside the three hot
// calls records a cudaEvent on the caller's stream; tt_prof_read sums the elapsed time per stage
// name.  Used by bench.py for the roofline line (per-kernel device time inside the timed region).
#include <atomic>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "tt_common.cuh"

namespace tt {
static std::atomic<uint64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

struct Mark {
    cudaEvent_t ev;
    const char* name;  // nullptr = end mark
};
static bool g_on = false;
static std::vector<Mark> g_marks;
static std::vector<cudaEvent_t> g_pool;
static size_t g_used = 0;
constexpr size_t kMaxMarks = 1 << 16;

static void mark(cudaStream_t s, const char* name) {
    if (!g_on || g_used >= kMaxMarks) return;
    if (g_used == g_pool.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return;
        g_pool.push_back(e);
    }
    cudaEvent_t e = g_pool[g_used++];
    cudaEventRecord(e, s);
    g_marks.push_back({e, name});
}
void prof_mark(cudaStream_t s, const char* name) { mark(s, name); }

// device counters sampled while profiling: copied to pinned host memory on the caller's stream
struct Counter {
    const char* name;
    uint32_t* host;  // pinned
};
static std::vector<Counter> g_counters;
// pinned slots are pooled and reused from one profiled pass to the next: cudaMallocHost is a slow, synchronous host call,
// and one per sample showed up as device idle time in whatever stage was open (bench.py, small configs)
static std::vector<uint32_t*> g_pinned;
void prof_counter(cudaStream_t s, const char* name, const uint32_t* d_value) {
    if (!g_on || g_counters.size() >= 4096) return;
    if (g_counters.size() == g_pinned.size()) {
        uint32_t* h = nullptr;
        if (cudaMallocHost(&h, sizeof(uint32_t)) != cudaSuccess) return;
        g_pinned.push_back(h);
    }
    uint32_t* h = g_pinned[g_counters.size()];
    *h = 0;
    cudaMemcpyAsync(h, d_value, sizeof(uint32_t), cudaMemcpyDeviceToHost, s);
    g_counters.push_back({name, h});
}
void prof_end(cudaStream_t s) { mark(s, nullptr); }
}  // namespace tt

extern "C" uint64_t tt_launch_count(void) { return tt::g_launches.load(); }

extern "C" int tt_prof_enable(int on) {
    tt::g_on = on != 0;
    tt::g_marks.clear();
    tt::g_used = 0;
    tt::g_counters.clear();  // the pinned slots stay in the pool
    return TT_OK;
}

// Writes "name ms count\n" lines (summed over everything recorded since tt_prof_enable) into buf.
// The caller must have synchronised the stream(s).  Returns the number of bytes written, or < 0.
extern "C" int tt_prof_read(char* buf, size_t cap) {
    using namespace tt;
    std::vector<std::string> names;
    std::vector<double> ms;
    std::vector<uint64_t> cnt;
    for (size_t k = 0; k + 1 < g_marks.size(); ++k) {
        if (!g_marks[k].name) continue;
        float t = 0;
        if (cudaEventElapsedTime(&t, g_marks[k].ev, g_marks[k + 1].ev) != cudaSuccess) {
            (void)cudaGetLastError();
            return TT_E_CUDA;
        }
        size_t j = 0;
        for (; j < names.size(); ++j)
            if (names[j] == g_marks[k].name) break;
        if (j == names.size()) { names.push_back(g_marks[k].name); ms.push_back(0); cnt.push_back(0); }
        ms[j] += t;
        cnt[j] += 1;
    }
    for (auto& c : g_counters) {  // counters: "ctr.<name> <sum of values> <samples>"
        const std::string nm = std::string("ctr.") + c.name;
        size_t j = 0;
        for (; j < names.size(); ++j)
            if (names[j] == nm) break;
        if (j == names.size()) { names.push_back(nm); ms.push_back(0); cnt.push_back(0); }
        ms[j] += (double)*c.host;
        cnt[j] += 1;
    }
    size_t off = 0;
    for (size_t j = 0; j < names.size(); ++j) {
        int w = std::snprintf(buf + off, off < cap ? cap - off : 0, "%s %.6f %llu\n", names[j].c_str(), ms[j],
                              (unsigned long long)cnt[j]);
        if (w < 0 || off + (size_t)w >= cap) return TT_E_INVAL;
        off += (size_t)w;
    }
    return (int)off;
}
