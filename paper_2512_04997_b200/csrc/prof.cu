// Optional per-kernel timing with CUDA events on the launching stream, and the launch counter.
// Off by default; bench.py switches it on to report the roofline of the dominant kernel measured
// inside the timed region (include/ledds.h: ledds_profile, ledds_profile_read, ledds_launch_count).
// The records are process-wide host state guarded by one mutex; the counter is atomic.
#include <atomic>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace {
struct Pair { cudaEvent_t a, b; };
std::mutex g_mu;
bool g_on = false;
std::vector<Pair> g_pairs[LEDDS_K_COUNT];
bool g_open[LEDDS_K_COUNT] = {};          // a start without its stop yet: only then may stop record
std::vector<cudaEvent_t> g_pool;
std::atomic<unsigned long long> g_launches{0};
const size_t kMaxPairs = 1 << 16;

cudaEvent_t get_event()
{
    cudaEvent_t e;
    if (!g_pool.empty()) { e = g_pool.back(); g_pool.pop_back(); return e; }
    cudaEventCreate(&e);
    return e;
}
}  // namespace

int ledds_sm_count()
{
    static std::atomic<int> cached{0};
    int n = cached.load(std::memory_order_relaxed);
    if (n > 0) return n;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1)
        n = 148;                                              // B200
    cached.store(n, std::memory_order_relaxed);
    return n;
}

void ledds_count_launch(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

void ledds_prof_start(int k, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_on || g_pairs[k].size() >= kMaxPairs) return;       // full: this group is not recorded (stop sees !g_open)
    Pair p{get_event(), get_event()};
    cudaEventRecord(p.a, st);
    g_pairs[k].push_back(p);
    g_open[k] = true;
}

void ledds_prof_stop(int k, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_on || !g_open[k]) return;
    cudaEventRecord(g_pairs[k].back().b, st);
    g_open[k] = false;
}

extern "C" int ledds_profile(int enable)
{
    std::lock_guard<std::mutex> lock(g_mu);
    for (int k = 0; k < LEDDS_K_COUNT; ++k) {
        for (Pair& p : g_pairs[k]) { g_pool.push_back(p.a); g_pool.push_back(p.b); }
        g_pairs[k].clear();
        g_open[k] = false;
    }
    g_on = enable != 0;
    return LEDDS_OK;
}

extern "C" int ledds_profile_read(int kernel_id, double* total_ms, int* launches)
{
    if (kernel_id < 0 || kernel_id >= LEDDS_K_COUNT) return LEDDS_EINVAL;
    std::lock_guard<std::mutex> lock(g_mu);
    double ms = 0.0;
    int n = 0;
    for (size_t i = 0; i < g_pairs[kernel_id].size(); ++i) {
        if (g_open[kernel_id] && i + 1 == g_pairs[kernel_id].size()) break;   // a group still open has no end event
        Pair& p = g_pairs[kernel_id][i];
        if (cudaEventSynchronize(p.b) != cudaSuccess) return LEDDS_ECUDA;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, p.a, p.b) != cudaSuccess) return LEDDS_ECUDA;
        ms += t;
        ++n;
    }
    if (total_ms) *total_ms = ms;
    if (launches) *launches = n;
    return LEDDS_OK;
}

extern "C" unsigned long long ledds_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
