// Optional per-kernel timing with CUDA events on the launching stream, and the launch counter.
// Off by default; bench.py switches it on to report the roofline of the dominant kernel measured
// inside the timed region (include/ledds.h: ledds_profile, ledds_profile_read, ledds_launch_count).
#include <vector>

#include "common.cuh"

namespace {
struct Pair { cudaEvent_t a, b; };
bool g_on = false;
std::vector<Pair> g_pairs[LEDDS_K_COUNT];
std::vector<cudaEvent_t> g_pool;
unsigned long long g_launches = 0;
const size_t kMaxPairs = 1 << 16;

cudaEvent_t get_event()
{
    cudaEvent_t e;
    if (!g_pool.empty()) { e = g_pool.back(); g_pool.pop_back(); return e; }
    cudaEventCreate(&e);
    return e;
}
}  // namespace

void ledds_count_launch(int n) { g_launches += (unsigned long long)n; }

void ledds_prof_start(int k, cudaStream_t st)
{
    if (!g_on || g_pairs[k].size() >= kMaxPairs) return;
    Pair p{get_event(), get_event()};
    cudaEventRecord(p.a, st);
    g_pairs[k].push_back(p);
}

void ledds_prof_stop(int k, cudaStream_t st)
{
    if (!g_on || g_pairs[k].empty() || g_pairs[k].size() > kMaxPairs) return;
    cudaEventRecord(g_pairs[k].back().b, st);
}

extern "C" int ledds_profile(int enable)
{
    for (int k = 0; k < LEDDS_K_COUNT; ++k) {
        for (Pair& p : g_pairs[k]) { g_pool.push_back(p.a); g_pool.push_back(p.b); }
        g_pairs[k].clear();
    }
    g_on = enable != 0;
    return LEDDS_OK;
}

extern "C" int ledds_profile_read(int kernel_id, double* total_ms, int* launches)
{
    if (kernel_id < 0 || kernel_id >= LEDDS_K_COUNT) return LEDDS_EINVAL;
    double ms = 0.0;
    for (Pair& p : g_pairs[kernel_id]) {
        if (cudaEventSynchronize(p.b) != cudaSuccess) return LEDDS_ECUDA;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, p.a, p.b) != cudaSuccess) return LEDDS_ECUDA;
        ms += t;
    }
    if (total_ms) *total_ms = ms;
    if (launches) *launches = (int)g_pairs[kernel_id].size();
    return LEDDS_OK;
}

extern "C" unsigned long long ledds_launch_count(void) { return g_launches; }
