// Optional per-kernel-class timing with CUDA events on the launching stream (bench.py's live
// roofline numbers).  Off by default; when off the cost is one branch per launch.
#include <vector>

#include "cbct_internal.h"

namespace {
struct Span { int tag; cudaEvent_t a, b; };
bool g_on = false;
std::vector<Span> g_spans;
std::vector<cudaEvent_t> g_pool;

cudaEvent_t get_event()
{
    if (!g_pool.empty()) { cudaEvent_t e = g_pool.back(); g_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
}  // namespace

bool cbct_profile_is_on() { return g_on; }

ProfileScope::ProfileScope(int tag, cudaStream_t st) : tag_(tag), st_(st), a_(nullptr)
{
    if (!g_on) return;
    a_ = get_event();
    if (a_) cudaEventRecord(a_, st_);
}

ProfileScope::~ProfileScope()
{
    if (!a_) return;
    cudaEvent_t b = get_event();
    if (b) cudaEventRecord(b, st_);
    g_spans.push_back({tag_, a_, b});
}

extern "C" cbct_status cbct_profile_enable(int on)
{
    g_on = on != 0;
    return CBCT_OK;
}

extern "C" cbct_status cbct_profile_read(double *h_ms, unsigned long long *h_count, int reset)
{
    if (!h_ms || !h_count) { cbct_set_error("cbct_profile_read: NULL argument"); return CBCT_ERR_INVALID_ARG; }
    for (int t = 0; t < CBCT_PROFILE_TAGS; ++t) { h_ms[t] = 0.0; h_count[t] = 0; }
    for (const Span &s : g_spans) {
        if (!s.a || !s.b) continue;
        CBCT_CUDA(cudaEventSynchronize(s.b));
        float ms = 0.f;
        CBCT_CUDA(cudaEventElapsedTime(&ms, s.a, s.b));
        h_ms[s.tag] += ms;
        h_count[s.tag] += 1;
    }
    if (reset) {
        for (const Span &s : g_spans) { if (s.a) g_pool.push_back(s.a); if (s.b) g_pool.push_back(s.b); }
        g_spans.clear();
    }
    return CBCT_OK;
}
