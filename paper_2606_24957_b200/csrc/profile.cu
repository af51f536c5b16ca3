// profile.cu -- launch bookkeeping: a process-wide launch counter and, when switched on by
// dustin_profile_enable(), one CUDA event pair around every kernel launch on the launching stream
// (measurement aid of bench.py; off by default, nothing is recorded or synchronised then).
#include "kernels.cuh"

#include <atomic>
#include <cstdlib>
#include <mutex>
#include <vector>

namespace dustin {

namespace {
std::atomic<unsigned long long> g_launches{0};
std::atomic<bool> g_on{false};
std::mutex g_mu;
struct Rec {
    int kid;
    cudaEvent_t a, b;
};
std::vector<Rec> g_recs;                 // recorded pairs of the current collection
std::vector<cudaEvent_t> g_free;         // recycled events
cudaEvent_t take_event() {
    if (!g_free.empty()) {
        cudaEvent_t e = g_free.back();
        g_free.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
const char* const kNames[kKernCount] = {"score_logits_kernel", "score_stats_kernel", "score_normalize_kernel",
                                        "fuse_kernel", "select_kernel", "attn_kernel", "attn_combine_kernel",
                                        "arr_kernel", "append_kernel"};
}  // namespace

ProfScope::ProfScope(int kid, cudaStream_t stream) : kid_(kid), stream_(stream), slot_(-1) {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (!g_on.load(std::memory_order_relaxed)) return;
    std::lock_guard<std::mutex> lk(g_mu);
    Rec r{kid, take_event(), take_event()};
    if (!r.a || !r.b) return;
    cudaEventRecord(r.a, stream);
    g_recs.push_back(r);
    slot_ = (long long)g_recs.size() - 1;
}

ProfScope::~ProfScope() {
    if (slot_ < 0) return;
    std::lock_guard<std::mutex> lk(g_mu);
    if (slot_ < (long long)g_recs.size()) cudaEventRecord(g_recs[slot_].b, stream_);
}

bool pdl_enabled() {
    static const bool on = [] {
        const char* e = getenv("DUSTIN_PDL");
        return !(e && e[0] == '0');
    }();
    return on;
}

unsigned long long prof_launch_count() { return g_launches.load(std::memory_order_relaxed); }

void prof_enable(bool on) {
    std::lock_guard<std::mutex> lk(g_mu);
    for (const Rec& r : g_recs) {
        g_free.push_back(r.a);
        g_free.push_back(r.b);
    }
    g_recs.clear();
    g_on.store(on, std::memory_order_relaxed);
}

cudaError_t prof_collect(double* ms_out, long long* launches_out) {
    std::lock_guard<std::mutex> lk(g_mu);
    for (int i = 0; i < kKernCount; ++i) {
        ms_out[i] = 0.0;
        launches_out[i] = 0;
    }
    cudaError_t err = cudaSuccess;
    for (const Rec& r : g_recs) {
        cudaError_t e = cudaEventSynchronize(r.b);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.a, r.b);
        if (e != cudaSuccess) {
            err = e;
            continue;
        }
        ms_out[r.kid] += ms;
        launches_out[r.kid] += 1;
    }
    for (const Rec& r : g_recs) {
        g_free.push_back(r.a);
        g_free.push_back(r.b);
    }
    g_recs.clear();
    return err;
}

const char* prof_kernel_name(int kid) { return kid >= 0 && kid < kKernCount ? kNames[kid] : nullptr; }

}  // namespace dustin
