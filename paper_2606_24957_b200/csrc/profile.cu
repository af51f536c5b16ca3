// profile.cu -- host-side bookkeeping shared by the launchers (everything behind include/dustin_debug.h):
//   * a process-wide launch counter and, when switched on by dustin_profile_enable(), one CUDA event pair around every
//     kernel launch on the launching stream (measurement aid of bench.py; off by default);
//   * the tuning knobs of dustin_debug.h (atomics; the library reads no environment variable);
//   * per-device caches: SM count, "dynamic shared memory attribute already raised on this device".
#include "kernels.cuh"

#include "../../include/dustin_debug.h"

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
                                        "fuse_kernel", "select_kernel", "attn_kernel", "select_draft_kernel",
                                        "arr_kernel", "append_kernel", "select_cluster_kernel", "quest_build_kernel",
                                        "quest_score_kernel", "quest_normalize_kernel"};
static_assert(kKernCount == DUSTIN_N_KERNELS, "dustin_debug.h and kernels.cuh disagree on the kernel count");
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

// ---- knobs (dustin_debug.h) ---------------------------------------------------------------------------------------
namespace {
constexpr int kKnobDefaults[DUSTIN_KNOB_COUNT] = {/*PDL*/ 1, /*FUSED_ROWS*/ 1, /*ATTN_TRACE*/ 0, /*SELECT_SPLIT*/ 0,
                                                  /*DRAFT_HOIST*/ 1, /*SCORE_CHUNK*/ 0, /*SELECT_TRACE*/ 0, /*L2_HYGIENE*/ 1};
std::atomic<int> g_knob[DUSTIN_KNOB_COUNT];
std::atomic<bool> g_knob_set[DUSTIN_KNOB_COUNT];
std::atomic<void*> g_trace_ptr{nullptr};
std::atomic<size_t> g_trace_bytes{0};
}  // namespace

int knob(int id) {
    if (id < 0 || id >= DUSTIN_KNOB_COUNT) return 0;
    return g_knob_set[id].load(std::memory_order_relaxed) ? g_knob[id].load(std::memory_order_relaxed) : kKnobDefaults[id];
}
void knob_set(int id, int value) {
    if (id < 0 || id >= DUSTIN_KNOB_COUNT) return;
    g_knob[id].store(value, std::memory_order_relaxed);
    g_knob_set[id].store(true, std::memory_order_relaxed);
}
void trace_buffer_set(void* p, size_t bytes) {
    g_trace_bytes.store(p ? bytes : 0, std::memory_order_relaxed);
    g_trace_ptr.store(p, std::memory_order_relaxed);
}
void* trace_buffer(size_t* bytes) {
    *bytes = g_trace_bytes.load(std::memory_order_relaxed);
    return g_trace_ptr.load(std::memory_order_relaxed);
}

bool pdl_enabled() { return knob(DUSTIN_KNOB_PDL) != 0; }

// ---- per-device caches ----------------------------------------------------------------------------------------------
namespace {
constexpr int kMaxDev = 64;
std::atomic<int> g_sm_count[kMaxDev];
}  // namespace

int current_device() {
    int dev = 0;
    return cudaGetDevice(&dev) == cudaSuccess ? dev : 0;
}

int device_sm_count() {
    const int dev = current_device();
    if (dev >= 0 && dev < kMaxDev) {
        const int c = g_sm_count[dev].load(std::memory_order_relaxed);
        if (c > 0) return c;
    }
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;   // B200
    if (dev >= 0 && dev < kMaxDev) g_sm_count[dev].store(v, std::memory_order_relaxed);
    return v;
}

cudaError_t ensure_dyn_smem(const void* func, int bytes, DeviceOnce& once) {
    const int dev = current_device();
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && (once.done.load(std::memory_order_acquire) >> dev) & 1ull) return cudaSuccess;
    // Racing first calls both set the same value: harmless.  The attribute is per device (and context).
    const cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && tracked) once.done.fetch_or(1ull << dev, std::memory_order_release);
    return e;
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
