// select.cu -- stage a3: tiered top-k of Eq. 6 with the protected sink + recent window counted
// inside the budget.  One CTA per (sequence, list) row.
//
// No sort.  Each tier is an exact selection over the ordered uint32 image of max(score, 0): a sampled threshold cuts
// the row down to a short candidate list, an offset-radix select on that list finds the threshold key, ties at the
// threshold are admitted in index order; rare shapes take a full 11/11/10-bit radix select.  The membership set is a
// bitmask in shared memory (N/8 bytes) and the ascending index list falls out of a prefix sum over its popcounts.
// The score rows (<= 512 KB) are re-read from L2 a handful of times; HBM sees them once.
//
// The fused entry point splits the stage in two launches (select_impl.inl, MODE): the draft tier, which depends on
// nothing that stage a1 produces, runs on a few SMs UNDER a1's K stream; only the target tier and the list emission
// remain on the critical path after a1.
#include "kernels.cuh"

#include "../../include/dustin_debug.h"

#include <climits>

namespace dustin {

namespace {

namespace sel1024 {
#define SEL_NT 1024
#include "select_impl.inl"
#undef SEL_NT
}  // namespace sel1024

// The draft-tier kernel of the fused call when many rows are in flight: 256 threads, so that one of its CTAs shares an
// SM with two CTAs of the scoring kernel and ALL rows are in flight at once (beside the saturating K stream every memory
// round trip of the selection takes several microseconds: rows in parallel hide that, more threads per row do not).
namespace sel256 {
#define SEL_NT 256
#include "select_impl.inl"
#undef SEL_NT
}  // namespace sel256

// The target tier when there are more rows than SMs but at most twice as many (the paged ragged workload: 256 rows): 512
// threads, two CTAs per SM, so that all rows run in ONE wave instead of a full wave and a straggling one.
namespace sel512 {
#define SEL_NT 512
#include "select_impl.inl"
#undef SEL_NT
}  // namespace sel512

// Shared-memory plan: bitmask (max_ctx / 8 bytes) + kBins * R histogram counters + a 2 * cap word candidate list,
// shrunk for very long rows so that everything fits the 227 KB of one SM.  light: the 256-thread draft-tier kernel
// (one histogram replica: ~90 KB at 32k tokens, beside two scoring CTAs of 64 KB).
void select_plan(int max_ctx, bool light, int* mask_words, int* replicas, int* list_cap) {
    // + 1024 words of padding: the sampled path reads the words of a whole 32768-element chunk past the row's end
    *mask_words = (int)select_mask_words(max_ctx) + 1024;
    const size_t mask_bytes = (size_t)*mask_words * 4;
    int R = 8, cap = 8192;
    if (mask_bytes > 64 * 1024) R = 4, cap = 4096;   // rows beyond 512k tokens
    if (light) R = 1;
    *replicas = R;
    *list_cap = cap;
}

size_t select_smem_bytes(int max_ctx, bool light) {
    int mw, R, cap;
    select_plan(max_ctx, light, &mw, &R, &cap);
    return ((size_t)mw + (size_t)sel1024::kBins * R + 2 * (size_t)cap) * 4;
}

// Opt the kernel in to the whole 227 KB of shared memory (the limit counts its static shared memory too), once per
// device.
template <auto Kern>   // the kernel itself, not its type: two kernels of one signature must not share the statics
cudaError_t raise_smem_limit() {
    static DeviceOnce once;
    static const int static_bytes = [] {
        cudaFuncAttributes fa;
        return cudaFuncGetAttributes(&fa, Kern) == cudaSuccess ? (int)fa.sharedSizeBytes : -1;
    }();
    if (static_bytes < 0) return cudaErrorUnknown;
    return ensure_dyn_smem(reinterpret_cast<const void*>(Kern), 227 * 1024 - static_bytes, once);
}

template <auto Kern>
cudaError_t launch_one(const SelectParams& p, dim3 grid, int threads, size_t smem, int kid, cudaStream_t stream) {
    const cudaError_t e = raise_smem_limit<Kern>();
    if (e != cudaSuccess) return e;
    ProfScope prof(kid, stream);
    return launch_pdl(Kern, grid, dim3(threads), smem, stream, p);
}

}  // namespace

cudaError_t launch_scan_test(int threads, int n_blocks, const uint32_t* in, uint32_t* out, uint32_t* total,
                             cudaStream_t stream) {
    if (threads == 256) sel256::scan_test_kernel<<<n_blocks, 256, 0, stream>>>(in, out, total);
    else if (threads == 512) sel512::scan_test_kernel<<<n_blocks, 512, 0, stream>>>(in, out, total);
    else if (threads == 1024) sel1024::scan_test_kernel<<<n_blocks, 1024, 0, stream>>>(in, out, total);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

size_t select_mask_words(int max_ctx) { return (size_t)(((max_ctx + 31) / 32 + 3) & ~3); }

cudaError_t launch_select(const SelectParams& p_in, cudaStream_t stream, int mode) {
    SelectParams p = p_in;
    // Draft tier alone (fused call): it runs beside the scoring kernel.  With many rows, one 256-thread CTA per row: every
    // row is in flight at once and a CTA leaves room for two scoring CTAs on its SM (measured: CTAs of that footprint cost
    // a1 ~1 us of 171; so do up to 32 whole SMs taken away).  With few rows, the fast 1024-thread kernel, one SM per row.
    const int n_rows = p.n_lists * p.batch;
    // (up to 32 SMs given up cost the scoring kernel 1-2 us; 48 cost it 13)
    const int sms = device_sm_count();
    const bool half = mode == 2 && n_rows > sms && n_rows <= 2 * sms && p.max_ctx <= (1 << 18) &&
                      knob(DUSTIN_KNOB_SELECT_SPLIT) != 1;
    const bool vec = (p.max_ctx & 3) == 0 && (((uintptr_t)p.s_draft | (uintptr_t)p.s_target) & 15) == 0 &&
                     (p.draft_batch_stride & 3) == 0 && (p.draft_list_stride & 3) == 0;
    // The light plan (one histogram replica) belongs to the small-CTA kernels only: the 512-thread target tier exists in
    // its vectorised form alone, so an unaligned row falls back to the 1024-thread kernel WITH the full plan.
    const bool light = (mode == 1 && n_rows > 32 && p.max_ctx <= (1 << 18)) || (half && vec);
    select_plan(p.max_ctx, light, &p.mask_words, &p.replicas, &p.list_cap);
    const size_t smem = select_smem_bytes(p.max_ctx, light);
    p.trace = nullptr;
    if (knob(DUSTIN_KNOB_SELECT_TRACE)) {
        size_t bytes = 0;
        void* buf = trace_buffer(&bytes);
        if (buf && bytes >= 2 * (size_t)n_rows * 64 * sizeof(unsigned long long))
            p.trace = static_cast<unsigned long long*>(buf);
    }
    using namespace sel1024;
    const dim3 rows(p.n_lists, p.batch);
    if (mode == 1) {
        // grid.x CTAs walk the rows blockIdx.x, blockIdx.x + gridDim.x, ...: here one row each
        // Fewer CTAs than rows when the scoring kernel beside it runs long enough (api.cu): the scoring kernel can only
        // start once EVERY CTA of this grid has started, and at the end of the previous layer's attention kernel only the
        // SMs that kernel left idle can take them early -- 43 CTAs of three rows instead of 128 of one: 224.3 -> 222.7 us
        // per layer at config 3 (six rows: 251 us, the draft tier then outlasts the K stream).
        const int rpc = light && p.draft_rows_per_cta > 1 ? p.draft_rows_per_cta : 1;
        const dim3 flat((n_rows + rpc - 1) / rpc);
        if (light)
            return vec ? launch_one<sel256::select_kernel<true, sel256::kSelDraft>>(p, flat, 256, smem, kKernSelectDraft, stream)
                       : launch_one<sel256::select_kernel<false, sel256::kSelDraft>>(p, flat, 256, smem, kKernSelectDraft, stream);
        return vec ? launch_one<select_kernel<true, kSelDraft>>(p, flat, 1024, smem, kKernSelectDraft, stream)
                   : launch_one<select_kernel<false, kSelDraft>>(p, flat, 1024, smem, kKernSelectDraft, stream);
    }
    if (mode == 2 && half && vec)
        return launch_one<sel512::select_kernel<true, sel512::kSelTarget>>(p, rows, 512, smem, kKernSelect, stream);
    if (mode == 2)
        return vec ? launch_one<select_kernel<true, kSelTarget>>(p, rows, 1024, smem, kKernSelect, stream)
                   : launch_one<select_kernel<false, kSelTarget>>(p, rows, 1024, smem, kKernSelect, stream);
    return vec ? launch_one<select_kernel<true, kSelBoth>>(p, rows, 1024, smem, kKernSelect, stream)
               : launch_one<select_kernel<false, kSelBoth>>(p, rows, 1024, smem, kKernSelect, stream);
}

}  // namespace dustin
