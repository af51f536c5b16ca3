// select.cu -- stage a3: tiered top-k of Eq. 6 with the protected sink + recent window counted
// inside the budget.  One CTA per (sequence, list) row.
//
// No sort.  Each tier is an exact radix select (11/11/10-bit digits, shared-memory histograms) over the ordered
// uint32 image of max(score, 0); ties at the threshold are admitted in index order through warp ballots; the
// membership set is a bitmask in shared memory (N/8 bytes) and the ascending index list falls out of a prefix
// sum over its popcounts.  The score rows (<= 512 KB) are re-read from L2 a handful of times; HBM sees them once.
#include "kernels.cuh"

#include <climits>

namespace dustin {

namespace {

namespace sel1024 {
#define SEL_NT 1024
#include "select_impl.inl"
#undef SEL_NT
}  // namespace sel1024

}  // namespace

// Shared-memory plan: bitmask (max_ctx / 8 bytes) + kBins * R histogram counters + a 2 * cap word candidate list,
// shrunk for very long rows so that everything fits the 227 KB of one SM.
void select_plan(int max_ctx, int* mask_words, int* replicas, int* list_cap) {
    // + 1024 words of padding: the sampled path reads the words of a whole 32768-element chunk past the row's end
    *mask_words = (((max_ctx + 31) / 32 + 3) & ~3) + 1024;
    const size_t mask_bytes = (size_t)*mask_words * 4;
    int R = 8, cap = 8192;
    if (mask_bytes > 64 * 1024) R = 4, cap = 4096;   // rows beyond 512k tokens
    *replicas = R;
    *list_cap = cap;
}

size_t select_smem_bytes(int max_ctx) {
    int mw, R, cap;
    select_plan(max_ctx, &mw, &R, &cap);
    return ((size_t)mw + (size_t)sel1024::kBins * R + 2 * (size_t)cap) * 4;
}


cudaError_t launch_select(const SelectParams& p_in, cudaStream_t stream) {
    SelectParams p = p_in;
    select_plan(p.max_ctx, &p.mask_words, &p.replicas, &p.list_cap);
    const size_t smem = select_smem_bytes(p.max_ctx);
    const bool vec = (p.max_ctx & 3) == 0 && (((uintptr_t)p.s_draft | (uintptr_t)p.s_target) & 15) == 0 &&
                     (p.draft_batch_stride & 3) == 0 && (p.draft_list_stride & 3) == 0;
    static bool attr_done = false;
    if (!attr_done) {
        cudaFuncAttributes fa;
        cudaError_t e = cudaFuncGetAttributes(&fa, sel1024::select_kernel<true>);
        if (e != cudaSuccess) return e;
        const int max_smem = 227 * 1024 - (int)fa.sharedSizeBytes;   // opt-in limit counts static shared memory too
        e = cudaFuncSetAttribute(sel1024::select_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(sel1024::select_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    ProfScope prof(kKernSelect, stream);
    if (vec)
        return launch_pdl(sel1024::select_kernel<true>, dim3(p.n_lists, p.batch), dim3(sel1024::kSelThreads), smem, stream, p);
    return launch_pdl(sel1024::select_kernel<false>, dim3(p.n_lists, p.batch), dim3(sel1024::kSelThreads), smem, stream, p);
}

}  // namespace dustin
