// common.cuh -- device helpers shared by the sm_100a kernels of the Dustin sparse-verification path.
// (CUDA path only; the CPU oracle under oracle/ shares nothing with this tree.)
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dustin.h"

namespace dustin {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

// Device view of dustin_kv_t (strides in elements).
struct KvView {
    const __nv_bfloat16* k;
    const __nv_bfloat16* v;
    long long stride_seq, stride_token, stride_head;
    const int* page_table;
    int page_size, max_pages;
    int page_shift;   // log2(page_size) when it is a power of two (the usual case: shift and mask, no division), else -1
    const int* seq_lens;
};

__device__ __forceinline__ int seq_len_of(const int* seq_lens, int b, int max_ctx) {
    if (seq_lens == nullptr) return max_ctx;
    int n = seq_lens[b];
    return n < 0 ? 0 : (n > max_ctx ? max_ctx : n);
}

// Element offset of cache row (b, n, g).
__device__ __forceinline__ long long kv_row_offset(const KvView& kv, int b, int n, int g) {
    if (kv.page_table == nullptr)
        return (long long)b * kv.stride_seq + (long long)n * kv.stride_token + (long long)g * kv.stride_head;
    const int pg = kv.page_shift >= 0 ? n >> kv.page_shift : n / kv.page_size;
    const int page = __ldg(kv.page_table + (long long)b * kv.max_pages + pg);
    return (long long)page * kv.stride_seq + (long long)(n - pg * kv.page_size) * kv.stride_token +
           (long long)g * kv.stride_head;
}

// ---- memory -------------------------------------------------------------------------------------------------
// The 128-byte line at p (aligned) is no longer needed: L2 may drop it without writing it back.  Its content is
// undefined afterwards.
__device__ __forceinline__ void l2_discard128(const void* p) {
    asm volatile("discard.global.L2 [%0], 128;" ::"l"(p) : "memory");
}

// 16-byte streaming load that does not pollute L1 (the K stream is read exactly once).
__device__ __forceinline__ uint4 ldg_stream16(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// cp.async 16 B global -> shared, bypassing L1; src_bytes = 0 zero-fills the destination.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
// The same with an L2 eviction-priority hint (createpolicy): a stream that is read exactly once is marked evict_first so
// that it does not push the small L2-resident working set of the other stages (scores, lists, masks) out to DRAM.
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void cp_async16_hint(uint32_t dst, const void* src, int src_bytes, uint64_t policy) {
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(dst), "l"(src), "r"(src_bytes),
                 "l"(policy)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// ---- tensor-core fragments (warp-level mma.sync; see DESIGN.md §5 for why not tcgen05 on this path) ----------
__device__ __forceinline__ void ldmatrix_x4(uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3, uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3,
                                                  uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
// D(16x8,f32) += A(16x16,bf16,row) * B(16x8,bf16,col)
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&t);
}

__device__ __forceinline__ float fast_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- programmatic dependent launch (PDL) ---------------------------------------------------------------------------
// The three kernels of a layer are launched with the programmatic-stream-serialization attribute: a kernel may start
// while its predecessor drains, runs its prologue (barrier init, TMEM allocation, index math on parameters), and calls
// pdl_wait() BEFORE its first access to global memory -- the wait returns once the predecessor grid has completed and
// its writes are visible.  pdl_trigger() at the end of a CTA's work lets the successor's CTAs be scheduled as soon
// as every CTA of this grid has got that far.  Both are no-ops when the kernel was launched the ordinary way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- softmax bookkeeping of stage a1 (shared by score.cu and the row materialisation inside select.cu; explicit
// fma / mul intrinsics so that both compile to the same arithmetic, bit for bit) ----------------------------------
// Merge (om, os) into the running (m, s): maxima and sums of exp2(l - max) in the log2 domain.
__device__ __forceinline__ void softmax_merge(float& m, float& s, float om, float os) {
    const float mn = fmaxf(m, om);
    s = (mn > -INFINITY) ? __fmaf_rn(s, exp2f(m - mn), __fmul_rn(os, exp2f(om - mn))) : 0.f;
    m = mn;
}
// (M, 1/Z) of one head from its n_chunks per-CTA partials; one warp, every lane receives the result.
__device__ __forceinline__ float2 fold_stats_warp(const float2* __restrict__ src, int n_chunks, int lane) {
    float m = -INFINITY, s = 0.f;
    for (int i0 = lane; i0 < n_chunks; i0 += 32 * 8) {   // eight loads in flight, merged in index order
        float2 o[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) o[u] = i0 + 32 * u < n_chunks ? __ldcg(src + i0 + 32 * u) : make_float2(-INFINITY, 0.f);
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (i0 + 32 * u < n_chunks) softmax_merge(m, s, o[u].x, o[u].y);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const float om = __shfl_xor_sync(0xffffffffu, m, off), os = __shfl_xor_sync(0xffffffffu, s, off);
        softmax_merge(m, s, om, os);
    }
    return make_float2(m, s > 0.f ? 1.f / s : 0.f);
}
// a += exp2(l - M) / Z for the four logits of one 16-byte load.
__device__ __forceinline__ void prob_accumulate4(float (&a)[4], const float4 l, const float2 st) {
    a[0] = __fmaf_rn(exp2f(l.x - st.x), st.y, a[0]);
    a[1] = __fmaf_rn(exp2f(l.y - st.x), st.y, a[1]);
    a[2] = __fmaf_rn(exp2f(l.z - st.x), st.y, a[2]);
    a[3] = __fmaf_rn(exp2f(l.w - st.x), st.y, a[3]);
}

// Host side: kernel launch with the PDL attribute (DUSTIN_PDL=0 in the environment: ordinary launches).
bool pdl_enabled();
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                              Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

}  // namespace dustin
