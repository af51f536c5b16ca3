// score.cu -- stage a1 (head-subset scoring) and stage a2 (Eq. 5 accumulation,
// PAPER.md:161-164) for sm_100a.
//
// a1 is one streaming read of the K rows of every KV group that holds a subset head (HBM-bound: DESIGN.md §4).
//   score_logits_kernel   every warp streams its 16-token K tiles through a private two-stage cp.async ring in shared
//                         memory (16-byte copies, whole rows per warp instruction, XOR-swizzled) and feeds mma.sync
//                         fragments from it (tokens on M, the <= 8 subset heads of the KV group on N, head_dim on K;
//                         the head_dim axis is permuted identically for both operands so each thread's 16 B feed two
//                         k-steps).  Writes log2-domain logits [B, nsel, N] (L2-resident scratch) and per-CTA
//                         softmax partials (max, sum).
//   score_stats_kernel    folds the partials into (M, 1/Z) per (sequence, head), in a fixed order.
//   score_normalize_kernel p = exp2(l - M) / Z summed over the heads of each list; optionally fused with the
//                         Eq. 5 accumulation into hist (the fused entry point never writes scores_now).
#include "kernels.cuh"

namespace dustin {

namespace {

constexpr int kScoreWarps = 8;
constexpr int kScoreThreads = kScoreWarps * 32;
constexpr int kTileTokens = 16;  // one m16n8k16 M tile

template <int D>
struct KFrag {
    uint4 lo[D / 32];  // row g      : 8 bf16 at dims j*32 + c*8
    uint4 hi[D / 32];  // row g + 8
};

// ---- shared-memory staging of the K stream -----------------------------------------------------------------------
// A warp owns a private ring of kStages tiles (16 tokens x D bf16).  issue_tile requests one tile with fully
// coalesced 16-byte cp.async (a warp instruction covers whole rows: 2 rows x 256 B at D = 128), zero-filling rows past
// N; frag_tile reads the mma A fragments back.  Chunk c of row r sits at chunk c ^ ((r & 1) << 2), which keeps the
// 16-byte fragment reads of the row pairs (g, g + 1) on disjoint banks.  No block-wide barrier anywhere: the ring is
// ordered by cp.async groups and __syncwarp.
constexpr int kStages = 2;

template <int D>
__device__ __forceinline__ void issue_tile(uint32_t stage, const ScoreParams& p, int b, int grp, int n0, int N, int lane,
                                           uint64_t policy) {
    constexpr int CPR = D / 8;              // 16-byte chunks per row
    constexpr int RPI = 32 / CPR;           // rows per warp instruction
    long long my = -1;                      // lanes 0..15: element offset of row n0 + lane (page table resolved once)
    if (lane < kTileTokens && n0 + lane < N) my = kv_row_offset(p.kv, b, n0 + lane, grp);
    const int ch = lane % CPR, r0 = lane / CPR;
#pragma unroll
    for (int i = 0; i < kTileTokens / RPI; ++i) {
        const int row = i * RPI + r0;
        const long long off = __shfl_sync(0xffffffffu, my, row);
        const __nv_bfloat16* src = off >= 0 ? p.kv.k + off + ch * 8 : p.kv.k;
        cp_async16_hint(stage + (uint32_t)row * (D * 2) + (uint32_t)((ch ^ ((row & 1) << 2)) << 4), src, off >= 0 ? 16 : 0,
                        policy);
    }
}

template <int D>
__device__ __forceinline__ void frag_tile(KFrag<D>& f, const unsigned char* stage, int lane) {
    const int g = lane >> 2, c = lane & 3;
    const unsigned char* lo = stage + g * (D * 2);
    const unsigned char* hi = lo + 8 * (D * 2);
    const int sw = (g & 1) << 2;
#pragma unroll
    for (int j = 0; j < D / 32; ++j) {
        f.lo[j] = *reinterpret_cast<const uint4*>(lo + (((4 * j + c) ^ sw) << 4));
        f.hi[j] = *reinterpret_cast<const uint4*>(hi + (((4 * j + c) ^ sw) << 4));
    }
}

// gridDim = (CTAs per sequence, batch).  Warp w serves scored KV group (w % group_slots) and, when fewer than 8 groups
// are scored, every n_sub-th tile: at any moment the warps of a CTA read the SAME tokens' records, each its own
// 256-byte piece.  Each warp streams its tiles through a private two-stage cp.async ring (3 CTAs = 24 warps x 8 KB
// per SM in flight) and feeds mma.sync from shared memory; no block-wide barrier.
template <int D>
__global__ void __launch_bounds__(kScoreThreads, 3) score_logits_kernel(const ScoreParams p) {
    extern __shared__ __align__(128) unsigned char s_ring[];   // [warp][stage][16 tokens][D] bf16
    __shared__ float2 s_part[kScoreWarps][8];                   // per-warp softmax partials of the (<= 8) heads of its group
    const int chunk = blockIdx.x, b = blockIdx.y;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, c = lane & 3;
    // defer_wait (fused call, hoisted draft tier): everything below reads q / K and WRITES the logits scratch without a
    // dependency wait of this kernel's own.  That is safe only because the kernel launched just before this one -- the
    // draft-tier selection (select_impl.inl, select_kernel, kSelDraft) -- executes griddepcontrol.wait BEFORE its
    // launch_dependents: by the time this grid may start, everything older than that kernel (in particular the previous
    // call's attention kernel, whose stream-K scratch overlaps the logits) is complete and visible.  The wait is per
    // waiting grid, so this ordering is transitive, not direct: keep "wait, then trigger" in that kernel
    // (tests/test_gpu_pdl_chain.py runs unsynchronised chains of calls on one workspace against synchronised ones).
    if (!p.defer_wait) pdl_wait();
    const int N = seq_len_of(p.kv.seq_lens, b, p.max_ctx);
    const int slots = p.group_slots, n_sub = kScoreWarps / slots;
    const int ws = warp / slots;                       // which tiles of the range
    // Tiles are dealt round-robin: CTA `chunk` takes the 16-token tiles chunk * n_sub + ws, + gridDim.x * n_sub, ... of the
    // sequence, so at any moment the CTAs of a sequence read ONE contiguous window of the cache.  Contiguous per-CTA
    // ranges put the concurrent streams a fixed stride apart, which loads the DRAM channels unevenly (measured: 174 to
    // 189 us at config 3 depending on that stride).
    // K is read exactly once: evict_first keeps the stream from displacing the logits scratch, the score rows and the
    // selection state that the following kernels (and the draft-tier selection running beside this one) read from L2
    const uint64_t policy = l2_policy_evict_first();
    // Ragged batches: a sequence of N tokens is shared by only as many of its gridDim.x CTAs as it has chunk_tokens-sized
    // pieces (the others find no tile and just leave their empty partials), so that a short sequence does not shrink the
    // work per CTA to a tile or two (measured on the paged ragged workload: 5.0 TB/s against 6.0 contiguous).
    const int n_active = max(1, min((int)gridDim.x, (N + p.chunk_tokens - 1) / p.chunk_tokens));
    const int chunk_lo = chunk * (kScoreWarps / p.group_slots) * kTileTokens;
    const int chunk_hi = chunk < n_active ? N : 0;

    for (int gi = warp % slots; gi < p.n_groups; gi += slots) {
        const int grp = p.group_id[gi], first = p.group_first[gi], nh = p.group_cnt[gi];
        // B fragments: head slot n = g of this KV group (zero beyond the subset), dims j*32 + c*8 .. +8.
        uint4 qf[D / 32];
#pragma unroll
        for (int j = 0; j < D / 32; ++j) qf[j] = make_uint4(0, 0, 0, 0);
        if (g < nh) {
            const __nv_bfloat16* qrow = p.q + (long long)b * p.q_stride_batch + p.sel_qoff[first + g] + c * 8;
#pragma unroll
            for (int j = 0; j < D / 32; ++j) qf[j] = *reinterpret_cast<const uint4*>(qrow + j * 32);
        }

        // this thread's logits: heads 2c, 2c+1 of tokens (g, g+8) of each tile
        float m0 = -INFINITY, m1 = -INFINITY, s0 = 0.f, s1 = 0.f;
        const bool h0 = 2 * c < nh, h1 = 2 * c + 1 < nh;
        float* l0 = p.logits + ((long long)b * p.nsel + first + 2 * c) * p.logit_stride;
        float* l1 = l0 + p.logit_stride;

        // Two tiles are always on their way: tile t + 1 while t is consumed, t + 2 requested as soon as t's fragments are
        // in registers (its stage is free then).
        constexpr int kTileBytes = kTileTokens * D * 2;
        unsigned char* ring = s_ring + warp * (kStages * kTileBytes);
        const uint32_t ring_u32 = smem_u32(ring);
        const int step = n_active * n_sub * kTileTokens;
        int n0 = chunk_lo + ws * kTileTokens;
        __syncwarp();                                        // the previous group's reads of the ring are done
        if (n0 < chunk_hi) issue_tile<D>(ring_u32, p, b, grp, n0, N, lane, policy);
        cp_async_commit();
        if (n0 + step < chunk_hi) issue_tile<D>(ring_u32 + kTileBytes, p, b, grp, n0 + step, N, lane, policy);
        cp_async_commit();
        KFrag<D> cur;
        for (int t = 0; n0 < chunk_hi; n0 += step, ++t) {
            cp_async_wait<1>();                              // tile t has landed (tile t + 1 may still be in flight)
            __syncwarp();
            frag_tile<D>(cur, ring + (t & 1) * kTileBytes, lane);
            __syncwarp();                                    // every lane has read stage t & 1: it can be refilled
            if (n0 + 2 * step < chunk_hi) issue_tile<D>(ring_u32 + (t & 1) * kTileBytes, p, b, grp, n0 + 2 * step, N, lane, policy);
            cp_async_commit();
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int j = 0; j < D / 32; ++j) {
                mma_bf16_16816(acc, cur.lo[j].x, cur.hi[j].x, cur.lo[j].y, cur.hi[j].y, qf[j].x, qf[j].y);
                mma_bf16_16816(acc, cur.lo[j].z, cur.hi[j].z, cur.lo[j].w, cur.hi[j].w, qf[j].z, qf[j].w);
            }
            const int n_lo = n0 + g, n_hi = n0 + g + 8;
            const bool v_lo = n_lo < N, v_hi = n_hi < N;
            const float a0 = v_lo ? acc[0] * p.scale_log2 : -INFINITY;   // (token g    , head 2c  )
            const float a1 = v_lo ? acc[1] * p.scale_log2 : -INFINITY;   // (token g    , head 2c+1)
            const float a2 = v_hi ? acc[2] * p.scale_log2 : -INFINITY;   // (token g + 8, head 2c  )
            const float a3 = v_hi ? acc[3] * p.scale_log2 : -INFINITY;   // (token g + 8, head 2c+1)
            if (h0) {
                if (v_lo) l0[n_lo] = a0;
                if (v_hi) l0[n_hi] = a2;
                const float mn = fmaxf(m0, fmaxf(a0, a2));
                if (mn > -INFINITY) {
                    s0 = s0 * exp2f(m0 - mn) + exp2f(a0 - mn) + exp2f(a2 - mn);
                    m0 = mn;
                }
            }
            if (h1) {
                if (v_lo) l1[n_lo] = a1;
                if (v_hi) l1[n_hi] = a3;
                const float mn = fmaxf(m1, fmaxf(a1, a3));
                if (mn > -INFINITY) {
                    s1 = s1 * exp2f(m1 - mn) + exp2f(a1 - mn) + exp2f(a3 - mn);
                    m1 = mn;
                }
            }
        }

        cp_async_wait<0>();
        // (max, sum) over the 8 lanes that share c (fixed order => deterministic); one partial per (warp, head)
#pragma unroll
        for (int off = 4; off < 32; off <<= 1) {
            const float om0 = __shfl_xor_sync(0xffffffffu, m0, off), os0 = __shfl_xor_sync(0xffffffffu, s0, off);
            const float om1 = __shfl_xor_sync(0xffffffffu, m1, off), os1 = __shfl_xor_sync(0xffffffffu, s1, off);
            const float n0m = fmaxf(m0, om0), n1m = fmaxf(m1, om1);
            s0 = (n0m > -INFINITY) ? s0 * exp2f(m0 - n0m) + os0 * exp2f(om0 - n0m) : 0.f;
            s1 = (n1m > -INFINITY) ? s1 * exp2f(m1 - n1m) + os1 * exp2f(om1 - n1m) : 0.f;
            m0 = n0m;
            m1 = n1m;
        }
        if (g == 0) {
            if (n_sub == 1) {   // one warp per KV group: its partial is the CTA's
                if (h0) p.part[((long long)b * p.nsel + first + 2 * c) * p.n_chunks + chunk] = make_float2(m0, s0);
                if (h1) p.part[((long long)b * p.nsel + first + 2 * c + 1) * p.n_chunks + chunk] = make_float2(m1, s1);
            } else {            // several warps share the group (each took every n_sub-th tile): folded below
                s_part[warp][2 * c] = make_float2(m0, s0);
                s_part[warp][2 * c + 1] = make_float2(m1, s1);
            }
        }
    }
    if (n_sub > 1) {
        // Fewer than eight scored KV groups: the warps ws = 0 .. n_sub-1 of a group fold their partials in that order, so
        // that the CTA leaves ONE partial per head (the consumers fold n_chunks of them per head; with a single scored
        // group that is an eighth of what it would be).  slots >= n_groups here, so the loop above ran at most once.
        __syncthreads();
        const int gi = warp;   // warps 0 .. slots-1 (ws == 0) finish the groups 0 .. slots-1
        if (gi < p.n_groups && gi < slots && lane < p.group_cnt[gi]) {
            float m = -INFINITY, s = 0.f;
            for (int i = 0; i < n_sub; ++i) {
                const float2 o = s_part[gi + slots * i][lane];
                softmax_merge(m, s, o.x, o.y);
            }
            p.part[((long long)b * p.nsel + p.group_first[gi] + lane) * p.n_chunks + chunk] = make_float2(m, s);
        }
    }
    // Fused call with a hoisted draft tier: ONE CTA -- the last of the grid, dispatched in the last wave -- waits for the
    // draft-tier kernel that runs beside this one, so that "a1 complete" implies "draft tier complete and visible" for the
    // kernels that follow.  (Every CTA waiting would park the early ones on their SMs until that kernel is done.)
    if (p.defer_wait && blockIdx.x == gridDim.x - 1 && blockIdx.y == gridDim.y - 1) pdl_wait();
    pdl_trigger();
}

// (M, 1/Z) of every subset head from the per-CTA partials: one warp per (head, sequence).
__global__ void __launch_bounds__(32) score_stats_kernel(const ScoreParams p) {
    const int j = blockIdx.x, b = blockIdx.y, lane = threadIdx.x;
    const float2 st = fold_stats_warp(p.part + ((long long)b * p.nsel + j) * p.n_chunks, p.n_chunks, lane);
    if (lane == 0) p.stats[(long long)b * p.nsel + j] = st;
}

// p = exp2(l - M) / Z, summed over the heads that feed list l; optional Eq. 5 accumulation into hist.
// VEC = 4: every row of scores_now / hist is 16-byte aligned (max_ctx % 4 == 0); VEC = 1: any max_ctx.
template <int VEC>
__global__ void __launch_bounds__(256) score_normalize_kernel(const ScoreParams p, float* __restrict__ scores_now,
                                                              float* __restrict__ hist, float alpha) {
    const int l = blockIdx.y, b = blockIdx.z;
    const int N = seq_len_of(p.kv.seq_lens, b, p.max_ctx);
    const int first = p.list_first[l], nh = p.list_cnt[l];
    __shared__ float2 st[64];
    if (threadIdx.x < nh) st[threadIdx.x] = p.stats[(long long)b * p.nsel + first + threadIdx.x];
    __syncthreads();
    const long long row = ((long long)b * p.n_lists + l) * p.max_ctx;
    const float* lg = p.logits + ((long long)b * p.nsel + first) * p.logit_stride;
    for (int n = (blockIdx.x * 256 + threadIdx.x) * VEC; n < p.max_ctx; n += gridDim.x * 256 * VEC) {
        float a[VEC];
#pragma unroll
        for (int i = 0; i < VEC; ++i) a[i] = 0.f;
        if (n < N) {
            for (int j = 0; j < nh; ++j) {
                if constexpr (VEC == 4) {
                    prob_accumulate4(a, __ldcg(reinterpret_cast<const float4*>(lg + (long long)j * p.logit_stride + n)),
                                     st[j]);
                } else {
                    a[0] = __fmaf_rn(exp2f(__ldcg(lg + (long long)j * p.logit_stride + n) - st[j].x), st[j].y, a[0]);
                }
            }
#pragma unroll
            for (int i = 1; i < VEC; ++i)
                if (n + i >= N) a[i] = 0.f;
        }
        if (VEC == 4) {
            if (scores_now)
                *reinterpret_cast<float4*>(scores_now + row + n) = make_float4(a[0], a[VEC > 1 ? 1 : 0], a[VEC > 2 ? 2 : 0], a[VEC > 3 ? 3 : 0]);
            if (hist && n < N) {
                float4 h = *reinterpret_cast<const float4*>(hist + row + n);
                h.x = __fmaf_rn(alpha, h.x, a[0]);
                if (n + 1 < N) h.y = __fmaf_rn(alpha, h.y, a[VEC > 1 ? 1 : 0]);
                if (n + 2 < N) h.z = __fmaf_rn(alpha, h.z, a[VEC > 2 ? 2 : 0]);
                if (n + 3 < N) h.w = __fmaf_rn(alpha, h.w, a[VEC > 3 ? 3 : 0]);
                *reinterpret_cast<float4*>(hist + row + n) = h;
            }
        } else {
            if (scores_now) scores_now[row + n] = a[0];
            if (hist && n < N) hist[row + n] = fmaf(alpha, hist[row + n], a[0]);
        }
    }
}

template <int VEC>
__global__ void __launch_bounds__(256) fuse_kernel(int max_ctx, const int* __restrict__ seq_lens,
                                                   const float* __restrict__ now, float* __restrict__ hist,
                                                   float alpha, int n_lists) {
    const int b = blockIdx.z, l = blockIdx.y;
    const int N = seq_len_of(seq_lens, b, max_ctx);
    const long long row = ((long long)b * n_lists + l) * max_ctx;
    for (int n = (blockIdx.x * 256 + threadIdx.x) * VEC; n < N; n += gridDim.x * 256 * VEC) {
        if (VEC == 4 && n + 3 < N) {
            const float4 a = *reinterpret_cast<const float4*>(now + row + n);
            float4 h = *reinterpret_cast<const float4*>(hist + row + n);
            h.x = fmaf(alpha, h.x, a.x);
            h.y = fmaf(alpha, h.y, a.y);
            h.z = fmaf(alpha, h.z, a.z);
            h.w = fmaf(alpha, h.w, a.w);
            *reinterpret_cast<float4*>(hist + row + n) = h;
        } else {
            for (int i = n; i < min(n + VEC, N); ++i) hist[row + i] = fmaf(alpha, hist[row + i], now[row + i]);
        }
    }
}

}  // namespace

cudaError_t launch_score(const ScoreParams& p, float* scores_now, float* hist, float alpha, bool logits_only,
                         cudaStream_t stream) {
    cudaError_t e0 = cudaSuccess;
    dim3 grid(p.n_chunks, p.batch);   // one softmax partial per (CTA, head)
    {
        ProfScope prof(kKernScoreLogits, stream);
        const int smem = kScoreWarps * kStages * kTileTokens * p.head_dim * 2;
        static DeviceOnce once;
        const cudaError_t ea = ensure_dyn_smem(reinterpret_cast<const void*>(score_logits_kernel<128>),
                                               kScoreWarps * kStages * kTileTokens * 128 * 2, once);
        if (ea != cudaSuccess) return ea;
        if (p.head_dim == 128)
            e0 = launch_pdl(score_logits_kernel<128>, grid, dim3(kScoreThreads), smem, stream, p);
        else
            e0 = launch_pdl(score_logits_kernel<64>, grid, dim3(kScoreThreads), smem, stream, p);
    }
    cudaError_t e = e0 != cudaSuccess ? e0 : cudaGetLastError();
    if (e != cudaSuccess || logits_only) return e;   // logits_only: the consumer (select.cu) normalises its own rows
    {
        ProfScope prof(kKernScoreStats, stream);
        score_stats_kernel<<<dim3(p.nsel, p.batch), 32, 0, stream>>>(p);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ProfScope prof(kKernScoreNormalize, stream);
    const int nblk = max(1, min((p.max_ctx + 1023) / 1024, 64));
    const bool vec = (p.max_ctx & 3) == 0 && (((uintptr_t)scores_now | (uintptr_t)hist) & 15) == 0;
    if (vec)
        score_normalize_kernel<4><<<dim3(nblk, p.n_lists, p.batch), 256, 0, stream>>>(p, scores_now, hist, alpha);
    else
        score_normalize_kernel<1><<<dim3(nblk, p.n_lists, p.batch), 256, 0, stream>>>(p, scores_now, hist, alpha);
    return cudaGetLastError();
}

cudaError_t launch_fuse(int batch, int n_lists, int max_ctx, const int* seq_lens, const float* now, float* hist,
                        float alpha, cudaStream_t stream) {
    const int nblk = max(1, min((max_ctx + 1023) / 1024, 64));
    const bool vec = (max_ctx & 3) == 0 && (((uintptr_t)now | (uintptr_t)hist) & 15) == 0;
    ProfScope prof(kKernFuse, stream);
    if (vec)
        fuse_kernel<4><<<dim3(nblk, n_lists, batch), 256, 0, stream>>>(max_ctx, seq_lens, now, hist, alpha, n_lists);
    else
        fuse_kernel<1><<<dim3(nblk, n_lists, batch), 256, 0, stream>>>(max_ctx, seq_lens, now, hist, alpha, n_lists);
    return cudaGetLastError();
}

}  // namespace dustin
