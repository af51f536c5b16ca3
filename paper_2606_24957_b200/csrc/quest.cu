// quest.cu -- the Quest-16 estimator the paper measures its head-subset scoring against ("scores KV pages
// using inexpensive min/max key statistics (avoiding exact QK^T)", :297-299 "Quest-16 denotes Quest with page size 16",
// :401 "aggregates token-level Key statistics (e.g., minimum and maximum values) into page-level metadata").
// DESIGN.md readings A20 (the channel-wise upper bound) and A21 (page scores in the format of stage a1).
//
//   quest_build_kernel      page metadata: per (sequence, 16-token page, KV head, channel) the min and the max of the keys.
//                           One warp per (page, KV head): 16 row loads of D * 2 bytes in flight per warp, one pass over K
//                           (HBM-bound, done once after prefill; after an append only the pages from `first_token` on).
//   quest_score_kernel      U_h[p] = scale * sum_c max(q_c * kmin_c, q_c * kmax_c) for the subset heads: one streaming read
//                           of the metadata of the scored KV groups (2 * D * 2 bytes per page and group = 1/8 of the K
//                           bytes that a1 reads for the same groups), a warp per page, four pages per round and the
//                           next round requested before the current one is consumed; log2-domain bounds to an L2-resident
//                           scratch.
//   quest_normalize_kernel  softmax over the pages that hold a token (max, sum, normalise: three passes over the small
//                           rows of bounds), summed over the heads that feed each list.
// Plain CUDA cores: 2 flop per byte, far below any tensor-core ridge -- these kernels only have to keep loads in flight.
#include "kernels.cuh"

namespace dustin {

namespace {

constexpr int kQuestWarps = 8;

__device__ __forceinline__ uint32_t bf162_min(uint32_t a, uint32_t b) {
    const __nv_bfloat162 r = __hmin2(*reinterpret_cast<const __nv_bfloat162*>(&a), *reinterpret_cast<const __nv_bfloat162*>(&b));
    return *reinterpret_cast<const uint32_t*>(&r);
}
__device__ __forceinline__ uint32_t bf162_max(uint32_t a, uint32_t b) {
    const __nv_bfloat162 r = __hmax2(*reinterpret_cast<const __nv_bfloat162*>(&a), *reinterpret_cast<const __nv_bfloat162*>(&b));
    return *reinterpret_cast<const uint32_t*>(&r);
}

template <int E>
struct LaneVec;                    // E bf16 values of one lane: D = 128 -> 8 bytes, D = 64 -> 4 bytes
template <>
struct LaneVec<4> {
    uint2 v;
    __device__ __forceinline__ void load(const __nv_bfloat16* p) { v = __ldcs(reinterpret_cast<const uint2*>(p)); }
    __device__ __forceinline__ void unpack(float (&f)[4]) const {
        f[0] = __uint_as_float(v.x << 16);
        f[1] = __uint_as_float(v.x & 0xffff0000u);
        f[2] = __uint_as_float(v.y << 16);
        f[3] = __uint_as_float(v.y & 0xffff0000u);
    }
    __device__ __forceinline__ uint32_t word(int e) const { return e == 0 ? v.x : v.y; }   // two bf16 each
    __device__ __forceinline__ static void store_words(__nv_bfloat16* p, const uint32_t (&w)[2]) {
        *reinterpret_cast<uint2*>(p) = make_uint2(w[0], w[1]);
    }
};
template <>
struct LaneVec<2> {
    uint32_t v;
    __device__ __forceinline__ void load(const __nv_bfloat16* p) { v = __ldcs(reinterpret_cast<const uint32_t*>(p)); }
    __device__ __forceinline__ void unpack(float (&f)[2]) const {
        f[0] = __uint_as_float(v << 16);
        f[1] = __uint_as_float(v & 0xffff0000u);
    }
    __device__ __forceinline__ uint32_t word(int) const { return v; }
    __device__ __forceinline__ static void store_words(__nv_bfloat16* p, const uint32_t (&w)[1]) {
        *reinterpret_cast<uint32_t*>(p) = w[0];
    }
};

// gridDim = (CTAs per sequence, batch); a warp takes the (page, KV head) items blockIdx.x * 8 + warp, + gridDim.x * 8, ...
template <int D>
__global__ void __launch_bounds__(kQuestWarps * 32) quest_build_kernel(const KvView kv, const int* __restrict__ first_token,
                                                                      __nv_bfloat16* __restrict__ meta, int n_kv_heads,
                                                                      int max_ctx, int n_pages) {
    constexpr int E = D / 32, P = DUSTIN_QUEST_PAGE;
    const int b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int N = seq_len_of(kv.seq_lens, b, max_ctx);
    int p_first = 0;
    if (first_token) {
        const int ft = first_token[b];
        p_first = (ft < 0 ? 0 : ft) / P;
    }
    const int total = n_pages * n_kv_heads;
    for (int item = p_first * n_kv_heads + blockIdx.x * kQuestWarps + warp; item < total; item += gridDim.x * kQuestWarps) {
        const int p = item / n_kv_heads, g = item - p * n_kv_heads;
        const int n0 = p * P, cnt = min(P, N - n0);
        LaneVec<E> rows[P];
#pragma unroll
        for (int i = 0; i < P; ++i)
            if (i < cnt) rows[i].load(kv.k + kv_row_offset(kv, b, n0 + i, g) + lane * E);
        // packed bf16x2 min / max (no unpacking: the float version executed 47 warp instructions per row load and was
        // issue-bound, ncu: 199 M instructions, issue active 73 %); a page without a token keeps the zeros
        uint32_t lo[E / 2], hi[E / 2];
#pragma unroll
        for (int e = 0; e < E / 2; ++e) lo[e] = hi[e] = cnt > 0 ? rows[0].word(e) : 0u;
#pragma unroll
        for (int i = 1; i < P; ++i)
            if (i < cnt) {
#pragma unroll
                for (int e = 0; e < E / 2; ++e) {
                    lo[e] = bf162_min(lo[e], rows[i].word(e));
                    hi[e] = bf162_max(hi[e], rows[i].word(e));
                }
            }
        __nv_bfloat16* dst = meta + ((((long long)b * n_pages + p) * n_kv_heads + g) * 2) * D + lane * E;
        LaneVec<E>::store_words(dst, lo);
        LaneVec<E>::store_words(dst + D, hi);
    }
}

// gridDim = (chunks of p.chunk_pages pages, batch).  Warp w serves scored KV group w % group_slots (as the scoring kernel of
// a1 does) and, when fewer than 8 groups are scored, every n_sub-th block of kQuestUnroll pages.  NH = compile-time bound of
// the subset heads per KV group (1, 2, 4 or 8).  The loop body is kept lean on purpose -- the first version (softmax
// bookkeeping per page, eight predicated head bodies, addresses recomputed per load) executed 136 warp instructions per
// 512-byte page and was ISSUE-bound at 1.4 TB/s (ncu: 35.8 M instructions, issue active 38 %, i-cache stalls): the
// softmax statistics now come from the normalise kernel, which re-reads the small L2-resident rows of bounds.
constexpr int kQuestUnroll = 4;
template <int D, int NH>
// Resident CTAs per SM that quest_plan counts on: three with one or two heads per KV group (<= 85 registers), else two.
__global__ void __launch_bounds__(kQuestWarps * 32, NH > 2 ? 2 : 3) quest_score_kernel(const QuestParams p) {
    constexpr int E = D / 32, U = kQuestUnroll;
    const int chunk = blockIdx.x, b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int N = seq_len_of(p.seq_lens, b, p.max_ctx);
    const int n_live = (N + DUSTIN_QUEST_PAGE - 1) / DUSTIN_QUEST_PAGE;
    const int p_lo = chunk * p.chunk_pages, p_hi = min(p_lo + p.chunk_pages, n_live);
    const int slots = p.group_slots, n_sub = kQuestWarps / slots, sub = warp / slots;
    const long long pstride = (long long)p.n_kv_heads * 2 * D;   // elements between consecutive pages of one KV head
    for (int gi = warp % slots; gi < p.n_groups; gi += slots) {
        const int grp = p.group_id[gi], first = p.group_first[gi], nh = p.group_cnt[gi];
        // max(q * kmin, q * kmax) = max(q, 0) * kmax + min(q, 0) * kmin: two FMAs per channel, one of them adding an exact
        // zero (bf16 x bf16 is exact in fp32), instead of two products, a max and an add
        float qp[NH][E], qn[NH][E];
#pragma unroll
        for (int j = 0; j < NH; ++j) {
#pragma unroll
            for (int e = 0; e < E; ++e) qp[j][e] = qn[j][e] = 0.f;
            if (j < nh) {
                LaneVec<E> t;
                float f[E];
                t.load(p.q + (long long)b * p.q_stride_batch + p.sel_qoff[first + j] + lane * E);
                t.unpack(f);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    qp[j][e] = fmaxf(f[e], 0.f);
                    qn[j][e] = fminf(f[e], 0.f);
                }
            }
        }
        const int step = n_sub * U;
        int pg = p_lo + sub * U;
        const __nv_bfloat16* src = p.meta + ((long long)b * p.n_pages * p.n_kv_heads + grp) * 2 * D + lane * E + pg * pstride;
        const long long sstep = step * pstride;
        float* urow = p.u + ((long long)b * p.nsel + first) * p.u_stride;
        float* brow = p.ub_out ? p.ub_out + ((long long)b * p.nsel + first) * p.n_pages : nullptr;
        // request the U pages from page pg0 on (src0 = address of page pg0)
        auto request = [&](LaneVec<E>(&mn)[U], LaneVec<E>(&mx)[U], const __nv_bfloat16* src0, int pg0) {
#pragma unroll
            for (int u = 0; u < U; ++u)
                if (pg0 + u < p_hi) {
                    mn[u].load(src0 + u * pstride);
                    mx[u].load(src0 + u * pstride + D);
                }
        };
        // bounds of the U pages from pg0 on, for every head of the group; lane u stores page pg0 + u
        auto consume = [&](const LaneVec<E>(&mn)[U], const LaneVec<E>(&mx)[U], int pg0) {
            float a[NH][U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                float fmn[E], fmx[E];
                mn[u].unpack(fmn);
                mx[u].unpack(fmx);
#pragma unroll
                for (int j = 0; j < NH; ++j) {
                    float t = 0.f;
#pragma unroll
                    for (int e = 0; e < E; ++e) t = __fmaf_rn(qn[j][e], fmn[e], __fmaf_rn(qp[j][e], fmx[e], t));
                    a[j][u] = t;
                }
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1)
#pragma unroll
                for (int j = 0; j < NH; ++j)
#pragma unroll
                    for (int u = 0; u < U; ++u) a[j][u] += __shfl_xor_sync(0xffffffffu, a[j][u], off);
#pragma unroll
            for (int j = 0; j < NH; ++j) {
                float v = a[j][0];
#pragma unroll
                for (int u = 1; u < U; ++u) v = lane == u ? a[j][u] : v;
                if (lane < U && pg0 + lane < p_hi && j < nh) {   // pages past p_hi hold stale registers: not stored
                    urow[(long long)j * p.u_stride + pg0 + lane] = v * p.scale_log2;
                    if (brow) brow[(long long)j * p.n_pages + pg0 + lane] = v * p.scale;
                }
            }
        };
        // two register buffers in turn: the next round is in flight while the current one is consumed, without copies
        LaneVec<E> amn[U], amx[U], bmn[U], bmx[U];
        request(amn, amx, src, pg);
        while (pg < p_hi) {
            request(bmn, bmx, src + sstep, pg + step);
            consume(amn, amx, pg);
            pg += step;
            src += sstep;
            if (pg >= p_hi) break;
            request(amn, amx, src + sstep, pg + step);
            consume(bmn, bmx, pg);
            pg += step;
            src += sstep;
        }
    }
    // ub_out of the pages without a token: 0
    if (p.ub_out) {
        const int q_lo = max(p_lo, n_live), q_hi = min(p_lo + p.chunk_pages, p.n_pages);
        for (int ord = warp; ord < p.nsel; ord += kQuestWarps)
            for (int pg = q_lo + lane; pg < q_hi; pg += 32) p.ub_out[((long long)b * p.nsel + ord) * p.n_pages + pg] = 0.f;
    }
}

// gridDim = (n_lists, batch), 1024 threads.  Per head of the list: max, then sum of exp2, over its row of bounds; then every
// thread writes its pages.  A list fed by many heads (>= 16) gives every warp whole heads; otherwise the whole CTA works
// on one head at a time (one warp per head took 15 us at 32k and 37 us at 128k: 64 to 256 dependent L2 loads per lane).
// Both orders are fixed (strided elements in index order per thread, xor tree per warp, warps in order): deterministic.
// The rows are small (n_pages floats per head) and L2-resident.
__global__ void __launch_bounds__(1024) quest_normalize_kernel(const QuestParams p, float* __restrict__ out) {
    const int l = blockIdx.x, b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int N = seq_len_of(p.seq_lens, b, p.max_ctx);
    const int n_live = (N + DUSTIN_QUEST_PAGE - 1) / DUSTIN_QUEST_PAGE;
    const int first = p.list_first[l], nh = p.list_cnt[l];
    __shared__ float2 st[64];
    __shared__ float red[32];
    const float* u = p.u + ((long long)b * p.nsel + first) * p.u_stride;
    if (nh >= 16) {
        for (int j = warp; j < nh; j += 32) {
            const float* row = u + (long long)j * p.u_stride;
            float m = -INFINITY;
            for (int pg = lane; pg < n_live; pg += 32) m = fmaxf(m, __ldcg(row + pg));
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
            float z = 0.f;
            for (int pg = lane; pg < n_live; pg += 32) z += exp2f(__ldcg(row + pg) - m);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) z += __shfl_xor_sync(0xffffffffu, z, off);
            if (lane == 0) st[j] = make_float2(m, z > 0.f ? 1.f / z : 0.f);
        }
    } else {
        for (int j = 0; j < nh; ++j) {
            const float* row = u + (long long)j * p.u_stride;
            float m = -INFINITY;
            for (int pg = threadIdx.x; pg < n_live; pg += 1024) m = fmaxf(m, __ldcg(row + pg));
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
            if (lane == 0) red[warp] = m;
            __syncthreads();
            m = red[lane];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
            __syncthreads();
            float z = 0.f;
            for (int pg = threadIdx.x; pg < n_live; pg += 1024) z += exp2f(__ldcg(row + pg) - m);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) z += __shfl_xor_sync(0xffffffffu, z, off);
            if (lane == 0) red[warp] = z;
            __syncthreads();
            z = red[lane];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) z += __shfl_xor_sync(0xffffffffu, z, off);
            if (threadIdx.x == 0) st[j] = make_float2(m, z > 0.f ? 1.f / z : 0.f);
            __syncthreads();
        }
    }
    __syncthreads();
    for (int pg = threadIdx.x; pg < p.n_pages; pg += 1024) {
        float a = 0.f;
        if (pg < n_live)
            for (int j = 0; j < nh; ++j) a = __fmaf_rn(exp2f(__ldcg(u + (long long)j * p.u_stride + pg) - st[j].x), st[j].y, a);
        out[((long long)b * p.n_lists + l) * p.n_pages + pg] = a;
    }
}

}  // namespace

// Scoring plan: which warps share a KV group and how many pages a CTA takes: one wave of resident CTAs over the whole
// grid, each at least two rounds long.
void quest_plan(int batch, int n_groups, int max_heads_per_group, int n_pages, int* group_slots, int* chunk_pages,
                int* n_chunks) {
    int slots = 1;
    while (slots < n_groups && slots < kQuestWarps) slots <<= 1;
    const int unit = kQuestUnroll * (kQuestWarps / slots);   // pages that the warps of one group take per round
    // CTAs per sequence for ONE wave: three CTAs fit an SM, two with more than two heads per group (the kernel's launch bounds);
    // rounded DOWN -- a grid just over the resident limit runs a second wave (measured: 93 -> 158 us)
    const int target = (max_heads_per_group > 2 ? 2 : 3) * device_sm_count() / batch;
    int chunk = (n_pages + target - 1) / (target > 0 ? target : 1);
    chunk = (chunk + unit - 1) / unit * unit;
    if (chunk < 2 * unit) chunk = 2 * unit;
    *group_slots = slots;
    *chunk_pages = chunk;
    *n_chunks = n_pages > 0 ? (n_pages + chunk - 1) / chunk : 1;
}

cudaError_t launch_quest_build(const KvView& kv, const int* first_token, __nv_bfloat16* meta, int batch, int n_kv_heads,
                               int head_dim, int max_ctx, int n_pages, cudaStream_t stream) {
    const int total = n_pages * n_kv_heads;
    if (total <= 0) return cudaSuccess;
    const int per_seq = (total + kQuestWarps - 1) / kQuestWarps;
    // enough CTAs for eight per SM over the whole grid, never more than one item per warp needs
    int gx = (8 * device_sm_count() + batch - 1) / batch;
    gx = gx < 1 ? 1 : (gx > per_seq ? per_seq : gx);
    ProfScope prof(kKernQuestBuild, stream);
    if (head_dim == 128)
        quest_build_kernel<128><<<dim3(gx, batch), kQuestWarps * 32, 0, stream>>>(kv, first_token, meta, n_kv_heads, max_ctx, n_pages);
    else
        quest_build_kernel<64><<<dim3(gx, batch), kQuestWarps * 32, 0, stream>>>(kv, first_token, meta, n_kv_heads, max_ctx, n_pages);
    return cudaGetLastError();
}

template <int D>
cudaError_t launch_quest_score_d(const QuestParams& p, int max_nh, cudaStream_t stream) {
    const dim3 grid(p.n_chunks, p.batch), block(kQuestWarps * 32);
    if (max_nh <= 1) quest_score_kernel<D, 1><<<grid, block, 0, stream>>>(p);
    else if (max_nh <= 2) quest_score_kernel<D, 2><<<grid, block, 0, stream>>>(p);
    else if (max_nh <= 4) quest_score_kernel<D, 4><<<grid, block, 0, stream>>>(p);
    else quest_score_kernel<D, 8><<<grid, block, 0, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_quest_score(const QuestParams& p, float* page_scores, cudaStream_t stream) {
    if (p.n_pages <= 0) return cudaSuccess;
    int max_nh = 1;
    for (int gi = 0; gi < p.n_groups; ++gi) max_nh = max(max_nh, (int)p.group_cnt[gi]);
    cudaError_t e;
    {
        ProfScope prof(kKernQuestScore, stream);
        e = p.head_dim == 128 ? launch_quest_score_d<128>(p, max_nh, stream) : launch_quest_score_d<64>(p, max_nh, stream);
    }
    if (e != cudaSuccess) return e;
    ProfScope prof(kKernQuestNormalize, stream);
    quest_normalize_kernel<<<dim3(p.n_lists, p.batch), 1024, 0, stream>>>(p, page_scores);
    return cudaGetLastError();
}

}  // namespace dustin
