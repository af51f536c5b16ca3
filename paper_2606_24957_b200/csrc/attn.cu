// attn.cu -- stage a4 (sparse verification attention over the selected KV, App. G :568) and a5
// (the full-cache verification baseline of PAPER.md:248 / :570: same kernel, idx == nullptr) for sm_100a.
//
// Flash-style, index-driven, split over the selected tokens, one thread-block CLUSTER per (sequence, KV head):
//   grid = (n_splits, Hkv, B), cluster = (n_splits, 1, 1).  CTA `split` owns a contiguous slice of the index list
//   of (b, KV head); split 0 also owns the T new draft rows (causal among themselves).
//   * Row addresses are resolved once (index -> page table -> global address of the K row and of the V row) into
//     a shared-memory table; K/V rows then stream global -> shared with 16-byte cp.async, 16 lanes per 256-byte
//     row, through a 3-stage ring of 64-token tiles (XOR-swizzled, ldmatrix-conflict-free).
//   * All T*r query rows that share the KV head sit on the M axis of bf16 mma.sync tiles (warp = one 16-row tile x
//     one token slice), fp32 online softmax in the log2 domain with the scale folded into the exponent, the O
//     rescale skipped while no row maximum moves, P re-used from the accumulator registers as the A operand of P.V.
//   * Token slices of a CTA merge in shared memory; the CTAs of a cluster leave their normalised partial in their
//     own shared memory and every CTA finishes a share of the query rows by reading its peers through DSMEM
//     (fixed split order => deterministic).  No partials in global memory, no second kernel.
#include "kernels.cuh"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace dustin {

namespace {

constexpr int kTileTokens = 64;   // tokens per pipeline stage
constexpr int kStages = 3;
constexpr int kMaxCluster = 8;    // portable cluster size
constexpr int kMaxTableTokens = 1024 + 16;   // address-table entries that still leave room for 2 CTAs per SM

enum AttnMode { kDense = 0, kGatherTable = 1, kGatherInline = 2 };

template <int D, int MT, int KS>
struct AttnCfg {
    static constexpr int kThreads = 32 * MT * KS;
    static constexpr int kWT = kTileTokens / KS;          // tokens per warp per stage
    static constexpr int kCH = D / 8;                     // 16-byte chunks per row
    static constexpr int kRowBytes = D * 2;
    static constexpr int kStageBytes = kTileTokens * kRowBytes;   // one K (or V) stage
    static constexpr int kOReg = D / 2;                   // fp32 accumulators per thread (16 x D tile)
    static constexpr size_t kPipeBytes = (size_t)kStages * kStageBytes * 2;
    static constexpr size_t kMergeBytes = (size_t)(KS - 1) * MT * 32 * (kOReg + 4) * 4;
    static constexpr size_t kPartBytes = (size_t)MT * 16 * (D + 1) * 4;   // cluster partial: o[rows][D] + lse[rows]
    static_assert(kMergeBytes + kPartBytes <= kPipeBytes, "epilogue buffers must fit the pipeline buffers");
    static constexpr int kRowsPerPass = kThreads / kCH;   // rows one cp.async pass of the CTA covers
    static constexpr int kPasses = (kTileTokens + kRowsPerPass - 1) / kRowsPerPass;
};

struct RowAddr {
    const __nv_bfloat16* k;
    const __nv_bfloat16* v;
};
// Shared-memory address table entry: K and V share one layout, so one element offset serves both; a new draft
// row u is stored as ~(its element offset in k_new / v_new) (negative).
typedef long long RowOff;

template <int D, int MT, int KS, int MODE>
__global__ void __launch_bounds__(32 * MT * KS) attn_kernel(const AttnParams p) {
    using C = AttnCfg<D, MT, KS>;
    constexpr int WT = C::kWT, CH = C::kCH, NT = C::kThreads;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* sK = smem_raw;
    unsigned char* sV = smem_raw + kStages * C::kStageBytes;
    RowOff* sTab = reinterpret_cast<RowOff*>(smem_raw + C::kPipeBytes);

    const int split = blockIdx.x, gkv = blockIdx.y, b = blockIdx.z;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int mt = warp % MT, ks = warp / MT;
    const int g = lane >> 2, c = lane & 3;
    const int T = p.n_new, r = p.group, rows = p.rows;
    const int list = p.n_lists == 1 ? 0 : gkv;
    // a caller-supplied cnt is clamped to [0, k_max] as in the tcgen05 kernel: the same inputs behave the same in both
    const int n_sel = MODE == kDense ? seq_len_of(p.kv.seq_lens, b, p.max_ctx)
                                     : (p.cnt ? max(0, min(p.cnt[b * p.n_lists + list], p.k_max)) : p.uniform_cnt);
    const int range_lo = split * p.split_tokens;
    const int n_range = max(0, min(p.split_tokens, n_sel - range_lo));
    const int nt = n_range + (split == 0 ? T : 0);        // this CTA's tokens: cache rows, then the new rows
    const int* list_idx = MODE == kDense ? nullptr : p.idx + ((long long)b * p.n_lists + list) * p.k_max + range_lo;

    // Global addresses of the K and V row of local token j.
    auto row_off = [&](int j) -> RowOff {
        if (j < n_range) {
            const int tok = MODE == kDense ? range_lo + j : __ldg(list_idx + j);
            return kv_row_offset(p.kv, b, tok, gkv);
        }
        return ~((((long long)b * T + (j - n_range)) * p.n_kv_heads + gkv) * D);
    };
    auto addr_of = [&](RowOff off) -> RowAddr {
        RowAddr a;
        a.k = off >= 0 ? p.kv.k + off : p.k_new + ~off;
        a.v = off >= 0 ? p.kv.v + off : p.v_new + ~off;
        return a;
    };
    if (MODE == kGatherTable)
        for (int j = tid; j < nt; j += NT) sTab[j] = row_off(j);

    // ---- Q fragments (A operand): rows mt*16 + g (+8), row = t*r + head-in-group -------------------------------
    uint32_t qa[D / 16][4];
    {
        const int r_lo = mt * 16 + g, r_hi = r_lo + 8;
        const __nv_bfloat16* q_lo = nullptr;
        const __nv_bfloat16* q_hi = nullptr;
        if (r_lo < rows) q_lo = p.q + (((long long)b * T + r_lo / r) * p.n_q_heads + gkv * r + r_lo % r) * D;
        if (r_hi < rows) q_hi = p.q + (((long long)b * T + r_hi / r) * p.n_q_heads + gkv * r + r_hi % r) * D;
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
            const int col = kk * 16 + 2 * c;
            qa[kk][0] = q_lo ? *reinterpret_cast<const uint32_t*>(q_lo + col) : 0u;
            qa[kk][1] = q_hi ? *reinterpret_cast<const uint32_t*>(q_hi + col) : 0u;
            qa[kk][2] = q_lo ? *reinterpret_cast<const uint32_t*>(q_lo + col + 8) : 0u;
            qa[kk][3] = q_hi ? *reinterpret_cast<const uint32_t*>(q_hi + col + 8) : 0u;
        }
    }
    __syncthreads();

    // ---- producer side: this thread copies chunk `ld_ch` of rows ld_row0, ld_row0 + kRowsPerPass, ... per tile --
    const int n_tiles = (nt + kTileTokens - 1) / kTileTokens;
    const int ld_ch = tid % CH, ld_row0 = tid / CH;
    const uint32_t sK_u32 = smem_u32(sK), sV_u32 = smem_u32(sV);
    auto issue = [&](int tile) {
        if (tile < n_tiles) {
            const uint32_t stage_off = (uint32_t)(tile % kStages) * C::kStageBytes;
            const int j0 = tile * kTileTokens;
#pragma unroll
            for (int i = 0; i < C::kPasses; ++i) {
                const int row = ld_row0 + i * C::kRowsPerPass;
                if (C::kPasses * C::kRowsPerPass > kTileTokens && row >= kTileTokens) break;
                const int j = j0 + row;
                const bool valid = j < nt;
                const RowAddr a = addr_of(MODE == kGatherTable ? sTab[valid ? j : 0] : row_off(valid ? j : 0));
                const uint32_t dst = stage_off + (uint32_t)row * C::kRowBytes + (uint32_t)((ld_ch ^ (row & 7)) << 4);
                cp_async16(sK_u32 + dst, a.k + ld_ch * 8, valid ? 16 : 0);
                cp_async16(sV_u32 + dst, a.v + ld_ch * 8, valid ? 16 : 0);
            }
        }
        cp_async_commit();
    };

    float o[D / 8][4];
#pragma unroll
    for (int i = 0; i < D / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
    // running maxima of the raw scores (q.k, unscaled) and running sums of exp2((s - m) * scale_log2)
    float m_lo = -INFINITY, m_hi = -INFINITY, l_lo = 0.f, l_hi = 0.f;
    const int t_lo = (mt * 16 + g) / r, t_hi = (mt * 16 + g + 8) / r;   // verify position of this thread's rows
    const float sl2 = p.scale_log2;

#pragma unroll
    for (int s = 0; s < kStages - 1; ++s) issue(s);

    for (int tile = 0; tile < n_tiles; ++tile) {
        cp_async_wait<kStages - 2>();
        __syncthreads();
        issue(tile + kStages - 1);
        const int j0 = tile * kTileTokens + ks * WT;       // first token of this warp's slice
        if (j0 >= nt) continue;
        const uint32_t tK = sK_u32 + (tile % kStages) * C::kStageBytes;
        const uint32_t tV = sV_u32 + (tile % kStages) * C::kStageBytes;

        // S = Q K^T
        float sc[WT / 8][4];
#pragma unroll
        for (int i = 0; i < WT / 8; ++i) sc[i][0] = sc[i][1] = sc[i][2] = sc[i][3] = 0.f;
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
#pragma unroll
            for (int np = 0; np < WT / 16; ++np) {
                const int mi = lane >> 3;
                const int row = ks * WT + np * 16 + (mi >> 1) * 8 + (lane & 7);
                const int ch = kk * 2 + (mi & 1);
                uint32_t b0, b1, b2, b3;
                ldmatrix_x4(b0, b1, b2, b3, tK + row * C::kRowBytes + ((ch ^ (row & 7)) << 4));
                mma_bf16_16816(sc[2 * np], qa[kk][0], qa[kk][1], qa[kk][2], qa[kk][3], b0, b1);
                mma_bf16_16816(sc[2 * np + 1], qa[kk][0], qa[kk][1], qa[kk][2], qa[kk][3], b2, b3);
            }
        }

        // mask (tail of the list; causality among the new rows) -- only the tiles that reach past the cache rows
        if (j0 + WT > n_range) {
#pragma unroll
            for (int i = 0; i < WT / 8; ++i) {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int j = j0 + i * 8 + 2 * c + (e & 1);
                    const int t = (e & 2) ? t_hi : t_lo;
                    if (j >= nt || (j >= n_range && j - n_range > t)) sc[i][e] = -INFINITY;
                }
            }
        }
        // online softmax: p = exp2((s - m) * scale_log2)
        float mx_lo = -INFINITY, mx_hi = -INFINITY;
#pragma unroll
        for (int i = 0; i < WT / 8; ++i) {
            mx_lo = fmaxf(mx_lo, fmaxf(sc[i][0], sc[i][1]));
            mx_hi = fmaxf(mx_hi, fmaxf(sc[i][2], sc[i][3]));
        }
        mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 1));
        mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 2));
        mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 1));
        mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 2));
        const bool moved = mx_lo > m_lo || mx_hi > m_hi;
        if (__any_sync(0xffffffffu, moved)) {   // some row maximum of this warp moved: rescale O and the sums
            const float mn_lo = fmaxf(m_lo, mx_lo), mn_hi = fmaxf(m_hi, mx_hi);
            const float al_lo = mn_lo == -INFINITY ? 1.f : fast_exp2((m_lo - mn_lo) * sl2);
            const float al_hi = mn_hi == -INFINITY ? 1.f : fast_exp2((m_hi - mn_hi) * sl2);
            m_lo = mn_lo;
            m_hi = mn_hi;
            l_lo *= al_lo;
            l_hi *= al_hi;
#pragma unroll
            for (int i = 0; i < D / 8; ++i) {
                o[i][0] *= al_lo;
                o[i][1] *= al_lo;
                o[i][2] *= al_hi;
                o[i][3] *= al_hi;
            }
        }
        const float ms_lo = m_lo == -INFINITY ? 0.f : m_lo * sl2, ms_hi = m_hi == -INFINITY ? 0.f : m_hi * sl2;
        float sum_lo = 0.f, sum_hi = 0.f;
#pragma unroll
        for (int i = 0; i < WT / 8; ++i) {
            sc[i][0] = fast_exp2(fmaf(sc[i][0], sl2, -ms_lo));
            sc[i][1] = fast_exp2(fmaf(sc[i][1], sl2, -ms_lo));
            sc[i][2] = fast_exp2(fmaf(sc[i][2], sl2, -ms_hi));
            sc[i][3] = fast_exp2(fmaf(sc[i][3], sl2, -ms_hi));
            sum_lo += sc[i][0] + sc[i][1];
            sum_hi += sc[i][2] + sc[i][3];
        }
        l_lo += sum_lo;
        l_hi += sum_hi;

        // O += P V
#pragma unroll
        for (int kk = 0; kk < WT / 16; ++kk) {
            const uint32_t a0 = pack_bf16(sc[2 * kk][0], sc[2 * kk][1]);
            const uint32_t a1 = pack_bf16(sc[2 * kk][2], sc[2 * kk][3]);
            const uint32_t a2 = pack_bf16(sc[2 * kk + 1][0], sc[2 * kk + 1][1]);
            const uint32_t a3 = pack_bf16(sc[2 * kk + 1][2], sc[2 * kk + 1][3]);
#pragma unroll
            for (int dp = 0; dp < D / 16; ++dp) {
                const int mi = lane >> 3;
                const int row = ks * WT + kk * 16 + (mi & 1) * 8 + (lane & 7);
                const int ch = dp * 2 + (mi >> 1);
                uint32_t b0, b1, b2, b3;
                ldmatrix_x4_trans(b0, b1, b2, b3, tV + row * C::kRowBytes + ((ch ^ (row & 7)) << 4));
                mma_bf16_16816(o[2 * dp], a0, a1, a2, a3, b0, b1);
                mma_bf16_16816(o[2 * dp + 1], a0, a1, a2, a3, b2, b3);
            }
        }
    }
    cp_async_wait<0>();
    __syncthreads();

    l_lo += __shfl_xor_sync(0xffffffffu, l_lo, 1);
    l_lo += __shfl_xor_sync(0xffffffffu, l_lo, 2);
    l_hi += __shfl_xor_sync(0xffffffffu, l_hi, 1);
    l_hi += __shfl_xor_sync(0xffffffffu, l_hi, 2);
    // from here on the maxima live in the log2 domain
    m_lo = m_lo == -INFINITY ? -INFINITY : m_lo * sl2;
    m_hi = m_hi == -INFINITY ? -INFINITY : m_hi * sl2;

    // ---- merge the KS token slices of this CTA through shared memory (pipeline buffers are free now) ----------
    if (KS > 1) {
        float* mg = reinterpret_cast<float*>(smem_raw);
        constexpr int kPer = C::kOReg + 4;
        if (ks > 0) {
            float* dst = mg + (size_t)((ks - 1) * MT + mt) * kPer * 32 + lane;
#pragma unroll
            for (int i = 0; i < D / 8; ++i)
#pragma unroll
                for (int e = 0; e < 4; ++e) dst[(i * 4 + e) * 32] = o[i][e];
            dst[(C::kOReg + 0) * 32] = m_lo;
            dst[(C::kOReg + 1) * 32] = m_hi;
            dst[(C::kOReg + 2) * 32] = l_lo;
            dst[(C::kOReg + 3) * 32] = l_hi;
        }
        __syncthreads();
        if (ks == 0) {
            for (int k2 = 1; k2 < KS; ++k2) {
                const float* src = mg + (size_t)((k2 - 1) * MT + mt) * kPer * 32 + lane;
                const float om_lo = src[(C::kOReg + 0) * 32], om_hi = src[(C::kOReg + 1) * 32];
                const float ol_lo = src[(C::kOReg + 2) * 32], ol_hi = src[(C::kOReg + 3) * 32];
                const float mn_lo = fmaxf(m_lo, om_lo), mn_hi = fmaxf(m_hi, om_hi);
                const float mu_lo = mn_lo == -INFINITY ? 0.f : mn_lo, mu_hi = mn_hi == -INFINITY ? 0.f : mn_hi;
                const float a_lo = fast_exp2(m_lo - mu_lo), b_lo = fast_exp2(om_lo - mu_lo);
                const float a_hi = fast_exp2(m_hi - mu_hi), b_hi = fast_exp2(om_hi - mu_hi);
#pragma unroll
                for (int i = 0; i < D / 8; ++i) {
                    o[i][0] = o[i][0] * a_lo + src[(i * 4 + 0) * 32] * b_lo;
                    o[i][1] = o[i][1] * a_lo + src[(i * 4 + 1) * 32] * b_lo;
                    o[i][2] = o[i][2] * a_hi + src[(i * 4 + 2) * 32] * b_hi;
                    o[i][3] = o[i][3] * a_hi + src[(i * 4 + 3) * 32] * b_hi;
                }
                l_lo = l_lo * a_lo + ol_lo * b_lo;
                l_hi = l_hi * a_hi + ol_hi * b_hi;
                m_lo = mn_lo;
                m_hi = mn_hi;
            }
        }
    }

    const float inv_lo = l_lo > 0.f ? 1.f / l_lo : 0.f, inv_hi = l_hi > 0.f ? 1.f / l_hi : 0.f;
    const float lse_lo = l_lo > 0.f ? m_lo + log2f(l_lo) : -INFINITY;   // log2-domain normaliser
    const float lse_hi = l_hi > 0.f ? m_hi + log2f(l_hi) : -INFINITY;

    if (p.n_splits == 1) {   // ---- single CTA per (b, KV head): write the bf16 output ------------------------------
        if (ks != 0) return;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const int row = mt * 16 + g + half * 8;
            if (row >= rows) continue;
            const float inv = half ? inv_hi : inv_lo, lse = half ? lse_hi : lse_lo;
            const int t = row / r, h = gkv * r + row % r;
            __nv_bfloat16* dst = p.out + (((long long)b * T + t) * p.n_q_heads + h) * D + 2 * c;
#pragma unroll
            for (int i = 0; i < D / 8; ++i)
                *reinterpret_cast<uint32_t*>(dst + i * 8) = pack_bf16(o[i][half * 2] * inv, o[i][half * 2 + 1] * inv);
            if (p.lse_out && c == 0) p.lse_out[((long long)b * p.n_q_heads + h) * T + t] = lse * kLn2;
        }
        return;
    }

    // ---- cluster combine: normalised partial -> own shared memory; every CTA finishes a share of the rows -------
    float* sPart = reinterpret_cast<float*>(smem_raw + C::kMergeBytes);   // [MT*16][D]
    float* sLse = sPart + MT * 16 * D;                                     // [MT*16]
    if (ks == 0) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const int row = mt * 16 + g + half * 8;
            const float inv = half ? inv_hi : inv_lo;
            float* dst = sPart + row * D + 2 * c;
#pragma unroll
            for (int i = 0; i < D / 8; ++i)
                *reinterpret_cast<float2*>(dst + i * 8) = make_float2(o[i][half * 2] * inv, o[i][half * 2 + 1] * inv);
            if (c == 0) sLse[row] = half ? lse_hi : lse_lo;
        }
    }
    cg::cluster_group cluster = cg::this_cluster();
    cluster.sync();
    {
        const int S = p.n_splits;
        const int rows_per = (rows + S - 1) / S;
        const int row_lo = split * rows_per, row_hi = min(rows, row_lo + rows_per);
        constexpr int V4 = D / 4;   // float4 chunks per row
        for (int item = tid; item < (row_hi - row_lo) * V4; item += NT) {
            const int row = row_lo + item / V4, ch = item % V4;
            float M = -INFINITY;
            for (int s = 0; s < S; ++s) M = fmaxf(M, *cluster.map_shared_rank(sLse + row, s));
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            float W = 0.f;
            for (int s = 0; s < S; ++s) {
                const float lse = *cluster.map_shared_rank(sLse + row, s);
                const float wgt = lse == -INFINITY ? 0.f : exp2f(lse - M);
                const float4 x = *reinterpret_cast<const float4*>(cluster.map_shared_rank(sPart + row * D + ch * 4, s));
                W += wgt;
                acc.x += wgt * x.x;
                acc.y += wgt * x.y;
                acc.z += wgt * x.z;
                acc.w += wgt * x.w;
            }
            const float inv = W > 0.f ? 1.f / W : 0.f;
            const int t = row / r, h = gkv * r + row % r;
            __nv_bfloat16* dst = p.out + (((long long)b * T + t) * p.n_q_heads + h) * D + ch * 4;
            *reinterpret_cast<uint2*>(dst) =
                make_uint2(pack_bf16(acc.x * inv, acc.y * inv), pack_bf16(acc.z * inv, acc.w * inv));
            if (p.lse_out && ch == 0)
                p.lse_out[((long long)b * p.n_q_heads + h) * T + t] = W > 0.f ? (M + log2f(W)) * kLn2 : -INFINITY;
        }
    }
    cluster.sync();   // peers may still be reading this CTA's shared memory
}

template <int D, int MT, int KS, int MODE>
cudaError_t launch_mode(const AttnParams& p, cudaStream_t stream) {
    using C = AttnCfg<D, MT, KS>;
    const size_t table = MODE == kGatherTable ? (size_t)(p.split_tokens + 16) * sizeof(RowOff) : 0;
    const size_t smem = C::kPipeBytes + table;
    static DeviceOnce once;   // per instantiation
    {
        const cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(attn_kernel<D, MT, KS, MODE>),
                                              (int)(C::kPipeBytes + kMaxTableTokens * sizeof(RowOff)), once);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.n_splits, p.n_kv_heads, p.batch);
    cfg.blockDim = dim3(C::kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = p.n_splits;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ProfScope prof(kKernAttn, stream);
    return cudaLaunchKernelEx(&cfg, attn_kernel<D, MT, KS, MODE>, p);
}

template <int D, int MT, int KS>
cudaError_t launch_cfg(const AttnParams& p, cudaStream_t stream) {
    if (p.idx == nullptr) return launch_mode<D, MT, KS, kDense>(p, stream);
    if (p.split_tokens + 16 <= kMaxTableTokens) return launch_mode<D, MT, KS, kGatherTable>(p, stream);
    return launch_mode<D, MT, KS, kGatherInline>(p, stream);
}

template <int D>
cudaError_t launch_d(const AttnParams& p, cudaStream_t stream) {
    switch ((p.rows + 15) / 16) {
        case 1: return launch_cfg<D, 1, 4>(p, stream);
        case 2: return launch_cfg<D, 2, 4>(p, stream);
        case 3: return launch_cfg<D, 3, 2>(p, stream);
        case 4: return launch_cfg<D, 4, 2>(p, stream);
        case 5: return launch_cfg<D, 5, 1>(p, stream);
        case 6: return launch_cfg<D, 6, 1>(p, stream);
        default: return cudaErrorInvalidValue;
    }
}

std::atomic<int> g_split_override{0};
std::atomic<int> g_impl{0};

}  // namespace

void attn_set_impl(int impl) { g_impl.store(impl >= 0 && impl <= 2 ? impl : 0, std::memory_order_relaxed); }
int attn_get_impl() { return g_impl.load(std::memory_order_relaxed); }

void attn_set_split_override(int split_tokens) { g_split_override.store(split_tokens > 0 ? split_tokens : 0, std::memory_order_relaxed); }

// CTAs (= cluster size) per (sequence, KV head): as many as fit one wave of 2 resident CTAs per SM (148 SMs on B200), at
// most the portable cluster size, at least one 64-token tile each; gather lists are cut so that the address table
// of a CTA stays within kMaxTableTokens when the cluster size allows.
void attn_plan(int batch, int n_kv_heads, int max_tokens, int* split_tokens, int* n_splits) {
    const int units = batch * n_kv_heads > 0 ? batch * n_kv_heads : 1;
    int tiles = (max_tokens + kTileTokens - 1) / kTileTokens;
    if (tiles < 1) tiles = 1;
    int ns;
    const int split_override = g_split_override.load(std::memory_order_relaxed);
    if (split_override > 0) {   // dustin_tune_attn_split_tokens
        ns = (max_tokens + split_override - 1) / split_override;
    } else {
        ns = (device_sm_count() * 2) / units;
        const int ns_table = (max_tokens + kMaxTableTokens - 17) / (kMaxTableTokens - 16);
        if (ns < ns_table) ns = ns_table;
    }
    if (ns > kMaxCluster) ns = kMaxCluster;
    if (ns > tiles) ns = tiles;
    if (ns < 1) ns = 1;
    const int tiles_per = (tiles + ns - 1) / ns;
    *split_tokens = tiles_per * kTileTokens;
    *n_splits = (tiles + tiles_per - 1) / tiles_per;
}

cudaError_t launch_attn(const AttnParams& p, cudaStream_t stream) {
    if (p.tc_ws != nullptr) return launch_attn_tc(p, p.tc_ws, stream);
    return p.head_dim == 128 ? launch_d<128>(p, stream) : launch_d<64>(p, stream);
}

}  // namespace dustin
