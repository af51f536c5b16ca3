// attn.cu -- stage a4 (sparse verification attention over the selected KV, App. G :568) and a5
// (the full-cache verification baseline of PAPER.md:248 / :570: same kernel, idx == nullptr) for sm_100a.
//
// Flash-style, index-driven, split over the selected tokens:
//   grid = (n_splits, Hkv, B); a CTA owns `split_tokens` entries of the index list of (b, KV head) -- split 0
//   also owns the T new draft rows (causal among themselves).  Row offsets are resolved once into shared memory
//   (index -> page table -> element offset); K/V rows then stream global -> shared with 16-byte cp.async through
//   a 3-stage ring (XOR-swizzled, ldmatrix-conflict-free).  All T*r query rows that share the KV head sit on the
//   M axis of bf16 mma.sync tiles (warp = one 16-row tile x one token slice), fp32 online softmax in the log2
//   domain, P re-used from the accumulator registers as the A operand of P.V.  Token slices of a CTA merge in
//   shared memory; CTAs of one (b, KV head) merge in attn_combine_kernel (n_splits > 1).
#include "kernels.cuh"

namespace dustin {

namespace {

constexpr int kTileTokens = 64;   // tokens per pipeline stage
constexpr int kStages = 3;
constexpr int kMaxSplitTokens = 4096;

template <int D, int MT, int KS>
struct AttnCfg {
    static constexpr int kThreads = 32 * MT * KS;
    static constexpr int kWT = kTileTokens / KS;          // tokens per warp per stage
    static constexpr int kCH = D / 8;                     // 16-byte chunks per row
    static constexpr int kStageElems = kTileTokens * D;   // bf16 elements per K (or V) stage
    static constexpr int kOReg = D / 2;                   // fp32 accumulators per thread (16 x D tile)
    static constexpr size_t kPipeBytes = (size_t)kStages * kStageElems * 2 * 2;
    static constexpr size_t kMergeBytes = (size_t)(KS - 1) * MT * 32 * (kOReg + 4) * 4;
};

template <int D, int MT, int KS>
__global__ void __launch_bounds__(32 * MT * KS) attn_kernel(const AttnParams p) {
    using C = AttnCfg<D, MT, KS>;
    constexpr int WT = C::kWT, CH = C::kCH, NT = C::kThreads;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __nv_bfloat16* sK = reinterpret_cast<__nv_bfloat16*>(smem_raw);
    __nv_bfloat16* sV = sK + kStages * C::kStageElems;
    long long* sOff = reinterpret_cast<long long*>(smem_raw + (C::kPipeBytes > C::kMergeBytes ? C::kPipeBytes
                                                                                             : C::kMergeBytes));

    const int split = blockIdx.x, gkv = blockIdx.y, b = blockIdx.z;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int mt = warp % MT, ks = warp / MT;
    const int g = lane >> 2, c = lane & 3;
    const int T = p.n_new, r = p.group, rows = p.rows;
    const int list = p.n_lists == 1 ? 0 : gkv;
    const int n_sel = p.idx ? p.cnt[b * p.n_lists + list] : seq_len_of(p.kv.seq_lens, b, p.max_ctx);
    const int range_lo = split * p.split_tokens;
    const int n_range = max(0, min(p.split_tokens, n_sel - range_lo));
    const int nt = n_range + (split == 0 ? T : 0);        // this CTA's tokens: cache rows, then the new rows

    // ---- row offsets (elements): >= 0 in the cache, -(1 + off) in k_new / v_new --------------------------------
    {
        const int* list_idx = p.idx ? p.idx + ((long long)b * p.n_lists + list) * p.k_max + range_lo : nullptr;
        for (int j = tid; j < nt; j += NT) {
            long long off;
            if (j < n_range) {
                const int tok = list_idx ? __ldg(list_idx + j) : range_lo + j;
                off = kv_row_offset(p.kv, b, tok, gkv);
            } else {
                off = -1 - (((long long)b * T + (j - n_range)) * p.n_kv_heads + gkv) * D;
            }
            sOff[j] = off;
        }
    }

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

    const int n_tiles = (nt + kTileTokens - 1) / kTileTokens;
    auto issue = [&](int tile) {
        if (tile < n_tiles) {
            const int slot = tile % kStages;
#pragma unroll 4
            for (int i = tid; i < 2 * kTileTokens * CH; i += NT) {
                const int which = i / (kTileTokens * CH);
                const int rem = i - which * (kTileTokens * CH);
                const int row = rem / CH, ch = rem % CH;
                const int j = tile * kTileTokens + row;
                const bool valid = j < nt;
                const long long off = valid ? sOff[j] : 0;
                const __nv_bfloat16* base = which ? (off >= 0 ? p.kv.v : p.v_new) : (off >= 0 ? p.kv.k : p.k_new);
                const __nv_bfloat16* src = base + (off >= 0 ? off : -1 - off) + ch * 8;
                __nv_bfloat16* dst = (which ? sV : sK) + slot * C::kStageElems + row * D + ((ch ^ (row & 7)) << 3);
                cp_async16(smem_u32(dst), src, valid ? 16 : 0);
            }
        }
        cp_async_commit();
    };

    float o[D / 8][4];
#pragma unroll
    for (int i = 0; i < D / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
    float m_lo = -INFINITY, m_hi = -INFINITY, l_lo = 0.f, l_hi = 0.f;
    const int t_lo = (mt * 16 + g) / r, t_hi = (mt * 16 + g + 8) / r;   // verify position of this thread's rows

#pragma unroll
    for (int s = 0; s < kStages - 1; ++s) issue(s);

    for (int tile = 0; tile < n_tiles; ++tile) {
        cp_async_wait<kStages - 2>();
        __syncthreads();
        issue(tile + kStages - 1);
        const int j0 = tile * kTileTokens + ks * WT;       // first token of this warp's slice
        if (j0 >= nt) continue;
        const __nv_bfloat16* tK = sK + (tile % kStages) * C::kStageElems;
        const __nv_bfloat16* tV = sV + (tile % kStages) * C::kStageElems;

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
                ldmatrix_x4(b0, b1, b2, b3, smem_u32(tK + row * D + ((ch ^ (row & 7)) << 3)));
                mma_bf16_16816(sc[2 * np], qa[kk][0], qa[kk][1], qa[kk][2], qa[kk][3], b0, b1);
                mma_bf16_16816(sc[2 * np + 1], qa[kk][0], qa[kk][1], qa[kk][2], qa[kk][3], b2, b3);
            }
        }

        // scale, mask (tail of the list; causality among the new rows), online softmax in the log2 domain
        const bool need_mask = j0 + WT > n_range;
        float mx_lo = -INFINITY, mx_hi = -INFINITY;
#pragma unroll
        for (int i = 0; i < WT / 8; ++i) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float v = sc[i][e] * p.scale_log2;
                if (need_mask) {
                    const int j = j0 + i * 8 + 2 * c + (e & 1);
                    const int t = (e & 2) ? t_hi : t_lo;
                    if (j >= nt || (j >= n_range && j - n_range > t)) v = -INFINITY;
                }
                sc[i][e] = v;
            }
            mx_lo = fmaxf(mx_lo, fmaxf(sc[i][0], sc[i][1]));
            mx_hi = fmaxf(mx_hi, fmaxf(sc[i][2], sc[i][3]));
        }
        mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 1));
        mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 2));
        mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 1));
        mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 2));
        const float mn_lo = fmaxf(m_lo, mx_lo), mn_hi = fmaxf(m_hi, mx_hi);
        const float mu_lo = mn_lo == -INFINITY ? 0.f : mn_lo, mu_hi = mn_hi == -INFINITY ? 0.f : mn_hi;
        const float al_lo = fast_exp2(m_lo - mu_lo), al_hi = fast_exp2(m_hi - mu_hi);
        m_lo = mn_lo;
        m_hi = mn_hi;
        float sum_lo = 0.f, sum_hi = 0.f;
#pragma unroll
        for (int i = 0; i < WT / 8; ++i) {
            sc[i][0] = fast_exp2(sc[i][0] - mu_lo);
            sc[i][1] = fast_exp2(sc[i][1] - mu_lo);
            sc[i][2] = fast_exp2(sc[i][2] - mu_hi);
            sc[i][3] = fast_exp2(sc[i][3] - mu_hi);
            sum_lo += sc[i][0] + sc[i][1];
            sum_hi += sc[i][2] + sc[i][3];
        }
        l_lo = l_lo * al_lo + sum_lo;
        l_hi = l_hi * al_hi + sum_hi;
#pragma unroll
        for (int i = 0; i < D / 8; ++i) {
            o[i][0] *= al_lo;
            o[i][1] *= al_lo;
            o[i][2] *= al_hi;
            o[i][3] *= al_hi;
        }

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
                ldmatrix_x4_trans(b0, b1, b2, b3, smem_u32(tV + row * D + ((ch ^ (row & 7)) << 3)));
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
    if (ks != 0) return;

    // ---- write: final bf16 output (one split) or the normalised fp32 partial + log2 normaliser -----------------
    const float inv_lo = l_lo > 0.f ? 1.f / l_lo : 0.f, inv_hi = l_hi > 0.f ? 1.f / l_hi : 0.f;
    const float lse_lo = l_lo > 0.f ? m_lo + log2f(l_lo) : -INFINITY;
    const float lse_hi = l_hi > 0.f ? m_hi + log2f(l_hi) : -INFINITY;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        const int row = mt * 16 + g + half * 8;
        if (row >= rows) continue;
        const float inv = half ? inv_hi : inv_lo, lse = half ? lse_hi : lse_lo;
        if (p.n_splits == 1) {
            const int t = row / r, h = gkv * r + row % r;
            __nv_bfloat16* dst = p.out + (((long long)b * T + t) * p.n_q_heads + h) * D + 2 * c;
#pragma unroll
            for (int i = 0; i < D / 8; ++i)
                *reinterpret_cast<uint32_t*>(dst + i * 8) = pack_bf16(o[i][half * 2] * inv, o[i][half * 2 + 1] * inv);
            if (p.lse_out && c == 0) p.lse_out[((long long)b * p.n_q_heads + h) * T + t] = lse * kLn2;
        } else {
            const long long pr = (((long long)b * p.n_kv_heads + gkv) * p.n_splits + split) * rows + row;
            float* dst = p.part_o + pr * D + 2 * c;
#pragma unroll
            for (int i = 0; i < D / 8; ++i)
                *reinterpret_cast<float2*>(dst + i * 8) = make_float2(o[i][half * 2] * inv, o[i][half * 2 + 1] * inv);
            if (c == 0) p.part_lse[pr] = lse;
        }
    }
}

// One warp per (b, KV head, query row): weighted sum of the split partials.
template <int D>
__global__ void __launch_bounds__(128) attn_combine_kernel(const AttnParams p) {
    const int w = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    const int rows = p.rows;
    if (w >= p.batch * p.n_kv_heads * rows) return;
    const int row = w % rows, bg = w / rows;
    const int b = bg / p.n_kv_heads, gkv = bg % p.n_kv_heads;
    const long long base = (long long)bg * p.n_splits * rows + row;
    float M = -INFINITY;
    for (int s = 0; s < p.n_splits; ++s) M = fmaxf(M, __ldcg(p.part_lse + base + (long long)s * rows));
    constexpr int V = D / 32;
    float acc[V];
#pragma unroll
    for (int i = 0; i < V; ++i) acc[i] = 0.f;
    float W = 0.f;
    for (int s = 0; s < p.n_splits; ++s) {
        const float lse = __ldcg(p.part_lse + base + (long long)s * rows);
        const float wgt = lse == -INFINITY ? 0.f : exp2f(lse - M);
        W += wgt;
        const float* src = p.part_o + (base + (long long)s * rows) * D + lane * V;
        if (wgt != 0.f) {
#pragma unroll
            for (int i = 0; i < V; i += 2) {
                const float2 x = __ldcg(reinterpret_cast<const float2*>(src + i));
                acc[i] += wgt * x.x;
                acc[i + 1] += wgt * x.y;
            }
        }
    }
    const float inv = W > 0.f ? 1.f / W : 0.f;
    const int t = row / p.group, h = gkv * p.group + row % p.group;
    __nv_bfloat16* dst = p.out + (((long long)b * p.n_new + t) * p.n_q_heads + h) * D + lane * V;
#pragma unroll
    for (int i = 0; i < V; i += 2) *reinterpret_cast<uint32_t*>(dst + i) = pack_bf16(acc[i] * inv, acc[i + 1] * inv);
    if (p.lse_out && lane == 0)
        p.lse_out[((long long)b * p.n_q_heads + h) * p.n_new + t] = W > 0.f ? (M + log2f(W)) * kLn2 : -INFINITY;
}

template <int D, int MT, int KS>
cudaError_t launch_cfg(const AttnParams& p, cudaStream_t stream) {
    using C = AttnCfg<D, MT, KS>;
    const size_t smem = (C::kPipeBytes > C::kMergeBytes ? C::kPipeBytes : C::kMergeBytes) +
                        (size_t)(p.split_tokens + 16) * sizeof(long long);
    static bool attr_done = false;   // per instantiation
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(attn_kernel<D, MT, KS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)(C::kPipeBytes + (kMaxSplitTokens + 16) * sizeof(long long)));
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    ProfScope prof(kKernAttn, stream);
    attn_kernel<D, MT, KS><<<dim3(p.n_splits, p.n_kv_heads, p.batch), C::kThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

template <int D>
cudaError_t launch_d(const AttnParams& p, cudaStream_t stream) {
    const int mt = (p.rows + 15) / 16;
    cudaError_t e;
    switch (mt) {
        case 1: e = launch_cfg<D, 1, 4>(p, stream); break;
        case 2: e = launch_cfg<D, 2, 4>(p, stream); break;
        case 3: e = launch_cfg<D, 3, 2>(p, stream); break;
        case 4: e = launch_cfg<D, 4, 2>(p, stream); break;
        case 5: e = launch_cfg<D, 5, 1>(p, stream); break;
        case 6: e = launch_cfg<D, 6, 1>(p, stream); break;
        default: return cudaErrorInvalidValue;
    }
    if (e != cudaSuccess || p.n_splits == 1) return e;
    const int warps = p.batch * p.n_kv_heads * p.rows;
    ProfScope prof(kKernAttnCombine, stream);
    attn_combine_kernel<D><<<(warps + 3) / 4, 128, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace

static int g_split_override = 0;
void attn_set_split_override(int split_tokens) { g_split_override = split_tokens > 0 ? split_tokens : 0; }

void attn_plan(int batch, int n_kv_heads, int max_tokens, int* split_tokens, int* n_splits) {
    const int units = batch * n_kv_heads > 0 ? batch * n_kv_heads : 1;
    int target = 148 * 4;   // CTAs wanted in flight: 148 SMs x the CTAs resident per SM
    int st = g_split_override;   // dustin_tune_attn_split_tokens
    if (st <= 0) {
        int ns = (target + units - 1) / units;
        if (ns < 1) ns = 1;
        st = (max_tokens + ns - 1) / ns;
    }
    st = ((st + kTileTokens - 1) / kTileTokens) * kTileTokens;
    if (st < kTileTokens) st = kTileTokens;
    if (st > kMaxSplitTokens) st = kMaxSplitTokens;
    int ns = (max_tokens + st - 1) / st;
    if (ns < 1) ns = 1;
    *split_tokens = st;
    *n_splits = ns;
}

cudaError_t launch_attn(const AttnParams& p, cudaStream_t stream) {
    return p.head_dim == 128 ? launch_d<128>(p, stream) : launch_d<64>(p, stream);
}

}  // namespace dustin
