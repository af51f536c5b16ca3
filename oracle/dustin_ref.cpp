// oracle/dustin_ref.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU restatement (fp64 arithmetic on the bf16-rounded inputs)
// of the per-layer sparse verification attention of "Dustin" (arxiv/paper_2606_24957), written
// from /root/reference/PAPER.md only.  It shares no code, header, table or helper with the CUDA
// path under paper_2606_24957_b200/csrc/.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may load this library.
//
// What each function follows (PAPER.md line : section / equation):
//   dustin_ref_score_heads        :159, :218, :391-393  "target attention tensor of the last generated
//                                 token", recomputed for the SRH subset only; Eq. 5 restricted to one layer
//                                 (sum over the selected heads).  DESIGN.md readings A2-A5.
//   dustin_ref_fuse_scores        :157-164 Eq. 5 (S_Target is a plain sum over heads and layers);
//                                 DESIGN.md reading A6 (S_tgt = alpha*H + A_now).
//   dustin_ref_topk_select        :166-169 Eq. 6 (I_prot, I_draft, I_target, I_verify), :443 (sink and
//                                 recent window are counted inside k).  Readings A7-A12.
//   dustin_ref_sparse_verify_attn :153 ("only the selected KV entries are retrieved ... used to verify the
//                                 speculative draft tokens"), App. G :568.  Reading A13 (T = Gamma+1 rows,
//                                 causal among the new tokens).  idx == NULL gives the full-cache
//                                 verification attention of :248 / :570.
//
//   dustin_ref_arr                :72-75 Eq. 1 (Attention Recovery Rate), Eq. 2-4 by composition.
//   dustin_ref_append_kv          :153 (accepted tokens appended, rejected discarded).
//   dustin_ref_draft_aggregate    :157-161 Eq. 5, first line (S_Draft = sum over draft heads, layers, lookahead tokens).
//   dustin_ref_quest_page_minmax  :401 "aggregates token-level Key statistics (e.g., minimum and maximum values) into
//                                 page-level metadata"; :297 "Quest-16 denotes Quest with page size 16".
//   dustin_ref_quest_score_pages  :51 "scores KV pages using inexpensive min/max key statistics (avoiding exact QK^T)",
//                                 :401 "estimate the relevance of a block of tokens using a single computation".
//                                 The paper names the estimator without its formula: DESIGN.md reading A20 takes the
//                                 channel-wise upper bound of the published method, reading A21 its use as a page-level
//                                 score in the format of O1.
//
// Pins (tests/test_oracle_pins.py): brute force on tiny inputs, closed forms (uniform softmax, one
// planted key, constant V, zero K), library cross-checks (torch fp64 softmax / SDPA, full sort),
// invariants (row sums, membership, thresholds, k = N reproduces dense), printed Eq. 7 arithmetic.
// No function here is "parity unpinned".
//
// Loops only; the one library routine used is std::stable_sort as the "sort" step of TopK.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <algorithm>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// bf16 bit pattern -> exact double (bf16 is the top 16 bits of an IEEE fp32).
inline double bf16_to_double(uint16_t bits) {
    uint32_t u = static_cast<uint32_t>(bits) << 16;
    float f;
    std::memcpy(&f, &u, sizeof f);
    return static_cast<double>(f);
}

struct KvView {
    const uint16_t* k;          // bf16 bits
    const uint16_t* v;
    int64_t stride_seq;         // elements between sequences (contiguous) or between pages (paged)
    int64_t stride_token;       // elements between consecutive tokens of a sequence / inside a page
    int64_t stride_head;        // elements between KV heads
    const int32_t* page_table;  // [batch, max_pages] or nullptr
    int32_t page_size, max_pages;
};

// Element offset of row (b, n, g) of the cache.
inline int64_t row_offset(const KvView& kv, int b, int n, int g) {
    if (kv.page_table == nullptr)
        return (int64_t)b * kv.stride_seq + (int64_t)n * kv.stride_token + (int64_t)g * kv.stride_head;
    int32_t page = kv.page_table[(int64_t)b * kv.max_pages + n / kv.page_size];
    return (int64_t)page * kv.stride_seq + (int64_t)(n % kv.page_size) * kv.stride_token +
           (int64_t)g * kv.stride_head;
}

inline int seq_len(const int32_t* seq_lens, int b, int max_ctx) {
    if (seq_lens == nullptr) return max_ctx;
    int n = seq_lens[b];
    return n < 0 ? 0 : (n > max_ctx ? max_ctx : n);
}

inline double scale_of(float sm_scale, int d) {
    return sm_scale == 0.0f ? 1.0 / std::sqrt((double)d) : (double)sm_scale;
}

}  // namespace

extern "C" {

int dustin_ref_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// ---------------------------------------------------------------------------------------------
// O1 -- head-subset scoring.  For every head h of the subset,
//   l_n = scale * sum_c q[b,h,c] * K[b,n,g(h),c],  p_{h,n} = softmax_n(l)  over the N_b cached tokens
// (reading A4: the normaliser runs over the cached context only), g(h) = h div r (reading A2).
// Eq. 5 for one layer is the plain sum over the subset heads.  n_lists = 1: one list per sequence,
// A[b,0,n] = sum_{h in subset} p_{h,n} (paper, :155).  n_lists = Hkv: A[b,g,n] = sum over the subset
// heads of KV group g; a group with no subset head receives the global sum (reading A2).
// scores_now: fp32 [batch, n_lists, max_ctx]; entries n >= N_b are written as 0.
// ---------------------------------------------------------------------------------------------
int dustin_ref_score_heads(int batch, int n_q_heads, int n_kv_heads, int head_dim, int max_ctx,
                           float sm_scale, const uint16_t* k_cache, int64_t stride_seq,
                           int64_t stride_token, int64_t stride_head, const int32_t* page_table,
                           int page_size, int max_pages, const int32_t* seq_lens, const uint16_t* q,
                           int64_t q_stride_batch, int64_t q_stride_head, uint64_t head_mask,
                           int n_lists, float* scores_now) {
    if (n_q_heads % n_kv_heads != 0 || (n_lists != 1 && n_lists != n_kv_heads)) return -1;
    const int r = n_q_heads / n_kv_heads;
    const double scale = scale_of(sm_scale, head_dim);
    KvView kv{k_cache, nullptr, stride_seq, stride_token, stride_head, page_table, page_size, max_pages};

#pragma omp parallel for schedule(dynamic)
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        // per-group sums and the global sum, in fp64
        std::vector<double> group_sum((size_t)n_kv_heads * N, 0.0), global_sum(N, 0.0);
        std::vector<int> heads_in_group(n_kv_heads, 0);
        std::vector<double> logit(N);
        for (int h = 0; h < n_q_heads; ++h) {
            if (!((head_mask >> h) & 1ull)) continue;
            const int g = h / r;
            heads_in_group[g] += 1;
            const uint16_t* qh = q + (int64_t)b * q_stride_batch + (int64_t)h * q_stride_head;
            double M = -INFINITY;
            for (int n = 0; n < N; ++n) {
                const uint16_t* krow = k_cache + row_offset(kv, b, n, g);
                double acc = 0.0;
                for (int c = 0; c < head_dim; ++c) acc += bf16_to_double(qh[c]) * bf16_to_double(krow[c]);
                logit[n] = acc * scale;
                if (logit[n] > M) M = logit[n];
            }
            double Z = 0.0;
            for (int n = 0; n < N; ++n) Z += std::exp(logit[n] - M);
            for (int n = 0; n < N; ++n) {
                const double p = std::exp(logit[n] - M) / Z;
                group_sum[(size_t)g * N + n] += p;
                global_sum[n] += p;
            }
        }
        for (int l = 0; l < n_lists; ++l) {
            float* dst = scores_now + ((int64_t)b * n_lists + l) * max_ctx;
            const bool use_global = (n_lists == 1) || heads_in_group[l] == 0;
            for (int n = 0; n < max_ctx; ++n) {
                double s = 0.0;
                if (n < N) s = use_global ? global_sum[n] : group_sum[(size_t)l * N + n];
                dst[n] = (float)s;
            }
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O2 -- Eq. 5 accumulation of the target signal (reading A6):
//   H <- alpha * H + A_now   (alpha = 1: plain sum over layers / steps; alpha = 0: H <- A_now).
// fp64 arithmetic, rounded once to fp32.  Entries n >= N_b are left untouched.
// ---------------------------------------------------------------------------------------------
int dustin_ref_fuse_scores(int batch, int n_lists, int max_ctx, const int32_t* seq_lens,
                           const float* scores_now, float* hist_inout, float alpha) {
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        for (int l = 0; l < n_lists; ++l) {
            const int64_t base = ((int64_t)b * n_lists + l) * max_ctx;
            for (int n = 0; n < N; ++n)
                hist_inout[base + n] =
                    (float)((double)alpha * (double)hist_inout[base + n] + (double)scores_now[base + n]);
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O3 -- tiered top-k, Eq. 6 with the protected-set rule of :443.
// Per (b, list):  N = N_b, k = k_b.
//   k >= N            -> everything is selected.
//   I_prot            = [0,S') U [N-W',N),  S' = min(S,N), W' = min(W,N-S')          (A10, A12)
//   c                 = k - |I_prot|,  m' = min(floor(c*m_num/m_den), c)                 (A9)
//   I_draft           = first m' of the candidates [S',N-W') ordered by (S_draft desc, index asc)
//   I_target          = first c-m' of the candidates not in I_draft ordered by (S_target desc, index asc)
//   I_verify          = I_prot U I_draft U I_target, written in ascending index order, tail = -1.
// Scores are compared as max(s, 0) (inputs are probabilities; negative/-0.0 count as 0; NaN undefined).
// ---------------------------------------------------------------------------------------------
int dustin_ref_topk_select(int batch, int max_ctx, const int32_t* seq_lens, int budget,
                           const int32_t* budgets, int n_sink, int n_recent, int m_num, int m_den,
                           int n_lists, const float* s_draft, int64_t draft_list_stride,
                           const float* s_target, int32_t* idx_out, int32_t* cnt_out, int k_max) {
    if (n_sink < 0 || n_recent < 0 || m_num < 0 || m_den <= 0 || m_num > m_den) return -1;
    const int64_t draft_batch_stride = draft_list_stride == 0 ? (int64_t)max_ctx : (int64_t)n_lists * max_ctx;
    int status = 0;
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < batch; ++b) {
        for (int l = 0; l < n_lists; ++l) {
            const int N = seq_len(seq_lens, b, max_ctx);
            int k = budgets ? budgets[b] : budget;
            int32_t* out = idx_out + ((int64_t)b * n_lists + l) * k_max;
            for (int i = 0; i < k_max; ++i) out[i] = -1;
            if (k > k_max || k < n_sink + n_recent) {  // A12: S + W > k is an argument error
#pragma omp critical
                status = -1;
                cnt_out[b * n_lists + l] = 0;
                continue;
            }
            const float* sd = s_draft + (int64_t)b * draft_batch_stride + (int64_t)l * draft_list_stride;
            const float* st = s_target + ((int64_t)b * n_lists + l) * max_ctx;
            std::vector<char> member(N > 0 ? N : 1, 0);
            int cnt;
            if (k >= N) {
                for (int n = 0; n < N; ++n) member[n] = 1;
                cnt = N;
            } else {
                const int S = std::min(n_sink, N);
                const int W = std::min(n_recent, N - S);
                for (int n = 0; n < S; ++n) member[n] = 1;          // I_sink
                for (int n = N - W; n < N; ++n) member[n] = 1;      // I_window
                const int c = k - S - W;
                const int m = (int)std::min<int64_t>((int64_t)c * m_num / m_den, c);
                auto key = [](float s) { return s > 0.0f ? s : 0.0f; };
                // I_draft = TopK(S_Draft \ I_prot, m)
                std::vector<int> cand;
                for (int n = S; n < N - W; ++n) cand.push_back(n);
                std::stable_sort(cand.begin(), cand.end(),
                                 [&](int a, int bb) { return key(sd[a]) > key(sd[bb]); });
                for (int i = 0; i < m && i < (int)cand.size(); ++i) member[cand[i]] = 1;
                // I_target = TopK(S_Target \ (I_prot U I_draft), k - m - |I_prot|)
                std::vector<int> rest;
                for (int n = S; n < N - W; ++n)
                    if (!member[n]) rest.push_back(n);
                std::stable_sort(rest.begin(), rest.end(),
                                 [&](int a, int bb) { return key(st[a]) > key(st[bb]); });
                for (int i = 0; i < c - m && i < (int)rest.size(); ++i) member[rest[i]] = 1;
                cnt = 0;
                for (int n = 0; n < N; ++n) cnt += member[n];
            }
            int w = 0;
            for (int n = 0; n < N; ++n)
                if (member[n]) out[w++] = n;  // ascending order
            cnt_out[b * n_lists + l] = cnt;
        }
    }
    return status;
}

// ---------------------------------------------------------------------------------------------
// O4 -- verification attention over the selected KV plus the new draft KV.
// For every (b, h, t): g = h div r, list l = (n_lists == 1 ? 0 : g); the visible set is the cnt[b,l]
// selected cache rows idx[b,l,:] and the new rows u <= t (causal, inclusive of self; reading A13).
// One joint softmax over that set with scale 1/sqrt(d), O = sum p V, LSE = M + log(sum exp).
// idx == NULL: all N_b cached rows (full-cache verification attention, :248, :570).
// out: fp64 [B,T,Hq,d]; lse: fp64 [B,Hq,T] or NULL.
// ---------------------------------------------------------------------------------------------
int dustin_ref_sparse_verify_attn(int batch, int n_q_heads, int n_kv_heads, int head_dim, int n_new,
                                  int max_ctx, float sm_scale, const uint16_t* k_cache,
                                  const uint16_t* v_cache, int64_t stride_seq, int64_t stride_token,
                                  int64_t stride_head, const int32_t* page_table, int page_size,
                                  int max_pages, const int32_t* seq_lens, const uint16_t* q,
                                  const uint16_t* k_new, const uint16_t* v_new, const int32_t* idx,
                                  const int32_t* cnt, int n_lists, int k_max, double* out, double* lse) {
    if (n_q_heads % n_kv_heads != 0 || (n_lists != 1 && n_lists != n_kv_heads)) return -1;
    const int r = n_q_heads / n_kv_heads, d = head_dim, T = n_new;
    const double scale = scale_of(sm_scale, d);
    KvView kv{k_cache, v_cache, stride_seq, stride_token, stride_head, page_table, page_size, max_pages};

#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < batch; ++b) {
        for (int h = 0; h < n_q_heads; ++h) {
            const int g = h / r;
            const int l = n_lists == 1 ? 0 : g;
            const int N = seq_len(seq_lens, b, max_ctx);
            const int n_sel = idx ? cnt[b * n_lists + l] : N;
            const int32_t* list = idx ? idx + ((int64_t)b * n_lists + l) * k_max : nullptr;
            std::vector<double> logit(n_sel + T);
            for (int t = 0; t < T; ++t) {
                const uint16_t* qrow = q + (((int64_t)b * T + t) * n_q_heads + h) * d;
                const int n_vis = n_sel + t + 1;
                double M = -INFINITY;
                for (int j = 0; j < n_vis; ++j) {
                    const uint16_t* krow;
                    if (j < n_sel) krow = k_cache + row_offset(kv, b, list ? list[j] : j, g);
                    else krow = k_new + (((int64_t)b * T + (j - n_sel)) * n_kv_heads + g) * d;
                    double acc = 0.0;
                    for (int c = 0; c < d; ++c) acc += bf16_to_double(qrow[c]) * bf16_to_double(krow[c]);
                    logit[j] = acc * scale;
                    if (logit[j] > M) M = logit[j];
                }
                double Z = 0.0;
                for (int j = 0; j < n_vis; ++j) Z += std::exp(logit[j] - M);
                double* orow = out + (((int64_t)b * T + t) * n_q_heads + h) * d;
                for (int c = 0; c < d; ++c) orow[c] = 0.0;
                for (int j = 0; j < n_vis; ++j) {
                    const double p = std::exp(logit[j] - M) / Z;
                    const uint16_t* vrow;
                    if (j < n_sel) vrow = v_cache + row_offset(kv, b, list ? list[j] : j, g);
                    else vrow = v_new + (((int64_t)b * T + (j - n_sel)) * n_kv_heads + g) * d;
                    for (int c = 0; c < d; ++c) orow[c] += p * bf16_to_double(vrow[c]);
                }
                if (lse) lse[((int64_t)b * n_q_heads + h) * T + t] = M + std::log(Z);
            }
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O5 -- Attention Recovery Rate, Eq. 1: ARR = sum_{j in K} A_j where A is normalised over the
// valid positions V = [0, N_b) (sum_{j in V} A_j = 1).  `a` arrives as any non-negative weights (e.g. the
// per-list sums of O1, which add up to the number of heads) and is normalised here: ARR = sum_K a / sum_V a;
// a row without mass gives 0.  K = the cnt[b,l] DISTINCT entries idx[b,l,:] (a set, as in Eq. 1).
// The windowed form (Eq. 2) and the SD-oracle bound (Eq. 3-4) follow by passing the window mean of A (Eq. 3's
// A-bar; a window SUM gives the same ratio) and, for Eq. 4, K = TopK_k(A-bar) from O3 with m = 0, S = W = 0.
// arr_out: fp64 [batch, n_lists].
// ---------------------------------------------------------------------------------------------
int dustin_ref_arr(int batch, int n_lists, int max_ctx, const int32_t* seq_lens, const float* a,
                   const int32_t* idx, const int32_t* cnt, int k_max, double* arr_out) {
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        for (int l = 0; l < n_lists; ++l) {
            const float* row = a + ((int64_t)b * n_lists + l) * max_ctx;
            double total = 0.0;
            for (int n = 0; n < N; ++n) total += (double)row[n];
            const int32_t* list = idx + ((int64_t)b * n_lists + l) * k_max;
            int c = cnt[(int64_t)b * n_lists + l];
            c = c < 0 ? 0 : (c > k_max ? k_max : c);
            double kept = 0.0;
            for (int i = 0; i < c; ++i)
                if (list[i] >= 0 && list[i] < N) kept += (double)row[list[i]];
            arr_out[(int64_t)b * n_lists + l] = total > 0.0 ? kept / total : 0.0;
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O6 -- KV append after verification ("accepted tokens are appended to the KV cache, rejected ones
// are discarded"; App. C.4 :453-466).  The first n_append[b] rows of the verify block (reading A13: row 0 is the
// last generated token, rows 1.. the accepted draft tokens) become cache rows N_b, N_b+1, ... of sequence b; rows
// that would not fit into max_ctx are dropped; seq_lens[b] grows accordingly.  When hist != NULL the accumulated
// target scores of the new positions start from 0 (Eq. 5 is a sum and nothing has been added yet).
// ---------------------------------------------------------------------------------------------
int dustin_ref_append_kv(int batch, int n_kv_heads, int head_dim, int n_new, int max_ctx, uint16_t* k_cache,
                         uint16_t* v_cache, int64_t stride_seq, int64_t stride_token, int64_t stride_head,
                         const int32_t* page_table, int page_size, int max_pages, int32_t* seq_lens,
                         const uint16_t* k_new, const uint16_t* v_new, const int32_t* n_append, float* hist,
                         int n_lists) {
    if (!seq_lens || !n_append) return -1;
    KvView kv{k_cache, v_cache, stride_seq, stride_token, stride_head, page_table, page_size, max_pages};
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        int a = n_append[b];
        a = a < 0 ? 0 : (a > n_new ? n_new : a);
        if (N + a > max_ctx) a = max_ctx - N;
        for (int u = 0; u < a; ++u)
            for (int g = 0; g < n_kv_heads; ++g) {
                const int64_t dst = row_offset(kv, b, N + u, g);
                const int64_t src = (((int64_t)b * n_new + u) * n_kv_heads + g) * head_dim;
                for (int c = 0; c < head_dim; ++c) {
                    k_cache[dst + c] = k_new[src + c];
                    v_cache[dst + c] = v_new[src + c];
                }
            }
        if (hist)
            for (int l = 0; l < n_lists; ++l)
                for (int u = 0; u < a; ++u) hist[((int64_t)b * n_lists + l) * max_ctx + N + u] = 0.0f;
        seq_lens[b] = N + a;
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O7 -- draft-side lookahead aggregation, Eq. 5 first line:
//   S_Draft[n] = sum_{h in H_d} sum_{l in L_sel} sum_{gamma < Gamma} A^Draft_{h,l,n,gamma},
// A^Draft_{h,l,.,gamma} = softmax over the N_b cached context tokens (reading A4) of the draft model's query of
// lookahead token gamma, head h, layer l, against that layer's K cache.  One global vector per sequence
// (PAPER.md:155).  Layer l's cache and queries are layer_k[l] (same strides / page table for all layers) and
// layer_q[l] = bf16 [batch, n_gamma, n_q_heads, head_dim].  s_draft: fp32 [batch, max_ctx], written (0 for n >= N_b).
// ---------------------------------------------------------------------------------------------
int dustin_ref_draft_aggregate(int batch, int n_q_heads, int n_kv_heads, int head_dim, int n_gamma, int max_ctx,
                               float sm_scale, int n_layers, const uint16_t* const* layer_k, int64_t stride_seq,
                               int64_t stride_token, int64_t stride_head, const int32_t* page_table, int page_size,
                               int max_pages, const int32_t* seq_lens, const uint16_t* const* layer_q,
                               uint64_t head_mask, float* s_draft) {
    if (n_q_heads % n_kv_heads != 0) return -1;
    const int r = n_q_heads / n_kv_heads;
    const double scale = scale_of(sm_scale, head_dim);
#pragma omp parallel for schedule(dynamic)
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        std::vector<double> sum(N, 0.0), logit(N);
        for (int l = 0; l < n_layers; ++l) {
            KvView kv{layer_k[l], nullptr, stride_seq, stride_token, stride_head, page_table, page_size, max_pages};
            for (int gam = 0; gam < n_gamma; ++gam)
                for (int h = 0; h < n_q_heads; ++h) {
                    if (!((head_mask >> h) & 1ull)) continue;
                    const int g = h / r;
                    const uint16_t* qh = layer_q[l] + (((int64_t)b * n_gamma + gam) * n_q_heads + h) * head_dim;
                    double M = -INFINITY;
                    for (int n = 0; n < N; ++n) {
                        const uint16_t* krow = layer_k[l] + row_offset(kv, b, n, g);
                        double acc = 0.0;
                        for (int c = 0; c < head_dim; ++c) acc += bf16_to_double(qh[c]) * bf16_to_double(krow[c]);
                        logit[n] = acc * scale;
                        if (logit[n] > M) M = logit[n];
                    }
                    double Z = 0.0;
                    for (int n = 0; n < N; ++n) Z += std::exp(logit[n] - M);
                    for (int n = 0; n < N; ++n) sum[n] += std::exp(logit[n] - M) / Z;
                }
        }
        float* dst = s_draft + (int64_t)b * max_ctx;
        for (int n = 0; n < max_ctx; ++n) dst[n] = n < N ? (float)sum[n] : 0.0f;
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O8 -- page-level key metadata of the Quest-style estimator (page size 16).
// Logical page p of sequence b holds the tokens [p*P, (p+1)*P) that exist (n < N_b), whatever the physical layout of
// the cache.  Per (b, p, KV head g, channel c):  kmin = min_n K[b,n,g,c],  kmax = max_n K[b,n,g,c].
// A page without any token (p*P >= N_b) gets kmin = kmax = 0.   Outputs: fp64 [batch, n_pages, n_kv_heads, head_dim]
// with n_pages = ceil(max_ctx / P)  (the values are bf16 numbers, so any float type holds them exactly).
// ---------------------------------------------------------------------------------------------
int dustin_ref_quest_page_minmax(int batch, int n_kv_heads, int head_dim, int max_ctx, const uint16_t* k_cache,
                                 int64_t stride_seq, int64_t stride_token, int64_t stride_head,
                                 const int32_t* page_table, int page_size, int max_pages, const int32_t* seq_lens,
                                 int quest_page, double* kmin_out, double* kmax_out) {
    if (quest_page <= 0) return -1;
    KvView kv{k_cache, nullptr, stride_seq, stride_token, stride_head, page_table, page_size, max_pages};
    const int n_pages = (max_ctx + quest_page - 1) / quest_page;
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        for (int p = 0; p < n_pages; ++p)
            for (int g = 0; g < n_kv_heads; ++g)
                for (int c = 0; c < head_dim; ++c) {
                    double lo = 0.0, hi = 0.0;
                    bool any = false;
                    for (int n = p * quest_page; n < (p + 1) * quest_page && n < N; ++n) {
                        const double x = bf16_to_double(k_cache[row_offset(kv, b, n, g) + c]);
                        if (!any || x < lo) lo = x;
                        if (!any || x > hi) hi = x;
                        any = true;
                    }
                    const int64_t o = (((int64_t)b * n_pages + p) * n_kv_heads + g) * head_dim + c;
                    kmin_out[o] = lo;
                    kmax_out[o] = hi;
                }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O9 -- page scores from the metadata alone (readings A20, A21).
// For every subset head h (KV group g = h div r) and every page p that holds a token (p*P < N_b):
//   U_h[p] = scale * sum_c max(q[b,h,c] * kmin[b,p,g,c], q[b,h,c] * kmax[b,p,g,c])
// -- per channel the larger of the two products bounds q_c * k_c for every key of the page, so U_h[p] is an upper
// bound of every exact logit scale * q.k_n inside the page, computed without touching K (A20).
//   P_h[p] = softmax_p(U_h) over the pages that hold a token;  page_scores[b,l,p] = sum of P_h over the subset heads
// feeding list l, with the list rule of O1 (n_lists = 1: all subset heads; n_lists = Hkv: the heads of KV group l, a
// group without a subset head receives the sum over all subset heads) (A21).  Pages without a token score 0.
//   kmin, kmax: fp64 [batch, n_pages, n_kv_heads, head_dim] (O8);  q as in O1.
//   page_scores: fp32 [batch, n_lists, n_pages];  ub_out (optional): fp64 [batch, n_q_heads, n_pages], U_h[p] for the
//   subset heads (0 elsewhere).
// ---------------------------------------------------------------------------------------------
int dustin_ref_quest_score_pages(int batch, int n_q_heads, int n_kv_heads, int head_dim, int max_ctx, float sm_scale,
                                 const int32_t* seq_lens, int quest_page, const double* kmin, const double* kmax,
                                 const uint16_t* q, int64_t q_stride_batch, int64_t q_stride_head, uint64_t head_mask,
                                 int n_lists, float* page_scores, double* ub_out) {
    if (quest_page <= 0 || n_q_heads % n_kv_heads != 0 || (n_lists != 1 && n_lists != n_kv_heads)) return -1;
    const int r = n_q_heads / n_kv_heads;
    const double scale = scale_of(sm_scale, head_dim);
    const int n_pages = (max_ctx + quest_page - 1) / quest_page;
    for (int b = 0; b < batch; ++b) {
        const int N = seq_len(seq_lens, b, max_ctx);
        const int n_live = (N + quest_page - 1) / quest_page;   // pages that hold a token
        std::vector<double> group_sum((size_t)n_kv_heads * n_pages, 0.0), global_sum(n_pages, 0.0), U(n_pages);
        std::vector<int> heads_in_group(n_kv_heads, 0);
        for (int h = 0; h < n_q_heads; ++h) {
            if (ub_out)
                for (int p = 0; p < n_pages; ++p) ub_out[((int64_t)b * n_q_heads + h) * n_pages + p] = 0.0;
            if (!((head_mask >> h) & 1ull)) continue;
            const int g = h / r;
            heads_in_group[g] += 1;
            const uint16_t* qh = q + (int64_t)b * q_stride_batch + (int64_t)h * q_stride_head;
            double M = -INFINITY;
            for (int p = 0; p < n_live; ++p) {
                const int64_t o = (((int64_t)b * n_pages + p) * n_kv_heads + g) * head_dim;
                double acc = 0.0;
                for (int c = 0; c < head_dim; ++c) {
                    const double qc = bf16_to_double(qh[c]);
                    acc += std::max(qc * kmin[o + c], qc * kmax[o + c]);
                }
                U[p] = acc * scale;
                if (U[p] > M) M = U[p];
                if (ub_out) ub_out[((int64_t)b * n_q_heads + h) * n_pages + p] = U[p];
            }
            double Z = 0.0;
            for (int p = 0; p < n_live; ++p) Z += std::exp(U[p] - M);
            for (int p = 0; p < n_live; ++p) {
                const double pr = std::exp(U[p] - M) / Z;
                group_sum[(size_t)g * n_pages + p] += pr;
                global_sum[p] += pr;
            }
        }
        for (int l = 0; l < n_lists; ++l) {
            float* dst = page_scores + ((int64_t)b * n_lists + l) * n_pages;
            const bool use_global = (n_lists == 1) || heads_in_group[l] == 0;
            for (int p = 0; p < n_pages; ++p) {
                double sc = 0.0;
                if (p < n_live) sc = use_global ? global_sum[p] : group_sum[(size_t)l * n_pages + p];
                dst[p] = (float)sc;
            }
        }
    }
    return 0;
}

}  // extern "C"
