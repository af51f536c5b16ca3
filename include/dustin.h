/* dustin.h -- C ABI of the B200-native sparse verification attention of "Dustin" (arxiv/paper_2606_24957).
 *
 * One decoder layer's sparse verification is four device stages:
 *   a1 dustin_score_heads        head-subset scoring against the full KV cache
 *   a2 dustin_fuse_scores        Eq. 5 accumulation of the target signal           PAPER.md:157-164 (Eq. 5)
 *   a3 dustin_topk_select        tiered top-k with protected sink + window         PAPER.md:166-169 (Eq. 6), :443
 *   a4 dustin_sparse_verify_attn (gamma+1)-query attention over the selected KV    PAPER.md:153, App. G :568
 *   a5 the same call with idx == NULL is the full-cache verification baseline
 *   a6 dustin_verify_layer_fused a1..a4 enqueued on one stream, no host sync
 * and the steps either side of it: dustin_arr (Eq. 1-4), dustin_append_kv,
 * dustin_draft_aggregate (Eq. 5, first line), the Quest-16 page estimator of Fig. 8 (dustin_quest_*).  Measurement / tuning / testing aids live in dustin_debug.h.
 *
 * Conventions (all entry points):
 *  - Every pointer marked "device" is a CUDA device pointer owned by the caller; the library never allocates,
 *    frees, synchronises, or dereferences device memory on the host.  Structs and scalars are host values.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Work is only enqueued.
 *  - Return value: DUSTIN_OK (0) or a negative dustin_status.  Only host-visible arguments are validated.
 *    No exception crosses the ABI.  After DUSTIN_ERR_CUDA, dustin_last_cuda_error() gives the cudaError_t.
 *  - bf16 tensors are raw 16-bit patterns; the last (head_dim) dimension is contiguous; 16-byte aligned rows.
 *  - Outputs are fully overwritten; `hist_inout` is the only in/out state.  Identical inputs give
 *    bit-identical outputs (no order-dependent floating-point atomics anywhere).
 *  - Thread safety: the entry points keep no mutable state of their own (per-device launch attributes are set once
 *    under std::call_once-style guards; the library reads no environment variable); calls on different streams and
 *    workspaces may come from different host threads.  Any device of the process may be current.
 *  - Limits: head_dim in {64,128}; n_q_heads <= 64 (the head subset is a 64-bit mask); n_new (T) <= 16;
 *    T * (n_q_heads / n_kv_heads) <= 96 query rows per KV head; at most 8 subset heads per KV group;
 *    max_ctx <= 2^20.  Outside them the call returns DUSTIN_ERR_UNSUPPORTED.
 */
#ifndef DUSTIN_H_
#define DUSTIN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DUSTIN_VERSION 100 /* 0.1.0 */

typedef enum dustin_status {
    DUSTIN_OK = 0,
    DUSTIN_ERR_INVALID_ARG = -1,   /* null pointer, negative size, Hq % Hkv != 0, S + W > k, empty head mask ...  */
    DUSTIN_ERR_UNSUPPORTED = -2,   /* a documented limit above is exceeded                                         */
    DUSTIN_ERR_WORKSPACE = -3,     /* ws == NULL or ws_bytes < dustin_workspace_bytes(...)                          */
    DUSTIN_ERR_CUDA = -4,          /* a launch failed; see dustin_last_cuda_error()                                 */
    DUSTIN_ERR_STATIC_SCRATCH = -5 /* dustin_score_heads_static only: the shape needs more scratch than
                                      DUSTIN_STATIC_SCRATCH_BYTES; nothing was enqueued                             */
} dustin_status;

/* Problem shape of one layer call.  T = n_new = gamma + 1 verify positions (reading A13). */
typedef struct dustin_shape {
    int32_t batch;       /* B                                                                                   */
    int32_t n_q_heads;   /* Hq                                                                                  */
    int32_t n_kv_heads;  /* Hkv; KV group of query head h is g = h / (Hq / Hkv)  (reading A2)                    */
    int32_t head_dim;    /* d                                                                                   */
    int32_t n_new;       /* T = gamma + 1                                                                       */
    int32_t max_ctx;     /* N: row length of every [.., N] score tensor; N_b <= N                               */
    float   sm_scale;    /* softmax scale; 0 => 1/sqrt(d)  (reading A5)                                         */
} dustin_shape_t;

/* bf16 GQA KV cache, contiguous or paged.  Strides are in ELEMENTS.
 * Contiguous (page_table == NULL): row (b, n, g) starts at  b*stride_seq + n*stride_token + g*stride_head.
 * Paged: row (b, n, g) starts at  page_table[b*max_pages + n/page_size]*stride_seq + (n%page_size)*stride_token
 *        + g*stride_head  (stride_seq is then the page stride).  k and v share the layout. */
typedef struct dustin_kv {
    const void*    k;            /* device, bf16                                                                */
    const void*    v;            /* device, bf16 (may be NULL for dustin_score_heads)                            */
    int64_t        stride_seq;
    int64_t        stride_token;
    int64_t        stride_head;
    const int32_t* page_table;   /* device int32 [batch, max_pages] or NULL                                      */
    int32_t        page_size;
    int32_t        max_pages;
    const int32_t* seq_lens;     /* device int32 [batch] (N_b, clamped to [0, max_ctx]) or NULL => all max_ctx   */
} dustin_kv_t;

/* Selection rule of Eq. 6.  S and W are counted inside k. */
typedef struct dustin_select {
    int32_t        budget;    /* k, used when budgets == NULL                                                     */
    const int32_t* budgets;   /* device int32 [batch] per-sequence k_b, or NULL; every k_b must be <= k_max and
                                 >= n_sink + n_recent (a violating row gets cnt = 0 and an all -1 list)          */
    int32_t        n_sink;    /* S: tokens [0, S) always kept                                                     */
    int32_t        n_recent;  /* W: tokens [N_b - W, N_b) always kept                                             */
    int32_t        m_num;     /* draft quota m = floor((k - S - W) * m_num / m_den)  (reading A9)                 */
    int32_t        m_den;     /*   0 <= m_num <= m_den, m_den > 0                                                 */
    int32_t        n_lists;   /* G: 1 (one list per sequence) or n_kv_heads (per KV head)           */
} dustin_select_t;

int         dustin_version(void);
const char* dustin_status_string(int status);
int         dustin_last_cuda_error(void);            /* cudaError_t of the last failed launch on this thread     */

/* Workspace.  The first DUSTIN_WS_HEADER_BYTES of a workspace persist between calls (completion flags of the
 * attention kernel): they must be ZERO before the first call that uses the buffer and must not
 * be written by the caller afterwards; every call that returns DUSTIN_OK and runs to completion leaves them zero
 * again, so one memset at allocation time serves any number of calls (and CUDA-graph replays).  The rest of the
 * buffer is plain scratch with no state.  One workspace must not be used by two calls that run concurrently.
 * After a failure (a call returned DUSTIN_ERR_CUDA, or a kernel of this library was aborted by a fault that left the
 * context usable) the header may hold flags of the aborted launch: zero it again (cudaMemsetAsync of
 * DUSTIN_WS_HEADER_BYTES on the same stream) before reusing the buffer.
 * cudaDeviceReset is NOT a supported recovery: the library remembers, per device and for the life of the process, that
 * it has raised its kernels' dynamic shared-memory limits there (and, for dustin_score_heads_static, a device address);
 * a reset silently undoes the former and invalidates the latter, after which launches fail with DUSTIN_ERR_CUDA.
 * Restart the process (or unload and reload the library) after a device reset.
 * Forward progress of the attention kernel when one (sequence, KV head) is cut across several CTAs (long or ragged
 * units): the CTA that merges a unit waits for partial results of CTAs with LOWER block indices only.  That the kernel
 * then needs no co-residency of its whole grid (MPS partitions, green contexts, concurrent kernels on other streams)
 * rests on an IMPLEMENTATION ASSUMPTION, not on a documented CUDA guarantee: that CTAs of a grid are dispatched in
 * ascending block-index order, as on every current GPU (decoupled look-back scans and stream-K GEMMs rely on the same
 * behaviour).  On hardware that dispatched out of order the wait could stall a partially resident grid. */
#define DUSTIN_WS_HEADER_BYTES 4096

/* Scratch (bytes of device memory, 256-byte aligned by the caller) that is enough for every entry point on this
 * shape: the scoring stage with the head subset `head_mask` (0 => sized for all n_q_heads heads) plus the
 * attention stage over at most `k_max` selected rows per list (k_max <= 0 => max_ctx rows, the dense case).
 * One buffer of this size serves dustin_verify_layer_fused.  Returns 0 on invalid arguments. */
size_t dustin_workspace_bytes(const dustin_shape_t* shape, uint64_t head_mask, int32_t k_max);

/* a1 -- head-subset scoring (PAPER.md:159 "target attention tensor of the last generated token", :218, :391).
 * For every head h with bit h of head_mask set:  p_h[n] = softmax_n( sm_scale * q[b,h,:] . K[b,n,g(h),:] ) over
 * the N_b cached tokens (reading A4).  n_lists == 1:  scores_now[b,0,n] = sum_h p_h[n];  n_lists == Hkv:
 * scores_now[b,g,n] = sum over the subset heads of KV group g, and a group with no subset head receives the sum
 * over all subset heads (reading A2).  Entries n >= N_b are written as 0.
 *   q: device bf16, row (b,h) at q + b*q_stride_batch + h*q_stride_head (elements): any verify position of the
 *      [B,T,Hq,d] query tensor can be scored (reading A3: position 0).
 *   scores_now: device fp32 [B, n_lists, max_ctx], written. */
int dustin_score_heads(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, int64_t q_stride_batch,
                       int64_t q_stride_head, uint64_t head_mask, int32_t n_lists, float* scores_now, void* ws,
                       size_t ws_bytes, void* stream);

/* a2 -- Eq. 5 accumulation (reading A6):  hist[b,l,n] <- alpha*hist[b,l,n] + scores_now[b,l,n]
 * for n < N_b (entries n >= N_b untouched).  Both device fp32 [batch, n_lists, max_ctx]. */
int dustin_fuse_scores(int32_t batch, int32_t n_lists, int32_t max_ctx, const int32_t* seq_lens,
                       const float* scores_now, float* hist_inout, float alpha, void* stream);

/* a3 -- tiered top-k, Eq. 6.  Per (b, list), N = N_b, k = k_b:
 *   k >= N: idx = 0..N-1, cnt = N.  Otherwise I_prot = [0,S') U [N-W',N) with S' = min(S,N), W' = min(W,N-S');
 *   I_draft = the m' = min(m, k-|I_prot|) best candidates of [S',N-W') by s_draft; I_target = the
 *   k-|I_prot|-m' best remaining candidates by s_target; ties -> lower index; scores compare as max(s, 0)
 *   (NaN undefined).  idx_out[b,l,:cnt] = I_verify in ascending order, tail = -1;  cnt_out[b,l] = |I_verify|.
 *   s_draft: device fp32; row (b,l) at s_draft + b*(draft_list_stride ? n_lists*max_ctx : max_ctx)
 *            + l*draft_list_stride  (draft_list_stride = 0: one [B,N] vector broadcast over the lists; = max_ctx:
 *            a [B,G,N] tensor).
 *   s_target: device fp32 [B, G, max_ctx].   idx_out: device int32 [B, G, k_max].   cnt_out: device int32 [B, G]. */
int dustin_topk_select(int32_t batch, int32_t max_ctx, const int32_t* seq_lens, const dustin_select_t* select,
                       const float* s_draft, int64_t draft_list_stride, const float* s_target, int32_t* idx_out,
                       int32_t* cnt_out, int32_t k_max, void* stream);

/* a4 / a5 -- verification attention (App. G :568; reading A13).  For every (b, h, t):
 * one softmax over the cnt[b,l] cache rows idx[b,l,:] (l = 0 if n_lists == 1 else g(h)) and the new rows u <= t
 * (causal among the T new tokens, self included), scale sm_scale;  out = sum p * V.
 * idx == NULL: all N_b cached rows (full-cache verification attention, the dense baseline).
 *   q: device bf16 [B,T,Hq,d];  k_new, v_new: device bf16 [B,T,Hkv,d];  idx: device int32 [B,n_lists,k_max]
 *   (entries in [0,N_b), any order);  cnt: device int32 [B,n_lists], or NULL = every list holds exactly k_max entries
 *   (needs k_max <= max_ctx and kv->seq_lens == NULL; the kernel then plans its work without reading a length from
 *   memory, which shortens its start);  out: device bf16 [B,T,Hq,d];
 *   lse_out: device fp32 [B,Hq,T] natural-log normaliser, or NULL. */
int dustin_sparse_verify_attn(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, const void* k_new,
                              const void* v_new, const int32_t* idx, const int32_t* cnt, int32_t n_lists,
                              int32_t k_max, void* out, float* lse_out, void* ws, size_t ws_bytes, void* stream);

/* a6 -- one layer, one call: a1 (query = verify position 0 of q) -> a2 (into hist_inout) -> a3 -> a4, enqueued
 * back to back on `stream` with no host synchronisation.  scores_now_out may be NULL (the per-call scores are
 * then never written to memory).  Other arguments as in the stage calls. */
int dustin_verify_layer_fused(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, const void* k_new,
                              const void* v_new, uint64_t head_mask, const float* s_draft,
                              int64_t draft_list_stride, float* hist_inout, float alpha,
                              const dustin_select_t* select, int32_t k_max, float* scores_now_out, void* out,
                              float* lse_out, int32_t* idx_out, int32_t* cnt_out, void* ws, size_t ws_bytes,
                              void* stream);

/* Cost hint for short contexts.  The one-shot call pays for a1 and a3 before it saves anything in a4, so below some
 * context length the dense call (dustin_sparse_verify_attn with idx == NULL) is faster: at k = 2048, B = 16 on the
 * Qwen2.5-72B-shaped layer the two cost the same near 10-12 k tokens, with the paper's 6.25 % budgets near 4 k
 * (profiles/r03_sweep.json, `crossover`).  The library never switches paths on its own (the caller owns the index lists
 * and the history); this helper returns 1 when dense is predicted to be at least as fast, 0 when the sparse layer is,
 * or a negative dustin_status, and optionally writes the two predicted times in microseconds.  The prediction is a
 * linear byte model fitted to B200 measurements of full-length sequences (shape->max_ctx tokens each) -- a hint, good
 * to roughly 10 % around the crossover on that machine, not a guarantee.  Host arithmetic only; no GPU is touched. */
int dustin_prefer_dense(const dustin_shape_t* shape, uint64_t head_mask, int32_t k, double* fused_us_out,
                        double* dense_us_out);

/* ---- steps either side of the layer path ---------------------------------------------------- */

/* Attention Recovery Rate, Eq. 1: the share of the attention mass of row (b,l) that the index list
 * keeps,  arr[b,l] = sum_{j in idx[b,l,:cnt[b,l]]} a[b,l,j] / sum_{j < N_b} a[b,l,j]   (0 for a row without mass).
 * `a` is any non-negative weight row (it is normalised here, as Eq. 1 requires sum_V A = 1); the listed indices
 * must be distinct (a set; dustin_topk_select's output is).  The windowed ARR of Eq. 2 and the SD-oracle bound of
 * Eq. 3-4 follow by composition: pass the window sum of A (dustin_fuse_scores with alpha = 1) and, for Eq. 4, the
 * list dustin_topk_select returns for it with m = 0, S = W = 0.
 *   a: device fp32 [B, n_lists, max_ctx];  idx: device int32 [B, n_lists, k_max];  cnt: device int32 [B, n_lists];
 *   arr_out: device fp32 [B, n_lists], written. */
int dustin_arr(int32_t batch, int32_t n_lists, int32_t max_ctx, const int32_t* seq_lens, const float* a,
               const int32_t* idx, const int32_t* cnt, int32_t k_max, float* arr_out, void* stream);

/* KV append after verification (accepted tokens are appended to the cache, rejected ones discarded).
 * The first n_append[b] rows (clipped to [0, T] and to the room left below max_ctx) of the verify block k_new /
 * v_new [B,T,Hkv,d] become cache rows N_b, N_b+1, ... of sequence b (kv->k / kv->v are WRITTEN; in a paged cache the
 * pages must already be mapped); seq_lens_inout[b] grows by that count.  kv->seq_lens is ignored (the lengths are
 * seq_lens_inout).  hist_inout (optional, device fp32 [B, n_lists, max_ctx]): the accumulated scores of the new
 * positions are set to 0 (Eq. 5 is a sum; nothing has been added for them yet).
 *   seq_lens_inout, n_append: device int32 [B]. */
int dustin_append_kv(const dustin_shape_t* shape, const dustin_kv_t* kv, int32_t* seq_lens_inout, const void* k_new,
                     const void* v_new, const int32_t* n_append, float* hist_inout, int32_t n_lists, void* stream);

/* Draft-side lookahead aggregation, Eq. 5 first line:
 *   s_draft[b,n] = sum_{h in head_mask} sum_{l < n_layers} sum_{gamma < T} softmax_n( sm_scale * q_l[b,gamma,h,:] . K_l[b,n,g(h),:] )
 * over the N_b cached tokens (reading A4), one vector per sequence.  `shape` describes the DRAFT model
 * (n_new = the number of lookahead queries per layer).  kv_layers: HOST array of n_layers cache descriptors (only k is
 * read);  q_layers: HOST array of n_layers device pointers, each bf16 [B, T, Hq, d].  One pass over each layer's K
 * cache with the T lookahead queries side by side when a KV group holds at most 8 (query, head) pairs and ws has
 * dustin_draft_workspace_bytes(shape, head_mask) bytes; otherwise one pass per (layer, lookahead token), for which
 * dustin_workspace_bytes(shape, head_mask, 1) bytes suffice.   s_draft: device fp32 [B, max_ctx], written (0 for
 * n >= N_b). */
size_t dustin_draft_workspace_bytes(const dustin_shape_t* shape, uint64_t head_mask);
int dustin_draft_aggregate(const dustin_shape_t* shape, const dustin_kv_t* kv_layers, const void* const* q_layers,
                           int32_t n_layers, uint64_t head_mask, float* s_draft, void* ws, size_t ws_bytes,
                           void* stream);

/* ---- alternative estimator: Quest with 16-token pages -----------------------------------
 * The estimator the paper measures its head-subset scoring against ("scores KV pages using inexpensive
 * min/max key statistics (avoiding exact QK^T)"; :297-299, Fig. 8 "Quest-16 denotes Quest with page size 16"; :401
 * "aggregates token-level Key statistics (e.g., minimum and maximum values) into page-level metadata ... reducing the
 * sequence length dimension for estimation from N to N/page size").  The paper names it without a formula; DESIGN.md
 * readings A20 / A21 fix one.  Logical page p of sequence b = the tokens [16p, 16p+16) below N_b, whatever the physical
 * layout of the cache.
 *
 * dustin_quest_build_pages: per (b, p, KV head g, channel c)  kmin = min_n K[b,n,g,c], kmax = max_n K[b,n,g,c] over the
 *   page's tokens (a page without a token: both 0).  page_meta: device bf16 [B, ceil(max_ctx/16), Hkv, 2, d] (kmin row,
 *   then kmax row; dustin_quest_meta_bytes bytes, 16-byte aligned), written.  first_token: device int32 [B] or NULL;
 *   when given, only the pages from first_token[b] / 16 on are rebuilt (after dustin_append_kv: pass the lengths from
 *   BEFORE the append, kv->seq_lens being the new ones); NULL rebuilds every page.  One pass over K (only kv->k is read).
 * dustin_quest_score_pages: for every subset head h (KV group g) and page p with a token
 *     U_h[p] = sm_scale * sum_c max(q[b,h,c] * kmin[b,p,g,c], q[b,h,c] * kmax[b,p,g,c])
 *   -- an upper bound of every exact logit sm_scale * q . K[b,n,g,:] of the page, from the metadata alone (A20) --
 *   then P_h = softmax over the pages that hold a token, and page_scores[b,l,p] = sum of P_h over the subset heads that
 *   feed list l, with the list rule of dustin_score_heads (A21); pages without a token score 0.  The result has the
 *   format of a1's scores with pages for tokens: dustin_topk_select with max_ctx = ceil(max_ctx/16) ranks pages.
 *   seq_lens: device int32 [B] or NULL (all max_ctx);  q, strides, head_mask, n_lists as in dustin_score_heads;
 *   page_scores: device fp32 [B, n_lists, ceil(max_ctx/16)], written;  ub_out: device fp32 [B, |subset|, ceil(max_ctx/16)]
 *   (subset heads in ascending order; U_h[p], 0 for pages without a token) or NULL;
 *   ws: dustin_workspace_bytes(shape, head_mask, 1) bytes are enough. */
#define DUSTIN_QUEST_PAGE 16
size_t dustin_quest_meta_bytes(const dustin_shape_t* shape);
int dustin_quest_build_pages(const dustin_shape_t* shape, const dustin_kv_t* kv, const int32_t* first_token,
                             void* page_meta, void* stream);
int dustin_quest_score_pages(const dustin_shape_t* shape, const int32_t* seq_lens, const void* page_meta, const void* q,
                             int64_t q_stride_batch, int64_t q_stride_head, uint64_t head_mask, int32_t n_lists,
                             float* page_scores, float* ub_out, void* ws, size_t ws_bytes, void* stream);

/* ---- a1 without a workspace argument --------------------------------------------------------------------------------
 * dustin_score_heads_static computes exactly what dustin_score_heads computes (same arguments, same kernels, same
 * bits in scores_now) but takes no `ws`: its scratch is a fixed array of DUSTIN_STATIC_SCRATCH_BYTES that is built into
 * the library.  The call allocates nothing -- no cudaMalloc / cudaFree, no memory pool, no allocating library routine.
 *
 * Who needs this.  Every other entry point asks the caller for a workspace, and some callers have no way to make one:
 *   - code running under a serving engine whose memory manager claimed (nearly) all of HBM at start-up, so that a
 *     cudaMalloc made behind the engine's back fails or eats into the KV-cache budget the engine thinks it owns;
 *   - an operator plugged into a host runtime whose operator signature carries inputs and outputs only, with no slot
 *     for a scratch buffer and no handle on the runtime's allocator;
 *   - a decode step that must not stall: cudaMalloc and cudaFree may synchronise the whole device, which a
 *     latency-bound loop cannot afford in the middle of a step.
 * Such a caller passes the inputs and the output as usual and nothing else.
 *
 * Limit.  The scratch the shape needs -- about 4 * batch * |head_mask| * max_ctx bytes of logits plus a few per cent of
 * softmax partials; dustin_workspace_bytes(shape, head_mask, 1) is a safe upper bound -- must not exceed
 * DUSTIN_STATIC_SCRATCH_BYTES (16 MiB: e.g. B = 4, 8 subset heads, 64k context).  A larger shape returns
 * DUSTIN_ERR_STATIC_SCRATCH before anything touches the device; use dustin_score_heads with your own workspace there.
 * The array costs its 16 MiB on every GPU on which the library's device code is loaded, from then until the process
 * exits, whether this entry point is ever called or not.
 *
 * First call on a device.  The first call made with a given device current does a one-time set-up for that device: it
 * makes the CUDA runtime load the library's device code there if it has not yet (that is when the array gets its memory)
 * and asks it for the array's device address (cudaGetSymbolAddress; a failure returns DUSTIN_ERR_CUDA).  Make that first
 * call during start-up, outside any stream capture; later calls on the same device only enqueue kernels.  The address is
 * kept for the life of the process: after cudaDeviceReset it is stale, do not call this entry point again then.
 *
 * Sharing.  There is ONE array per GPU and every call on that GPU uses it, whatever the stream or host thread: two calls
 * whose kernels may overlap on the GPU race on it and both get garbage -- keep them on one stream or order them with
 * events.  The array keeps what the last call wrote; no call depends on that (nothing in it needs to start at zero: each
 * call writes every word it later reads), so calls of different shapes may follow each other freely.
 * Arguments, layouts and the other error codes: see dustin_score_heads. */
#define DUSTIN_STATIC_SCRATCH_BYTES (16 * 1024 * 1024)
int dustin_score_heads_static(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q,
                              int64_t q_stride_batch, int64_t q_stride_head, uint64_t head_mask, int32_t n_lists,
                              float* scores_now, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DUSTIN_H_ */
