// api.cu -- the C ABI of include/dustin.h: host-side validation, workspace carving and stage launches.
// No device memory is allocated, freed, read or synchronised here; every call only enqueues on `stream`.
#include "kernels.cuh"

#include "../../include/dustin_debug.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>

namespace dustin {
namespace {

thread_local int g_last_cuda_error = 0;

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int fail_cuda(cudaError_t e) {
    g_last_cuda_error = (int)e;
    return DUSTIN_ERR_CUDA;
}

// ---- shape / cache validation ---------------------------------------------------------------------------------
int check_shape(const dustin_shape_t* s) {
    if (!s) return DUSTIN_ERR_INVALID_ARG;
    if (s->batch <= 0 || s->n_q_heads <= 0 || s->n_kv_heads <= 0 || s->head_dim <= 0 || s->n_new <= 0 ||
        s->max_ctx < 0 || !(s->sm_scale >= 0.f) || !std::isfinite(s->sm_scale))
        return DUSTIN_ERR_INVALID_ARG;
    if (s->n_q_heads % s->n_kv_heads != 0) return DUSTIN_ERR_INVALID_ARG;
    if (s->head_dim != 64 && s->head_dim != 128) return DUSTIN_ERR_UNSUPPORTED;
    if (s->n_q_heads > 64 || s->n_new > 16 || s->max_ctx > (1 << 20) || s->batch > 65535 || s->n_kv_heads > 65535)
        return DUSTIN_ERR_UNSUPPORTED;
    if (s->n_new * (s->n_q_heads / s->n_kv_heads) > 96) return DUSTIN_ERR_UNSUPPORTED;
    return DUSTIN_OK;
}

int check_kv(const dustin_shape_t* s, const dustin_kv_t* kv, bool need_v, KvView* out) {
    if (!kv || !kv->k || (need_v && !kv->v)) return DUSTIN_ERR_INVALID_ARG;
    if (kv->stride_seq < 0 || kv->stride_token <= 0 || kv->stride_head < 0) return DUSTIN_ERR_INVALID_ARG;
    // 16-byte row alignment (dustin.h): 8 bf16 elements
    if ((kv->stride_seq | kv->stride_token | kv->stride_head) & 7) return DUSTIN_ERR_INVALID_ARG;
    if (((uintptr_t)kv->k & 15) || ((uintptr_t)kv->v & 15)) return DUSTIN_ERR_INVALID_ARG;
    if (kv->page_table) {
        if (kv->page_size <= 0 || kv->max_pages <= 0) return DUSTIN_ERR_INVALID_ARG;
        if ((long long)kv->page_size * kv->max_pages < s->max_ctx) return DUSTIN_ERR_INVALID_ARG;
    }
    out->k = static_cast<const __nv_bfloat16*>(kv->k);
    out->v = static_cast<const __nv_bfloat16*>(kv->v);
    out->stride_seq = kv->stride_seq;
    out->stride_token = kv->stride_token;
    out->stride_head = kv->stride_head;
    out->page_table = kv->page_table;
    out->page_size = kv->page_table ? kv->page_size : 1;
    out->page_shift = -1;
    if ((out->page_size & (out->page_size - 1)) == 0)
        for (int s2 = 0; s2 < 31; ++s2)
            if ((1 << s2) == out->page_size) out->page_shift = s2;
    out->max_pages = kv->page_table ? kv->max_pages : 0;
    out->seq_lens = kv->seq_lens;
    return DUSTIN_OK;
}

constexpr int kMinScoreChunk = 64;   // fewest tokens per scoring CTA (the workspace holds one softmax partial per CTA and head)

float scale_log2_of(const dustin_shape_t* s) {
    const float sc = s->sm_scale == 0.f ? (float)(1.0 / std::sqrt((double)s->head_dim)) : s->sm_scale;
    return sc * kLog2e;
}

// ---- scoring plan ---------------------------------------------------------------------------------------------
// Tokens per scoring CTA = CTAs per sequence (the 16-token tiles of a sequence are dealt round-robin to its CTAs, score.cu,
// so the chunk only sets the CTA count).  group_slots = how many scored KV groups the 8 warps of a CTA serve side by side;
// the 8 / group_slots warps that share a group take every (8 / group_slots)-th tile each.  n_parts = softmax partials per
// (sequence, head) = CTAs per sequence.
// The rule is "a fixed number of tiles per warp", whatever the grid then is -- measured in round 2 on every workload of
// bench.py (fused layer, us; tiles per warp 4 / 8 / 16 / 32 where it was tried):
//   8 scored groups (Qwen spread):  32k B=16  226.3 / 224.2 / 228.6 / 236.4;  16k  148.2 / 147.6 / 149.6 / 155.8;
//                                   8k  108.1 / 107.2 / 110.7 / 116.3;  4k  91.7 / 91.7 / 93.9 / 97.8;  32k B=4  - / 93.4 / 100.9 / 99.4
//   4 scored groups (Llama spread): 32k  156.5 / 154.9 / 158.0 / -;  16k  112.6 / 114.2 / 114.5 / -;  8k  89.6 / 90.0 / 95.2 / -
//   1 scored group (packed):        32k  95.2 / 95.7 / 88.8 (16 tiles) ;  128k B=4  97.1 / 96.3 / 92.3;  8k  77.2 / 75.6 / 76.9
//   paged ragged (4 groups):        380.4 / 344.6 / 338.0 / 344.2
// i.e. 8 tiles per warp, 16 when the CTA's warps share one or two groups or the cache is paged.  Round 1 used >= 256 tokens
// per CTA and cut grids of one to three waves down to exactly one wave: at 8 groups that is 16 tiles per warp or more --
// config 3 loses 4 us per layer to it, 16k 14 us, 32k at batch 4 13 us.
// The plan does not depend on which entry point asks: the staged and the one-shot call must cut a sequence into the same
// CTAs, or their softmax partials fold in different groupings and the two paths stop being bit-identical.  (A one-wave
// grid for the staged call alone -- a1 at B = 16: 4k 37 -> 30 us, 8k 56 -> 53 us -- was dropped for that reason.)
void score_plan(int batch, int n_groups, int max_ctx, bool paged, int* chunk_tokens, int* n_parts, int* group_slots) {
    (void)batch;
    int slots = 1;
    while (slots < n_groups && slots < 8) slots <<= 1;
    const int n_sub = 8 / slots;
    const int tiles_per_warp = (slots <= 2 || paged) ? 16 : 8;
    int chunk = 16 * n_sub * tiles_per_warp;
    const int forced = knob(DUSTIN_KNOB_SCORE_CHUNK);   // tuning aid: tokens per scoring CTA (multiple of 16)
    if (forced >= kMinScoreChunk) chunk = (forced + 15) / 16 * 16;
    *chunk_tokens = chunk;
    *group_slots = slots;
    *n_parts = max_ctx > 0 ? (max_ctx + chunk - 1) / chunk : 1;   // one partial per (CTA, head): the warps of a CTA that
                                                                  // share a KV group fold theirs before writing
}

struct ScoreWs {
    size_t logits, part, stats, total;
};
ScoreWs score_ws(int batch, int nsel, int max_ctx) {
    // upper bound of the partial count: one per CTA at the smallest chunk
    const size_t stride = ((size_t)max_ctx + 3) & ~(size_t)3;
    const size_t n_chunks = ((size_t)max_ctx + kMinScoreChunk - 1) / kMinScoreChunk + 1;   // score_plan never goes below it
    ScoreWs w;
    w.logits = 0;
    w.part = align256(w.logits + (size_t)batch * nsel * stride * sizeof(float));
    w.stats = align256(w.part + (size_t)batch * nsel * n_chunks * sizeof(float2));
    w.total = align256(w.stats + (size_t)batch * nsel * sizeof(float2));
    return w;
}

// Fills the head-subset tables of ScoreParams.  Ordinals follow ascending head index.
int build_subset(const dustin_shape_t* s, uint64_t head_mask, int n_lists, ScoreParams* p) {
    const int Hq = s->n_q_heads, Hkv = s->n_kv_heads, r = Hq / Hkv;
    if (Hq < 64 && (head_mask >> Hq) != 0) return DUSTIN_ERR_INVALID_ARG;
    if (head_mask == 0) return DUSTIN_ERR_INVALID_ARG;
    if (n_lists != 1 && n_lists != Hkv) return DUSTIN_ERR_INVALID_ARG;
    if (Hkv > 64) return DUSTIN_ERR_UNSUPPORTED;
    int nsel = 0, n_groups = 0;
    int first_of_group[64], cnt_of_group[64];
    for (int g = 0; g < Hkv; ++g) {
        first_of_group[g] = nsel;
        cnt_of_group[g] = 0;
        for (int j = 0; j < r; ++j) {
            const int h = g * r + j;
            if ((head_mask >> h) & 1ull) {
                p->sel_head[nsel++] = (unsigned char)h;
                cnt_of_group[g]++;
            }
        }
        if (cnt_of_group[g] > 8) return DUSTIN_ERR_UNSUPPORTED;
        if (cnt_of_group[g] > 0) {
            p->group_id[n_groups] = (unsigned char)g;
            p->group_first[n_groups] = (unsigned char)first_of_group[g];
            p->group_cnt[n_groups] = (unsigned char)cnt_of_group[g];
            ++n_groups;
        }
    }
    p->nsel = nsel;
    p->n_groups = n_groups;
    for (int l = 0; l < n_lists; ++l) {
        if (n_lists == 1 || cnt_of_group[l] == 0) {   // one global list, or an empty group (reading A2)
            p->list_first[l] = 0;
            p->list_cnt[l] = (unsigned char)nsel;
        } else {
            p->list_first[l] = (unsigned char)first_of_group[l];
            p->list_cnt[l] = (unsigned char)cnt_of_group[l];
        }
    }
    return DUSTIN_OK;
}

// Membership bitmasks I_prot U I_draft that the draft-tier selection kernel of the fused call hands to the target-tier
// kernel: one row of select_mask_words(max_ctx) words per (sequence, list); lives right after the scoring scratch.
size_t select_ws_bytes(const dustin_shape_t* s) {
    return align256((size_t)s->batch * s->n_kv_heads * select_mask_words(s->max_ctx) * sizeof(uint32_t));
}

int popcount64(uint64_t x) {
    int c = 0;
    for (; x; x &= x - 1) ++c;
    return c;
}

// ---- attention plan -------------------------------------------------------------------------------------------
struct AttnWs {
    size_t total;
    int split_tokens, n_splits;
    bool tc;
};
AttnWs attn_ws(const dustin_shape_t* s, int max_tokens) {
    // tcgen05 kernel (attn_tc.cu): arrival counters + stream-K partials.  mma.sync cluster kernel (attn.cu): the
    // split partials are combined through distributed shared memory, no global scratch.
    AttnWs w;
    attn_plan(s->batch, s->n_kv_heads, max_tokens, &w.split_tokens, &w.n_splits);
    const int rows = s->n_new * (s->n_q_heads / s->n_kv_heads);
    w.tc = attn_get_impl() != 1 && attn_tc_usable(s->batch, s->n_kv_heads, s->head_dim, rows, max_tokens, s->n_new);
    w.total = w.tc ? attn_tc_ws_bytes(s->batch, s->n_kv_heads, rows) : 0;
    return w;
}

// norm_out != nullptr: launch only the logits kernel and describe the pending normalisation + Eq. 5 accumulation for
// the selection kernel, which then does it row by row (SelectParams::Norm).
int run_score(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, int64_t q_stride_batch,
              int64_t q_stride_head, uint64_t head_mask, int32_t n_lists, float* scores_now, float* hist,
              float alpha, void* ws, size_t ws_bytes, cudaStream_t stream, SelectParams::Norm* norm_out = nullptr,
              int n_queries = 1, int64_t q_stride_query = 0, bool defer_wait = false) {
    // n_queries > 1 (draft-side aggregation, n_lists == 1): every subset head is scored for n_queries query rows
    // q_stride_query apart in ONE pass over K -- the (query, head) pairs are the "heads" of the kernel, <= 8 per KV group
    // and <= 64 in all (DUSTIN_ERR_UNSUPPORTED otherwise; the caller then scores one query row per pass).
    int rc = check_shape(shape);
    if (rc) return rc;
    ScoreParams p;
    std::memset(&p, 0, sizeof p);
    rc = check_kv(shape, kv, false, &p.kv);
    if (rc) return rc;
    if (!q || ((uintptr_t)q & 15) || ((q_stride_batch | q_stride_head) & 7) || q_stride_batch < 0 ||
        q_stride_head < 0)
        return DUSTIN_ERR_INVALID_ARG;
    if (!scores_now && !hist) return DUSTIN_ERR_INVALID_ARG;
    rc = build_subset(shape, head_mask, n_lists, &p);
    if (rc) return rc;
    for (int i = 0; i < p.nsel; ++i) p.sel_qoff[i] = (int)(p.sel_head[i] * q_stride_head);
    if (n_queries > 1) {
        if (n_lists != 1 || p.nsel * n_queries > 64 || q_stride_query < 0 || (q_stride_query & 7))
            return DUSTIN_ERR_UNSUPPORTED;
        ScoreParams v = p;
        int ord = 0;
        for (int gi = 0; gi < p.n_groups; ++gi) {
            if (p.group_cnt[gi] * n_queries > 8) return DUSTIN_ERR_UNSUPPORTED;
            v.group_first[gi] = (unsigned char)ord;
            v.group_cnt[gi] = (unsigned char)(p.group_cnt[gi] * n_queries);
            for (int qi = 0; qi < n_queries; ++qi)
                for (int j = 0; j < p.group_cnt[gi]; ++j) {
                    const int base = p.group_first[gi] + j;
                    v.sel_head[ord] = p.sel_head[base];
                    v.sel_qoff[ord] = (int)(qi * q_stride_query) + p.sel_qoff[base];
                    ++ord;
                }
        }
        v.nsel = ord;
        v.list_first[0] = 0;
        v.list_cnt[0] = (unsigned char)ord;
        p = v;
    }
    const ScoreWs w = score_ws(shape->batch, p.nsel, shape->max_ctx);
    if (!ws || ws_bytes < kWsHeader + w.total || ((uintptr_t)ws & 255)) return DUSTIN_ERR_WORKSPACE;
    p.q = static_cast<const __nv_bfloat16*>(q);
    p.q_stride_batch = q_stride_batch;
    p.q_stride_head = q_stride_head;
    p.batch = shape->batch;
    p.head_dim = shape->head_dim;
    p.max_ctx = shape->max_ctx;
    p.n_lists = n_lists;
    p.scale_log2 = scale_log2_of(shape);
    p.defer_wait = defer_wait ? 1 : 0;
    score_plan(p.batch, p.n_groups, p.max_ctx, p.kv.page_table != nullptr, &p.chunk_tokens, &p.n_chunks, &p.group_slots);
    p.logit_stride = ((long long)p.max_ctx + 3) & ~3ll;
    char* base = static_cast<char*>(ws) + kWsHeader;   // the persistent header belongs to the attention stage
    p.logits = reinterpret_cast<float*>(base + w.logits);
    p.part = reinterpret_cast<float2*>(base + w.part);
    p.stats = reinterpret_cast<float2*>(base + w.stats);
    if (p.max_ctx == 0) return DUSTIN_OK;
    if (norm_out) {
        norm_out->logits = p.logits;
        norm_out->part = p.part;
        norm_out->logit_stride = p.logit_stride;
        norm_out->nsel = p.nsel;
        norm_out->n_chunks = p.n_chunks;
        norm_out->alpha = alpha;
        // one reader per logits row: one list per sequence, or every KV group has a subset head of its own (no empty group
        // that would read all rows, reading A2); rows made of whole 128-byte lines
        norm_out->discard_logits = (n_lists == 1 || p.n_groups == shape->n_kv_heads) && (p.logit_stride & 31) == 0 &&
                                   knob(DUSTIN_KNOB_L2_HYGIENE) != 0;
        std::memcpy(norm_out->list_first, p.list_first, sizeof p.list_first);
        std::memcpy(norm_out->list_cnt, p.list_cnt, sizeof p.list_cnt);
    }
    const cudaError_t e = launch_score(p, scores_now, hist, alpha, norm_out != nullptr, stream);
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

// DUSTIN_KNOB_FUSED_ROWS = 0 keeps the separate stats / normalise kernels in the fused entry point (A/B measurements).
bool fused_rows_disabled() { return knob(DUSTIN_KNOB_FUSED_ROWS) == 0; }

int check_select(const dustin_select_t* sel, int32_t k_max) {
    if (!sel) return DUSTIN_ERR_INVALID_ARG;
    if (sel->n_sink < 0 || sel->n_recent < 0 || sel->m_num < 0 || sel->m_den <= 0 || sel->m_num > sel->m_den ||
        sel->n_lists <= 0 || k_max <= 0)
        return DUSTIN_ERR_INVALID_ARG;
    if (!sel->budgets) {
        if (sel->budget < 0 || sel->budget > k_max) return DUSTIN_ERR_INVALID_ARG;
        if (sel->n_sink + sel->n_recent > sel->budget) return DUSTIN_ERR_INVALID_ARG;   // reading A12
    }
    return DUSTIN_OK;
}

int run_select(int32_t batch, int32_t max_ctx, const int32_t* seq_lens, const dustin_select_t* sel,
               const float* s_draft, int64_t draft_list_stride, const float* s_target, int32_t* idx_out,
               int32_t* cnt_out, int32_t k_max, cudaStream_t stream, const SelectParams::Norm* norm = nullptr,
               int mode = 0, uint32_t* draft_mask = nullptr, int draft_rows_per_cta = 1) {
    int rc = check_select(sel, k_max);
    if (rc) return rc;
    if (batch <= 0 || max_ctx < 0 || !s_draft || !s_target || !idx_out || !cnt_out) return DUSTIN_ERR_INVALID_ARG;
    if (mode != 0 && !draft_mask) return DUSTIN_ERR_INVALID_ARG;
    if (draft_list_stride != 0 && draft_list_stride != max_ctx) return DUSTIN_ERR_INVALID_ARG;
    if (max_ctx > (1 << 20) || batch > 65535) return DUSTIN_ERR_UNSUPPORTED;
    SelectParams p;
    p.batch = batch;
    p.max_ctx = max_ctx;
    p.n_lists = sel->n_lists;
    p.k_max = k_max;
    p.seq_lens = seq_lens;
    p.budget = sel->budget;
    p.budgets = sel->budgets;
    p.n_sink = sel->n_sink;
    p.n_recent = sel->n_recent;
    p.m_num = sel->m_num;
    p.m_den = sel->m_den;
    p.s_draft = s_draft;
    p.draft_list_stride = draft_list_stride;
    p.draft_batch_stride = draft_list_stride == 0 ? (long long)max_ctx : (long long)sel->n_lists * max_ctx;
    p.s_target = s_target;
    p.idx_out = idx_out;
    p.cnt_out = cnt_out;
    std::memset(&p.norm, 0, sizeof p.norm);
    if (norm) p.norm = *norm;
    p.draft_mask = draft_mask;
    p.draft_mask_stride = (long long)select_mask_words(max_ctx);
    p.draft_rows_per_cta = draft_rows_per_cta;
    p.trace = nullptr;
    if (mode == 2 && norm) {   // few long rows: one thread-block cluster per row (select_cluster.cu)
        const int C = select_cluster_size(p);
        if (C > 0) {
            const cudaError_t e = launch_select_cluster(p, C, stream);
            return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
        }
    }
    const cudaError_t e = launch_select(p, stream, mode);
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int run_attn(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, const void* k_new,
             const void* v_new, const int32_t* idx, const int32_t* cnt, int32_t n_lists, int32_t k_max, void* out,
             float* lse_out, void* ws, size_t ws_bytes, cudaStream_t stream, int uniform_cnt = -1) {
    int rc = check_shape(shape);
    if (rc) return rc;
    AttnParams p;
    std::memset(&p, 0, sizeof p);
    rc = check_kv(shape, kv, true, &p.kv);
    if (rc) return rc;
    if (!q || !k_new || !v_new || !out) return DUSTIN_ERR_INVALID_ARG;
    if (((uintptr_t)q | (uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)out) & 15) return DUSTIN_ERR_INVALID_ARG;
    if (idx) {
        if (k_max <= 0 || (n_lists != 1 && n_lists != shape->n_kv_heads)) return DUSTIN_ERR_INVALID_ARG;
        if (!cnt) {   // cnt == NULL: every list holds exactly k_max entries (dustin.h)
            if (k_max > shape->max_ctx || kv->seq_lens) return DUSTIN_ERR_INVALID_ARG;
            uniform_cnt = k_max;
        }
    } else {
        n_lists = 1;
        k_max = 0;
        uniform_cnt = kv->seq_lens ? -1 : shape->max_ctx;   // dense baseline over full-length sequences
    }
    const int max_tokens = idx ? (k_max < shape->max_ctx ? k_max : shape->max_ctx) : shape->max_ctx;
    const AttnWs w = attn_ws(shape, max_tokens > 0 ? max_tokens : 1);
    if (w.total > 0 && (!ws || ws_bytes < w.total || ((uintptr_t)ws & 255))) return DUSTIN_ERR_WORKSPACE;
    p.q = static_cast<const __nv_bfloat16*>(q);
    p.k_new = static_cast<const __nv_bfloat16*>(k_new);
    p.v_new = static_cast<const __nv_bfloat16*>(v_new);
    p.idx = idx;
    p.cnt = cnt;
    p.uniform_cnt = uniform_cnt;
    p.batch = shape->batch;
    p.n_q_heads = shape->n_q_heads;
    p.n_kv_heads = shape->n_kv_heads;
    p.group = shape->n_q_heads / shape->n_kv_heads;
    p.head_dim = shape->head_dim;
    p.n_new = shape->n_new;
    p.max_ctx = shape->max_ctx;
    p.n_lists = n_lists;
    p.k_max = k_max;
    p.scale_log2 = scale_log2_of(shape);
    p.rows = p.n_new * p.group;
    p.split_tokens = w.split_tokens;
    p.n_splits = w.n_splits;
    p.tc_ws = w.tc ? ws : nullptr;
    p.out = static_cast<__nv_bfloat16*>(out);
    p.lse_out = lse_out;
    const cudaError_t e = launch_attn(p, stream);
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

}  // namespace
}  // namespace dustin

using namespace dustin;

extern "C" {

int dustin_version(void) { return DUSTIN_VERSION; }

const char* dustin_status_string(int status) {
    switch (status) {
        case DUSTIN_OK: return "ok";
        case DUSTIN_ERR_INVALID_ARG: return "invalid argument";
        case DUSTIN_ERR_UNSUPPORTED: return "unsupported shape (see the limits in dustin.h)";
        case DUSTIN_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case DUSTIN_ERR_CUDA: return "CUDA launch error (see dustin_last_cuda_error)";
        case DUSTIN_ERR_STATIC_SCRATCH:
            return "shape needs more scratch than DUSTIN_STATIC_SCRATCH_BYTES: use dustin_score_heads with your own workspace";
        default: return "unknown status";
    }
}

int dustin_last_cuda_error(void) { return g_last_cuda_error; }

void dustin_tune_attn_split_tokens(int32_t split_tokens) { attn_set_split_override(split_tokens); }

void dustin_tune_attn_impl(int32_t impl) { attn_set_impl(impl); }

void dustin_tune_set(int32_t knob_id, int32_t value) { knob_set(knob_id, value); }

int32_t dustin_tune_get(int32_t knob_id) { return knob(knob_id); }

void dustin_debug_trace_buffer(void* device_ptr, size_t bytes) { trace_buffer_set(device_ptr, bytes); }

uint64_t dustin_launch_count(void) { return prof_launch_count(); }

void dustin_profile_enable(int32_t on) { prof_enable(on != 0); }

int dustin_profile_collect(double* ms_out, int64_t* launches_out) {
    if (!ms_out || !launches_out) return DUSTIN_ERR_INVALID_ARG;
    long long n[kKernCount];
    const cudaError_t e = prof_collect(ms_out, n);
    for (int i = 0; i < kKernCount; ++i) launches_out[i] = n[i];
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

const char* dustin_kernel_name(int32_t kernel_id) { return prof_kernel_name(kernel_id); }

size_t dustin_workspace_bytes(const dustin_shape_t* shape, uint64_t head_mask, int32_t k_max) {
    if (check_shape(shape) != DUSTIN_OK) return 0;
    const int nsel = head_mask ? popcount64(head_mask) : shape->n_q_heads;
    const ScoreWs sw = score_ws(shape->batch, nsel, shape->max_ctx);
    int max_tokens = (k_max > 0 && k_max < shape->max_ctx) ? k_max : shape->max_ctx;
    if (max_tokens < 1) max_tokens = 1;
    const AttnWs aw = attn_ws(shape, max_tokens);
    return kWsHeader + sw.total + select_ws_bytes(shape) + aw.total + 256;
}

int dustin_score_heads(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, int64_t q_stride_batch,
                       int64_t q_stride_head, uint64_t head_mask, int32_t n_lists, float* scores_now, void* ws,
                       size_t ws_bytes, void* stream) {
    if (!scores_now) return DUSTIN_ERR_INVALID_ARG;
    return run_score(shape, kv, q, q_stride_batch, q_stride_head, head_mask, n_lists, scores_now, nullptr, 0.f, ws,
                     ws_bytes, static_cast<cudaStream_t>(stream));
}

int dustin_fuse_scores(int32_t batch, int32_t n_lists, int32_t max_ctx, const int32_t* seq_lens,
                       const float* scores_now, float* hist_inout, float alpha, void* stream) {
    if (batch <= 0 || n_lists <= 0 || max_ctx < 0 || !scores_now || !hist_inout || !std::isfinite(alpha))
        return DUSTIN_ERR_INVALID_ARG;
    if (batch > 65535 || n_lists > 65535) return DUSTIN_ERR_UNSUPPORTED;
    if (max_ctx == 0) return DUSTIN_OK;
    const cudaError_t e = launch_fuse(batch, n_lists, max_ctx, seq_lens, scores_now, hist_inout, alpha,
                                     static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_topk_select(int32_t batch, int32_t max_ctx, const int32_t* seq_lens, const dustin_select_t* select,
                       const float* s_draft, int64_t draft_list_stride, const float* s_target, int32_t* idx_out,
                       int32_t* cnt_out, int32_t k_max, void* stream) {
    return run_select(batch, max_ctx, seq_lens, select, s_draft, draft_list_stride, s_target, idx_out, cnt_out,
                      k_max, static_cast<cudaStream_t>(stream));
}

int dustin_sparse_verify_attn(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, const void* k_new,
                              const void* v_new, const int32_t* idx, const int32_t* cnt, int32_t n_lists,
                              int32_t k_max, void* out, float* lse_out, void* ws, size_t ws_bytes, void* stream) {
    return run_attn(shape, kv, q, k_new, v_new, idx, cnt, n_lists, k_max, out, lse_out, ws, ws_bytes,
                    static_cast<cudaStream_t>(stream));
}

int dustin_verify_layer_fused(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, const void* k_new,
                              const void* v_new, uint64_t head_mask, const float* s_draft,
                              int64_t draft_list_stride, float* hist_inout, float alpha,
                              const dustin_select_t* select, int32_t k_max, float* scores_now_out, void* out,
                              float* lse_out, int32_t* idx_out, int32_t* cnt_out, void* ws, size_t ws_bytes,
                              void* stream) {
    // Validate everything before the first launch so that an argument error enqueues nothing (hist_inout, the only
    // in/out state, is then untouched): the union of the checks of run_score, run_select and run_attn.
    int rc = check_shape(shape);
    if (rc) return rc;
    rc = check_select(select, k_max);
    if (rc) return rc;
    if (!hist_inout || !s_draft || !idx_out || !cnt_out || !out || !q || !k_new || !v_new || !kv || !kv->v ||
        !std::isfinite(alpha))
        return DUSTIN_ERR_INVALID_ARG;
    {
        KvView view;
        rc = check_kv(shape, kv, true, &view);   // strides, 16-byte alignment of k and v, page-table geometry
        if (rc) return rc;
        if (((uintptr_t)q | (uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)out) & 15) return DUSTIN_ERR_INVALID_ARG;
        ScoreParams probe;
        std::memset(&probe, 0, sizeof probe);
        rc = build_subset(shape, head_mask, select->n_lists, &probe);   // mask inside Hq, <= 8 heads per KV group, n_lists
        if (rc) return rc;
    }
    if (select->n_lists != 1 && select->n_lists != shape->n_kv_heads) return DUSTIN_ERR_INVALID_ARG;
    if (draft_list_stride != 0 && draft_list_stride != shape->max_ctx) return DUSTIN_ERR_INVALID_ARG;
    const int nsel = popcount64(head_mask);
    if (nsel == 0) return DUSTIN_ERR_INVALID_ARG;
    const ScoreWs sw = score_ws(shape->batch, nsel, shape->max_ctx);
    const int max_tokens = k_max < shape->max_ctx ? k_max : shape->max_ctx;
    const AttnWs aw = attn_ws(shape, max_tokens > 0 ? max_tokens : 1);
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < kWsHeader + sw.total + select_ws_bytes(shape) + aw.total)
        return DUSTIN_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char* base = static_cast<char*>(ws);
    // a3, draft tier (Eq. 6: I_draft = TopK(S_Draft \ I_prot, m)) needs nothing that a1 produces: its kernel is launched
    // FIRST, releases the scoring kernel at once and works beside it; the bitmask I_prot U I_draft waits in the workspace.
    uint32_t* draft_mask = reinterpret_cast<uint32_t*>(base + kWsHeader + sw.total);
    const bool hoist = knob(DUSTIN_KNOB_DRAFT_HOIST) != 0 && pdl_enabled() && shape->max_ctx > 0;
    if (hoist) {
        // Rows per draft-tier CTA (select.cu: fewer CTAs let the scoring kernel start earlier).  The draft tier must stay
        // well inside the K stream it hides under: a row of N tokens takes it about 13 us + 0.6 ns per token there, the
        // stream groups * B * N * 256 B at ~6.4 TB/s; rows per CTA = three quarters of that ratio, at most 4 (measured, fused
        // layer, us, 1 / 2 / 3 / 4 / 6 rows: 32k B=16  224.3 / 224.0 / 222.7 / 222.5 / 251.0;  16k  147.7 / 146.3 / 146.0 /
        // 154.9 / 179;  8k  107.4 / 107.5 / 117.8 / 128 / 149;  64k B=8  226.3 / 226.5 / 247 / 279 / 339).  Ragged batches
        // keep one row per CTA: the lengths are device data, and a stream shorter than estimated would expose the tier.
        int rpc = 1;
        if (!kv->seq_lens) {
            int n_groups = 0;
            const int r = shape->n_q_heads / shape->n_kv_heads;
            for (int g = 0; g < shape->n_kv_heads; ++g) {
                const uint64_t gm = (r >= 64 ? ~0ull : ((1ull << r) - 1ull)) << (g * r);
                if (head_mask & gm) ++n_groups;
            }
            const double t_row = 13.0 + 0.6e-3 * shape->max_ctx;
            const double t_a1 = (double)n_groups * shape->batch * shape->max_ctx * shape->head_dim * 2.0 / 6.4e6;
            rpc = (int)(0.75 * t_a1 / t_row);
            rpc = rpc < 1 ? 1 : (rpc > 4 ? 4 : rpc);
        }
        rc = run_select(shape->batch, shape->max_ctx, kv->seq_lens, select, s_draft, draft_list_stride, hist_inout,
                        idx_out, cnt_out, k_max, st, nullptr, 1, draft_mask, rpc);
        if (rc) return rc;
    }
    // a1 + a2: scores of verify position 0 (reading A3), accumulated straight into hist (Eq. 5)
    // With enough rows to fill the GPU the selection kernel normalises and accumulates its own rows (no separate
    // stats / normalise launches, no extra pass over the scores); it needs 16-byte rows and no scores_now output.
    SelectParams::Norm norm;
    bool rows_in_select = !scores_now_out && (shape->max_ctx & 3) == 0 && shape->max_ctx > 0 &&
                          (((uintptr_t)hist_inout | (uintptr_t)s_draft) & 15) == 0 && !fused_rows_disabled();
    if (rows_in_select && (long long)shape->batch * select->n_lists < 64) {
        // few rows: worth it only when a thread-block cluster shares each row (one CTA per row would push the logits of
        // every head of the list through a single SM)
        SelectParams probe;
        std::memset(&probe, 0, sizeof probe);
        probe.batch = shape->batch;
        probe.n_lists = select->n_lists;
        probe.max_ctx = shape->max_ctx;
        probe.s_target = hist_inout;
        probe.draft_mask = draft_mask;
        probe.norm.logits = reinterpret_cast<const float*>(base);   // non-null marker: the rows will be materialised
        rows_in_select = hoist && select_cluster_size(probe) > 0;
    }
    rc = run_score(shape, kv, q, (int64_t)shape->n_new * shape->n_q_heads * shape->head_dim, shape->head_dim,
                   head_mask, select->n_lists, scores_now_out, hist_inout, alpha, ws, ws_bytes, st,
                   rows_in_select ? &norm : nullptr, 1, 0, hoist);
    if (rc) return rc;
    // a3, target tier + list (or both tiers when the draft tier was not hoisted)
    rc = run_select(shape->batch, shape->max_ctx, kv->seq_lens, select, s_draft, draft_list_stride, hist_inout,
                    idx_out, cnt_out, k_max, st, rows_in_select ? &norm : nullptr, hoist ? 2 : 0, draft_mask);
    if (rc) return rc;
    // a4.  One budget for all sequences and no ragged lengths: every list will hold min(k, N) entries (Eq. 6 with the
    // clipping of reading A12), which the attention kernel then need not read back to plan its work.
    const int uniform_cnt = (!select->budgets && !kv->seq_lens)
                                ? (select->budget < shape->max_ctx ? select->budget : shape->max_ctx) : -1;
    return run_attn(shape, kv, q, k_new, v_new, idx_out, cnt_out, select->n_lists, k_max, out, lse_out,
                    ws, ws_bytes, st, uniform_cnt);
}

int dustin_probe_gather(const dustin_shape_t* shape, const dustin_kv_t* kv, const int32_t* idx, const int32_t* cnt,
                        int32_t n_lists, int32_t k_max, void* ws, size_t ws_bytes, void* stream) {
    int rc = check_shape(shape);
    if (rc) return rc;
    KvView view;
    rc = check_kv(shape, kv, true, &view);
    if (rc) return rc;
    if (!idx || !cnt || k_max <= 0 || (n_lists != 1 && n_lists != shape->n_kv_heads)) return DUSTIN_ERR_INVALID_ARG;
    if (!ws || ws_bytes < kWsHeader + 4 * (size_t)shape->batch * shape->n_kv_heads) return DUSTIN_ERR_WORKSPACE;
    const cudaError_t e = launch_gather_probe(view, idx, cnt, shape->batch, shape->n_kv_heads, shape->head_dim, n_lists,
                                              k_max, static_cast<char*>(ws) + kWsHeader, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_debug_occupy(int32_t n_ctas, int32_t threads, int32_t smem_bytes, int32_t microseconds, void* stream) {
    if (n_ctas <= 0 || threads <= 0 || threads > 1024 || smem_bytes < 0 || smem_bytes > 227 * 1024 || microseconds < 0)
        return DUSTIN_ERR_INVALID_ARG;
    const cudaError_t e = launch_occupy(n_ctas, threads, smem_bytes, microseconds, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_debug_block_scan(int32_t threads, int32_t n_blocks, const uint32_t* in, uint32_t* out, uint32_t* total,
                            void* stream) {
    if ((threads != 256 && threads != 512 && threads != 1024) || n_blocks <= 0 || !in || !out || !total)
        return DUSTIN_ERR_INVALID_ARG;
    const cudaError_t e = launch_scan_test(threads, n_blocks, in, out, total, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_arr(int32_t batch, int32_t n_lists, int32_t max_ctx, const int32_t* seq_lens, const float* a,
               const int32_t* idx, const int32_t* cnt, int32_t k_max, float* arr_out, void* stream) {
    if (batch <= 0 || n_lists <= 0 || max_ctx < 0 || k_max <= 0 || !a || !idx || !cnt || !arr_out)
        return DUSTIN_ERR_INVALID_ARG;
    if (batch > 65535) return DUSTIN_ERR_UNSUPPORTED;
    const cudaError_t e = launch_arr(batch, n_lists, max_ctx, seq_lens, a, idx, cnt, k_max, arr_out,
                                     static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_append_kv(const dustin_shape_t* shape, const dustin_kv_t* kv, int32_t* seq_lens_inout, const void* k_new,
                     const void* v_new, const int32_t* n_append, float* hist_inout, int32_t n_lists, void* stream) {
    int rc = check_shape(shape);
    if (rc) return rc;
    KvView view;
    rc = check_kv(shape, kv, true, &view);
    if (rc) return rc;
    if (!seq_lens_inout || !k_new || !v_new || !n_append || (hist_inout && n_lists <= 0)) return DUSTIN_ERR_INVALID_ARG;
    if (((uintptr_t)k_new | (uintptr_t)v_new) & 15) return DUSTIN_ERR_INVALID_ARG;
    view.seq_lens = seq_lens_inout;
    const cudaError_t e = launch_append(view, seq_lens_inout, n_append, static_cast<const __nv_bfloat16*>(k_new),
                                        static_cast<const __nv_bfloat16*>(v_new), shape->batch, shape->n_new,
                                        shape->n_kv_heads, shape->head_dim, shape->max_ctx, hist_inout, n_lists,
                                        static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_draft_aggregate(const dustin_shape_t* shape, const dustin_kv_t* kv_layers, const void* const* q_layers,
                           int32_t n_layers, uint64_t head_mask, float* s_draft, void* ws, size_t ws_bytes,
                           void* stream) {
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!kv_layers || !q_layers || n_layers <= 0 || !s_draft) return DUSTIN_ERR_INVALID_ARG;
    for (int l = 0; l < n_layers; ++l)
        if (!q_layers[l]) return DUSTIN_ERR_INVALID_ARG;
    const int64_t q_stride_batch = (int64_t)shape->n_new * shape->n_q_heads * shape->head_dim;
    const int64_t q_stride_query = (int64_t)shape->n_q_heads * shape->head_dim;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    bool first = true;   // the first term overwrites s_draft (and writes the zeros beyond N_b), the others accumulate
    for (int l = 0; l < n_layers; ++l) {
        // One pass over the layer's K cache with all T lookahead queries side by side (the (query, head) pairs ride the
        // N axis of the MMA) when they fit -- <= 8 pairs per KV group -- and the workspace holds their logits ...
        rc = run_score(shape, &kv_layers[l], q_layers[l], q_stride_batch, shape->head_dim, head_mask, 1,
                       first ? s_draft : nullptr, first ? nullptr : s_draft, 1.0f, ws, ws_bytes, st, nullptr,
                       shape->n_new, q_stride_query);
        if (rc == DUSTIN_OK) {
            first = false;
            continue;
        }
        if (rc != DUSTIN_ERR_UNSUPPORTED && rc != DUSTIN_ERR_WORKSPACE) return rc;
        // ... otherwise one pass per lookahead token (Eq. 5 is a plain sum).
        for (int gam = 0; gam < shape->n_new; ++gam) {
            const __nv_bfloat16* q = static_cast<const __nv_bfloat16*>(q_layers[l]) + (int64_t)gam * q_stride_query;
            rc = run_score(shape, &kv_layers[l], q, q_stride_batch, shape->head_dim, head_mask, 1,
                           first ? s_draft : nullptr, first ? nullptr : s_draft, 1.0f, ws, ws_bytes, st);
            if (rc) return rc;
            first = false;
        }
    }
    return DUSTIN_OK;
}

// ---- cost hint: one-shot sparse layer or dense attention? ---------------------------------------------------------------
// Linear models fitted to the B200 measurements of profiles/r03_sweep.json (Qwen2.5-72B-shaped layer, gamma 4; within
// ~8 % of every point of the fixed-2048 and paper-512 series): each stage is a fixed cost plus its algorithmic bytes over
// the bandwidth that stage reaches.
int dustin_prefer_dense(const dustin_shape_t* shape, uint64_t head_mask, int32_t k, double* fused_us_out,
                        double* dense_us_out) {
    if (check_shape(shape) != DUSTIN_OK || head_mask == 0 || k <= 0) return DUSTIN_ERR_INVALID_ARG;
    const int r = shape->n_q_heads / shape->n_kv_heads;
    int groups = 0;
    for (int g = 0; g < shape->n_kv_heads; ++g) {
        const uint64_t gm = (r >= 64 ? ~0ull : ((1ull << r) - 1ull)) << (g * r);
        if (head_mask & gm) ++groups;
    }
    const double row = (double)shape->head_dim * 2.0;                                     // bytes of one K (or V) row
    const double BN = (double)shape->batch * shape->max_ctx;
    const double keep = k < shape->max_ctx ? (double)k : (double)shape->max_ctx;
    const double a1_us = 12.0 + groups * BN * row / 6.65e6;                               // K stream of the scored groups
    const double a3_us = 27.0;                                                            // selection left on the critical path
    const double a4_us = 9.0 + 2.0 * shape->n_kv_heads * shape->batch * keep * row / 6.1e6;   // gather of the kept K and V rows
    const double a5_us = 12.0 + 2.0 * shape->n_kv_heads * BN * row / 6.6e6;               // every K and V row
    const double fused = a1_us + a3_us + a4_us;
    if (fused_us_out) *fused_us_out = fused;
    if (dense_us_out) *dense_us_out = a5_us;
    return a5_us <= fused ? 1 : 0;
}

// ---- Quest-16 estimator -------------------------------------------------------------------------------------------------
size_t dustin_quest_meta_bytes(const dustin_shape_t* shape) {
    if (check_shape(shape) != DUSTIN_OK) return 0;
    const size_t n_pages = ((size_t)shape->max_ctx + DUSTIN_QUEST_PAGE - 1) / DUSTIN_QUEST_PAGE;
    return (size_t)shape->batch * n_pages * shape->n_kv_heads * 2 * shape->head_dim * sizeof(__nv_bfloat16);
}

int dustin_quest_build_pages(const dustin_shape_t* shape, const dustin_kv_t* kv, const int32_t* first_token,
                             void* page_meta, void* stream) {
    int rc = check_shape(shape);
    if (rc) return rc;
    KvView view;
    rc = check_kv(shape, kv, false, &view);
    if (rc) return rc;
    if (!page_meta || ((uintptr_t)page_meta & 15)) return DUSTIN_ERR_INVALID_ARG;
    const int n_pages = (shape->max_ctx + DUSTIN_QUEST_PAGE - 1) / DUSTIN_QUEST_PAGE;
    const cudaError_t e = launch_quest_build(view, first_token, static_cast<__nv_bfloat16*>(page_meta), shape->batch,
                                             shape->n_kv_heads, shape->head_dim, shape->max_ctx, n_pages,
                                             static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

int dustin_quest_score_pages(const dustin_shape_t* shape, const int32_t* seq_lens, const void* page_meta, const void* q,
                             int64_t q_stride_batch, int64_t q_stride_head, uint64_t head_mask, int32_t n_lists,
                             float* page_scores, float* ub_out, void* ws, size_t ws_bytes, void* stream) {
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!page_meta || ((uintptr_t)page_meta & 15) || !page_scores) return DUSTIN_ERR_INVALID_ARG;
    if (!q || ((uintptr_t)q & 15) || ((q_stride_batch | q_stride_head) & 7) || q_stride_batch < 0 || q_stride_head < 0)
        return DUSTIN_ERR_INVALID_ARG;
    ScoreParams sp;
    std::memset(&sp, 0, sizeof sp);
    rc = build_subset(shape, head_mask, n_lists, &sp);   // same subset / list tables as stage a1
    if (rc) return rc;
    QuestParams p;
    std::memset(&p, 0, sizeof p);
    p.meta = static_cast<const __nv_bfloat16*>(page_meta);
    p.q = static_cast<const __nv_bfloat16*>(q);
    p.q_stride_batch = q_stride_batch;
    p.seq_lens = seq_lens;
    p.batch = shape->batch;
    p.n_kv_heads = shape->n_kv_heads;
    p.head_dim = shape->head_dim;
    p.max_ctx = shape->max_ctx;
    p.n_pages = (shape->max_ctx + DUSTIN_QUEST_PAGE - 1) / DUSTIN_QUEST_PAGE;
    p.n_lists = n_lists;
    p.scale_log2 = scale_log2_of(shape);
    p.scale = p.scale_log2 / kLog2e;
    p.nsel = sp.nsel;
    p.n_groups = sp.n_groups;
    int max_nh = 1;
    for (int gi = 0; gi < sp.n_groups; ++gi) max_nh = sp.group_cnt[gi] > max_nh ? sp.group_cnt[gi] : max_nh;
    quest_plan(p.batch, p.n_groups, max_nh, p.n_pages, &p.group_slots, &p.chunk_pages, &p.n_chunks);
    for (int i = 0; i < sp.nsel; ++i) p.sel_qoff[i] = (int)(sp.sel_head[i] * q_stride_head);
    std::memcpy(p.group_id, sp.group_id, sizeof p.group_id);
    std::memcpy(p.group_first, sp.group_first, sizeof p.group_first);
    std::memcpy(p.group_cnt, sp.group_cnt, sizeof p.group_cnt);
    std::memcpy(p.list_first, sp.list_first, sizeof p.list_first);
    std::memcpy(p.list_cnt, sp.list_cnt, sizeof p.list_cnt);
    p.u_stride = ((long long)p.n_pages + 3) & ~3ll;
    const size_t u_bytes = align256((size_t)p.batch * p.nsel * p.u_stride * sizeof(float));
    if (!ws || ((uintptr_t)ws & 255) || ws_bytes < kWsHeader + u_bytes) return DUSTIN_ERR_WORKSPACE;
    char* base = static_cast<char*>(ws) + kWsHeader;   // the persistent header belongs to the attention stage
    p.u = reinterpret_cast<float*>(base);
    p.ub_out = ub_out;
    const cudaError_t e = launch_quest_score(p, page_scores, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? DUSTIN_OK : fail_cuda(e);
}

size_t dustin_draft_workspace_bytes(const dustin_shape_t* shape, uint64_t head_mask) {
    if (check_shape(shape) != DUSTIN_OK || head_mask == 0) return 0;
    int nsel = popcount64(head_mask) * shape->n_new;
    if (nsel > 64) nsel = popcount64(head_mask);   // the per-token fallback
    return kWsHeader + score_ws(shape->batch, nsel, shape->max_ctx).total + 256;
}

}  // extern "C"

// ---- dustin_score_heads_static: a1 for callers that have no device memory to give (dustin.h) ------------------------
// The scratch of the scoring kernels (log2-domain logits, per-CTA softmax partials, per-head statistics) lives in this
// array instead of a caller-provided workspace.  It is part of the library image: the driver places it on every GPU on
// which the library's code gets loaded and it stays there until the process exits -- DUSTIN_STATIC_SCRATCH_BYTES per GPU,
// used or not.  In host code the name `g_static_scratch` is only a handle for the runtime, NOT a device address: the
// address a kernel can use is asked for below, once per device, with cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[DUSTIN_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kStaticMaxDev = 64;
std::mutex g_static_mu;
void* g_static_ptr[kStaticMaxDev];   // device ordinal -> device address of g_static_scratch there (nullptr: not asked yet)

// Device address of the array on the CURRENT device.  The first call per device is the set-up step: it makes the
// runtime load the library's device code there (which is when the array gets its memory) and looks the symbol up.
cudaError_t static_scratch_here(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" {

int dustin_score_heads_static(const dustin_shape_t* shape, const dustin_kv_t* kv, const void* q, int64_t q_stride_batch,
                              int64_t q_stride_head, uint64_t head_mask, int32_t n_lists, float* scores_now,
                              void* stream) {
    if (!scores_now) return DUSTIN_ERR_INVALID_ARG;
    // Size first, from host values alone: a shape that cannot fit is refused before the device is touched.
    if (check_shape(shape) == DUSTIN_OK && head_mask != 0) {
        const size_t need = kWsHeader + score_ws(shape->batch, popcount64(head_mask), shape->max_ctx).total;
        if (need > (size_t)DUSTIN_STATIC_SCRATCH_BYTES) return DUSTIN_ERR_STATIC_SCRATCH;
    }
    void* scratch = nullptr;
    const cudaError_t e = static_scratch_here(&scratch);
    if (e != cudaSuccess) return fail_cuda(e);
    // Same validation, plan and kernels as dustin_score_heads; only the scratch pointer differs.  Nothing in the scratch
    // has to start at zero (the kernels write every logit, partial and statistic before they read it), so whatever the
    // previous call left behind is harmless and nothing is cleared here.
    return run_score(shape, kv, q, q_stride_batch, q_stride_head, head_mask, n_lists, scores_now, nullptr, 0.f, scratch,
                     (size_t)DUSTIN_STATIC_SCRATCH_BYTES, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
