// kernels.cuh -- parameter blocks and launchers of the four stages (internal; the public surface is dustin.h).
#pragma once

#include "common.cuh"

#include <atomic>

namespace dustin {

// ---- a1 / a2 ------------------------------------------------------------------------------------------------
struct ScoreParams {
    KvView kv;
    const __nv_bfloat16* q;
    long long q_stride_batch, q_stride_head;
    int batch, head_dim, max_ctx, n_lists;
    float scale_log2;        // sm_scale * log2(e): logits live in the log2 domain
    int nsel;                // |subset|; ordinals follow ascending head index, so a KV group's heads are contiguous
    int n_groups;            // KV groups holding >= 1 subset head (the only K rows that are read)
    int chunk_tokens, n_chunks;     // tokens per scoring CTA; softmax partials per (sequence, head) = CTAs per sequence
    int group_slots;                // scored KV groups served side by side by the 8 warps of a CTA: 1, 2, 4 or 8
    int defer_wait;                 // fused call with a hoisted draft tier: the kernel launched just before this one is the
                                    // draft-tier selection, whose results a1 does not need -- the dependency wait moves from
                                    // the start of the kernel to its end (it stays, so that "a1 complete" still implies
                                    // "everything before it complete" for the kernels that follow)
    unsigned char sel_head[64];     // ordinal -> query head
    int sel_qoff[64];               // ordinal -> element offset of its query row inside q + b * q_stride_batch
    unsigned char group_id[64];     // scored group slot -> KV head
    unsigned char group_first[64];  // scored group slot -> first ordinal
    unsigned char group_cnt[64];    // scored group slot -> number of subset heads (<= 8)
    unsigned char list_first[64];   // list -> first ordinal feeding it
    unsigned char list_cnt[64];     // list -> number of ordinals feeding it (empty group => all, reading A2)
    long long logit_stride;         // max_ctx rounded up to a multiple of 4
    float* logits;                  // ws: [B, nsel, logit_stride] log2-domain logits
    float2* part;                   // ws: [B, nsel, n_chunks] (max, sum) in the log2 domain
    float2* stats;                  // ws: [B, nsel] (M, 1/Z)
};

// logits_only: stop after the logits + per-CTA partials; launch_select (SelectParams::norm) then normalises and
// accumulates each row itself.
cudaError_t launch_score(const ScoreParams& p, float* scores_now, float* hist, float alpha, bool logits_only,
                         cudaStream_t stream);
cudaError_t launch_fuse(int batch, int n_lists, int max_ctx, const int* seq_lens, const float* now, float* hist,
                        float alpha, cudaStream_t stream);

// ---- a3 -----------------------------------------------------------------------------------------------------
struct SelectParams {
    int batch, max_ctx, n_lists, k_max;
    const int* seq_lens;
    int budget;
    const int* budgets;
    int n_sink, n_recent, m_num, m_den;
    const float* s_draft;
    long long draft_batch_stride, draft_list_stride;
    const float* s_target;
    int* idx_out;
    int* cnt_out;
    int mask_words, replicas, list_cap;   // shared-memory plan, filled by launch_select
    unsigned long long* trace;            // DUSTIN_KNOB_SELECT_TRACE: [n_ctas][64] %globaltimer samples, else nullptr
    // Split selection of the fused call (select.cu): membership bitmask I_prot U I_draft per (b, list) row, written by
    // the draft-tier kernel and read by the target-tier kernel; draft_mask_stride words per row.
    uint32_t* draft_mask;
    long long draft_mask_stride;
    int draft_rows_per_cta;   // draft-tier kernel of the fused call: rows that one of its CTAs walks (0 / 1: one row each)
    // Row materialisation (fused entry point): when norm.logits != nullptr the kernel first computes its own target
    // row, s_target[b,l,n] = alpha * s_target[b,l,n] + sum_j exp2(logit_j[n] - M_j) / Z_j (a1's normalisation and
    // Eq. 5), from the logits and partials that score_logits_kernel left in the workspace, and writes it back.
    struct Norm {
        const float* logits;            // [B, nsel, logit_stride]
        const float2* part;             // [B, nsel, n_chunks]
        long long logit_stride;
        int nsel, n_chunks;
        int discard_logits;             // every logits row has ONE reader (the CTA of the list it feeds) and is made of whole
                                        // 128-byte lines: that CTA drops the row from L2 when it is done (the lines are dirty
                                        // scratch: left alone they are written back to HBM under the attention kernel's gather)
        float alpha;
        unsigned char list_first[64], list_cnt[64];
    } norm;
};
// mode: 0 = both tiers + list (staged call), 1 = draft tier only (-> p.draft_mask; launched before the scoring kernel
// of the fused call, which it releases at once), 2 = target tier + list (reads p.draft_mask).
cudaError_t launch_select(const SelectParams& p, cudaStream_t stream, int mode = 0);
size_t select_mask_words(int max_ctx);   // words per row of SelectParams::draft_mask
// Few long rows (select_cluster.cu): the target tier (mode 2, with row materialisation) by one thread-block cluster per
// row.  select_cluster_size: CTAs per row, or 0 when one CTA per row serves better / the shape does not qualify.
int select_cluster_size(const SelectParams& p);
cudaError_t launch_select_cluster(const SelectParams& p, int C, cudaStream_t stream);

// ---- a4 / a5 ------------------------------------------------------------------------------------------------
struct AttnParams {
    KvView kv;
    const __nv_bfloat16* q;       // [B,T,Hq,d]
    const __nv_bfloat16* k_new;   // [B,T,Hkv,d]
    const __nv_bfloat16* v_new;
    const int* idx;               // [B,G,k_max] or nullptr (dense)
    const int* cnt;               // [B,G]; may be nullptr when uniform_cnt >= 0
    int uniform_cnt;              // >= 0: every unit holds exactly this many cache rows, known on the host (uniform budget
                                  // and full-length sequences, or the dense baseline without seq_lens): the kernels plan
                                  // without reading a length from memory.  -1: read cnt / seq_lens.
    int batch, n_q_heads, n_kv_heads, group, head_dim, n_new, max_ctx, n_lists, k_max;
    float scale_log2;
    int rows;                     // T * group query rows per KV head
    int split_tokens, n_splits;   // cache tokens per CTA; CTAs per (b, KV head)
    int dbg;
    void* tc_ws;                  // ws of the tcgen05 kernel (attn_tc_ws_bytes), or nullptr => mma.sync cluster kernel
    __nv_bfloat16* out;           // [B,T,Hq,d]
    float* lse_out;               // [B,Hq,T] or nullptr
};
cudaError_t launch_attn(const AttnParams& p, cudaStream_t stream);
// Host-side split heuristic shared by workspace sizing and launch.
void attn_plan(int batch, int n_kv_heads, int max_tokens, int* split_tokens, int* n_splits);
void attn_set_split_override(int split_tokens);
// Bytes at the start of every workspace that persist between calls (completion flags of attn_tc.cu): zero before
// the first use, never touched by the other stages, whose scratch starts right after it.
constexpr size_t kWsHeader = DUSTIN_WS_HEADER_BYTES;
// tcgen05 kernel (attn_tc.cu): head_dim 128, stream-K over tokens, partials + arrival counters in the workspace.
bool attn_tc_usable(int batch, int n_kv_heads, int head_dim, int rows, int max_tokens, int n_new);
size_t attn_tc_ws_bytes(int batch, int n_kv_heads, int rows);
cudaError_t launch_attn_tc(const AttnParams& p, void* ws_base, cudaStream_t stream);
void attn_set_impl(int impl);   // 0 auto, 1 mma.sync cluster kernel, 2 tcgen05 kernel where usable
int attn_get_impl();

// ---- steps either side of the layer path (extras.cu) -----------------------------------------
cudaError_t launch_arr(int batch, int n_lists, int max_ctx, const int* seq_lens, const float* a, const int* idx,
                       const int* cnt, int k_max, float* arr_out, cudaStream_t stream);
// kv.seq_lens must be seq_lens (the lengths before the append); k / v of the view are written.
cudaError_t launch_append(const KvView& kv, int* seq_lens, const int* n_append, const __nv_bfloat16* k_new,
                          const __nv_bfloat16* v_new, int batch, int T, int n_kv_heads, int head_dim, int max_ctx,
                          float* hist, int n_lists, cudaStream_t stream);

// ---- Quest-16 estimator (quest.cu) ----------------------------------------------------------
struct QuestParams {
    const __nv_bfloat16* meta;      // [B, n_pages, Hkv, 2, D]: kmin then kmax of every 16-token page
    const __nv_bfloat16* q;
    long long q_stride_batch;
    const int* seq_lens;
    int batch, n_kv_heads, head_dim, max_ctx, n_pages, n_lists;
    float scale, scale_log2;
    int nsel, n_groups, n_chunks;   // subset size; scored KV groups; scoring CTAs per sequence
    int group_slots, chunk_pages;   // scored KV groups served side by side by the 8 warps of a CTA; pages per CTA (quest_plan)
    int sel_qoff[64];
    unsigned char group_id[64], group_first[64], group_cnt[64], list_first[64], list_cnt[64];   // as in ScoreParams
    long long u_stride;             // n_pages rounded up to a multiple of 4
    float* u;                       // ws: [B, nsel, u_stride] upper-bound logits, log2 domain
    float* ub_out;                  // optional output [B, nsel, n_pages]: the upper-bound logits themselves, or nullptr
};
void quest_plan(int batch, int n_groups, int max_heads_per_group, int n_pages, int* group_slots, int* chunk_pages,
                int* n_chunks);
cudaError_t launch_quest_build(const KvView& kv, const int* first_token, __nv_bfloat16* meta, int batch, int n_kv_heads,
                               int head_dim, int max_ctx, int n_pages, cudaStream_t stream);
cudaError_t launch_quest_score(const QuestParams& p, float* page_scores, cudaStream_t stream);

// Measurement aid: reads the K / V rows that a4 would gather for these lists and does nothing else (sink: >= batch *
// n_kv_heads words of scratch).
cudaError_t launch_gather_probe(const KvView& kv, const int* idx, const int* cnt, int batch, int n_kv_heads, int head_dim,
                                int n_lists, int k_max, void* sink, cudaStream_t stream);

// Test hook: the block-wide exclusive scan of the selection kernels alone, per CTA-size instantiation (256 / 512 / 1024).
cudaError_t launch_scan_test(int threads, int n_blocks, const uint32_t* in, uint32_t* out, uint32_t* total,
                             cudaStream_t stream);

cudaError_t launch_occupy(int n_ctas, int threads, int smem_bytes, int microseconds, cudaStream_t stream);

// ---- launch bookkeeping (profile.cu) ----------------------------------------------------------------------------
enum KernelId {
    kKernScoreLogits = 0, kKernScoreStats, kKernScoreNormalize, kKernFuse, kKernSelect, kKernAttn, kKernSelectDraft,
    kKernArr, kKernAppend, kKernSelectCluster, kKernQuestBuild, kKernQuestScore, kKernQuestNormalize,
    kKernCount
};
// Put one on the stack around a kernel launch: counts it and, when profiling is on, brackets it with CUDA events.
class ProfScope {
public:
    ProfScope(int kid, cudaStream_t stream);
    ~ProfScope();
    ProfScope(const ProfScope&) = delete;
    ProfScope& operator=(const ProfScope&) = delete;
private:
    int kid_;
    cudaStream_t stream_;
    long long slot_;
};
// Tuning knobs of dustin_debug.h (ids: enum dustin_knob), the trace buffer, and per-device caches.
int knob(int id);
void knob_set(int id, int value);
void trace_buffer_set(void* p, size_t bytes);
void* trace_buffer(size_t* bytes);
int current_device();
int device_sm_count();                  // SMs of the current device (cached per device)
struct DeviceOnce {                     // one bit per device ordinal: "attribute already set there"
    std::atomic<unsigned long long> done{0};
};
// cudaFuncAttributeMaxDynamicSharedMemorySize := bytes on the current device, once per (kernel, device); thread-safe.
cudaError_t ensure_dyn_smem(const void* func, int bytes, DeviceOnce& once);
unsigned long long prof_launch_count();
void prof_enable(bool on);
cudaError_t prof_collect(double* ms_out, long long* launches_out);
const char* prof_kernel_name(int kid);

}  // namespace dustin
