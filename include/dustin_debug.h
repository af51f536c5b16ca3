/* dustin_debug.h -- measurement, tuning and testing aids of libdustin.so.  NOT part of the product surface: nothing a
 * deployment needs is declared here (that is dustin.h).  bench.py, the tests and profiling scripts use these.
 *
 * Everything in this header is PROCESS-WIDE state (atomics; safe to call from any thread, but a switch flipped while
 * another thread is inside an entry point may or may not apply to that call).  A knob changes which kernel variant
 * serves a call or adds instrumentation; results stay within the tolerances of dustin.h (bitwise equal where dustin.h
 * says bitwise).  The library reads no environment variable.
 */
#ifndef DUSTIN_DEBUG_H_
#define DUSTIN_DEBUG_H_

#include "dustin.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Cache rows per attention CTA of the mma.sync cluster kernel; 0 restores the built-in heuristic.
 * Query dustin_workspace_bytes again after changing it. */
void dustin_tune_attn_split_tokens(int32_t split_tokens);

/* Which attention kernel serves a4/a5.  0 = automatic (the tcgen05 kernel for head_dim 128 and batch * n_kv_heads <=
 * 1024, else the mma.sync cluster kernel), 1 = always the mma.sync cluster kernel, 2 = same as 0.  Results of the two
 * agree within the a4 tolerance, not bitwise.  Query dustin_workspace_bytes again after changing it. */
void dustin_tune_attn_impl(int32_t impl);

/* Generic switches (A/B measurements and test coverage of the rarely taken paths).  Unknown knobs are ignored;
 * dustin_tune_get returns the current value (the default when never set). */
typedef enum dustin_knob {
    DUSTIN_KNOB_PDL = 0,            /* 1 (default): programmatic dependent launch between the kernels of a layer; 0: plain */
    DUSTIN_KNOB_FUSED_ROWS = 1,     /* 1 (default): the fused call normalises + accumulates rows inside the selection
                                       kernels; 0: separate stats / normalise launches as in the staged calls            */
    DUSTIN_KNOB_ATTN_TRACE = 2,     /* bit mask, tcgen05 attention kernel: 8 = timeline samples per role (SM clock, via shared
                                       memory) into the workspace tail, [63] / [62] = %globaltimer at the CTA's start / end;
                                       32 = force equal token ranges (stream-K) even when the whole-unit or even-pieces plan
                                       applies; 64 = griddepcontrol.launch_dependents at the end of the kernel instead of its
                                       start; 1 / 2 = skip the P.V / S MMAs (timing experiments only, results are then wrong: these two
                                       bits act only in a library built with -DDUSTIN_DEBUG_BUILD, the shipped one ignores them) */
    DUSTIN_KNOB_SELECT_SPLIT = 3,   /* CTAs per selection row (thread-block cluster): 0 (default) = heuristic, 1/2/4/8    */
    DUSTIN_KNOB_DRAFT_HOIST = 4,    /* 1 (default): the fused call runs the draft tier of Eq. 6 (I_draft) in a kernel of its
                                       own beside the K stream of a1; 0: both tiers after a1                               */
    DUSTIN_KNOB_SCORE_CHUNK = 5,    /* tokens per CTA of the scoring kernel (multiple of 16, >= 64); 0 (default) = score_plan */
    DUSTIN_KNOB_SELECT_TRACE = 6,   /* 1: selection kernels write %globaltimer samples per phase into the buffer given to
                                       dustin_debug_trace_buffer                                                           */
    DUSTIN_KNOB_L2_HYGIENE = 7,     /* fused call, 1 (default): a selection CTA drops the logits scratch of its row from L2
                                       (discard.global.L2) when it is done, where every logits row has a single reader; 0: the
                                       17 MB of dirty lines per layer are written back while the attention kernel gathers    */
    DUSTIN_KNOB_COUNT = 16
} dustin_knob;
void    dustin_tune_set(int32_t knob, int32_t value);
int32_t dustin_tune_get(int32_t knob);

/* Device buffer that receives the timestamps of DUSTIN_KNOB_SELECT_TRACE: uint64 [n_ctas][64].  NULL / 0 detaches. */
void dustin_debug_trace_buffer(void* device_ptr, size_t bytes);

/* dustin_launch_count: kernels launched by this library in this process so far.
 * dustin_profile_enable(1) starts bracketing every kernel launch with a CUDA event pair on the launching stream
 * (and drops earlier records); dustin_profile_enable(0) stops.  dustin_profile_collect is the one call that
 * synchronises: it waits for the recorded events and writes, per kernel id in [0, DUSTIN_N_KERNELS), the summed
 * device time in ms and the number of launches (host arrays), then clears the records. */
#define DUSTIN_N_KERNELS 13
uint64_t    dustin_launch_count(void);
void        dustin_profile_enable(int32_t on);
int         dustin_profile_collect(double* ms_out, int64_t* launches_out);
const char* dustin_kernel_name(int32_t kernel_id);   /* NULL outside [0, DUSTIN_N_KERNELS) */

/* Reads exactly the K and V rows that dustin_sparse_verify_attn would gather for these index lists -- plain 16-byte
 * loads, no arithmetic -- and writes nothing of interest: its duration is the practical floor of the gather on this
 * memory system.  ws: any scratch of >= DUSTIN_WS_HEADER_BYTES + 4 * batch * n_kv_heads bytes.  Not counted as a launch. */
int dustin_probe_gather(const dustin_shape_t* shape, const dustin_kv_t* kv, const int32_t* idx, const int32_t* cnt,
                        int32_t n_lists, int32_t k_max, void* ws, size_t ws_bytes, void* stream);

/* Occupancy experiments: n_ctas CTAs of `threads` threads and `smem_bytes` of dynamic shared memory that do nothing but
 * hold their SM resources for `microseconds` (they poll %globaltimer).  Launched on `stream`; not counted as a launch. */
int dustin_debug_occupy(int32_t n_ctas, int32_t threads, int32_t smem_bytes, int32_t microseconds, void* stream);

/* Unit-test hook for the block-wide exclusive prefix sum inside the selection kernels (select_impl.inl, block_excl_scan),
 * which is compiled once per CTA size: `threads` in {256, 512, 1024} picks the instantiation.  Every CTA scans its own
 * `threads` values twice, v and v + 1 (mod 2^32).  in: device uint32 [n_blocks][threads];  out: device uint32
 * [2][n_blocks][threads] (exclusive prefixes);  total: device uint32 [2][n_blocks] (block sums).  Not counted as a launch. */
int dustin_debug_block_scan(int32_t threads, int32_t n_blocks, const uint32_t* in, uint32_t* out, uint32_t* total,
                            void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DUSTIN_DEBUG_H_ */
