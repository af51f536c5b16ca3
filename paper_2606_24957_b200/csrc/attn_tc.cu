// attn_tc.cu -- stage a4 / a5 on the 5th-generation tensor cores (tcgen05 + TMEM) for head_dim 128.
// Sparse verification attention over the selected KV (App. G :568) and, with idx == nullptr, the
// full-cache verification baseline.  DESIGN.md section 5.1.
//
// Decomposition ("stream-K" over tokens).  A unit is one (sequence b, KV head g): its token list is the tile of the T new
// draft rows (needs no index list, so it is worked through while the first gathered rows travel) followed by the cnt[b,l]
// selected cache rows.  The token lists of all units are laid end to end and cut
// into gridDim.x equal ranges, one persistent CTA per SM; a CTA therefore works on a few SEGMENTS (pieces of
// units).  A unit that lies inside one CTA is written straight to `out`; otherwise each piece leaves a normalised
// partial (o, lse) and a completion flag in the workspace, and the CTA that holds the unit's FIRST piece merges them in
// segment order once their flags are up (it pulls from CTAs with lower block indices only, see `rid` below), so the
// result does not depend on the order in which the pieces finish; the merging CTA clears the flags it consumed.
//
// Roles inside a CTA (384 threads; setmaxnreg moves registers from the other warpgroups to the softmax one: 240 / 96 / 96;
// with two softmax warpgroups, 512 threads: 200 / 200 / 56 / 56 -- measured: resolvers or producers below 56 registers
// spill into their loops and cost 2-4 us per launch, 208 for the softmax leaves them 48):
//   warps 0-3  softmax warpgroup: thread = one token of the 128-token tile = one TMEM lane
//   warp  8    MMA issuer (one thread) and TMEM allocation (warps 9-11 only donate their registers)
//   warps 4-7  producers: resolve index -> (page table ->) row address, stream K and V tiles with 16-byte cp.async
//              into the 128-byte-swizzled UMMA layout [64-dim half][token][128 B]; a ring of 32 KB slots in the
//              order K0 V0 K1 V1 ...; completion via cp.async.mbarrier.arrive.noinc on the slot's mbarrier.
// Per tile j:  S^T_j[token,row] = K_j . Q^T   (A = K tile, K-major;  B = Q, K-major;  M = 128, N = NQ, 8 k-steps)
//              P^T_j = exp2(S^T_j * scale - m_ref[row])  written as bf16 into an MN-major (row-contiguous) buffer
//              O^T[dim,row] += V_j^T . P^T_j           (A = V tile, MN-major;  B = P^T, MN-major;  M = 128)
// m_ref is a per-row reference exponent (log2 domain) that is moved only when a score exceeds it by more than 16 (decided
// CTA-uniformly with one bar.red per tile); O^T and the running sums are then rescaled.
#include "kernels.cuh"

#include "../../include/dustin_debug.h"

#include <climits>

// DUSTIN_KNOB_ATTN_TRACE bits 1 / 2 (skip the P.V / S MMAs: timing experiments whose results are wrong) exist only in a
// library built with -DDUSTIN_DEBUG_BUILD; the shipped build has no run-time branch in the MMA issue loop.
#ifdef DUSTIN_DEBUG_BUILD
#define DUSTIN_DBG_SKIP(dbg, bit) (((dbg) & (bit)) != 0)
#else
#define DUSTIN_DBG_SKIP(dbg, bit) false
#endif

namespace dustin {

namespace {

constexpr int kTcThreads = 384;        // three warpgroups: softmax | producers | MMA issuer + resolvers (+ 1 idle warp);
                                       // wide rows: a fourth, the second softmax warpgroup
constexpr int kTile = 128;            // tokens per tile (UMMA M)
constexpr int kD = 128;               // head_dim served by this kernel
constexpr int kSlotBytes = kTile * kD * 2;   // 32 KB: one K or V tile
constexpr int kMaxUnits = 1024;       // prefix array in shared memory
constexpr float kRefSlack = 16.f;     // log2 units a score may exceed m_ref before the reference is moved
constexpr float kRefInit = 0.f;        // reference exponent at the start of a piece (the first tile always moves it)
constexpr float kRefFloor = -1.0e30f;  // lowest reference (rows that have seen nothing but masked tokens)
constexpr long long kInvalidRow = LLONG_MIN;
constexpr int kMergeFast = 4;          // rows of the merge-weight array (only the first is used: the pieces of a cut unit are
                                       // folded in one at a time.  Batching the flag / normaliser loads of up to 8 pieces and
                                       // double-buffering their partial outputs was measured in round 2: 22.7 -> 22.1 us at 128k /
                                       // B = 4, but the extra live registers spill in the 48-row kernel and cost the whole-unit
                                       // case 0.7 us per launch, 31.2 -> 31.9 -- not kept)

// ---- PTX wrappers ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// The mbarrier receives one arrival when all cp.async issued so far by this thread have landed.
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint32_t bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// generic-proxy writes (st.shared, cp.async) -> async-proxy reads (tcgen05.mma operands)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]; bf16 inputs, fp32 accumulate; issued by ONE thread.
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// The mbarrier receives one arrival when every tcgen05.mma issued so far by this thread has completed.
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// This thread's TMEM lane, 16 consecutive 32-bit columns.
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(
            taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}
// 8-column forms (row counts per softmax warpgroup that are multiples of 8 but not of 16: 40 rows at Gamma = 8)
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(v[0]),
                 "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}
// N consecutive columns of this thread's lane (N a multiple of 8) into v
template <int N>
__device__ __forceinline__ void tmem_ld_cols(uint32_t taddr, uint32_t (&v)[N]) {
    static_assert(N % 8 == 0, "column count");
#pragma unroll
    for (int c = 0; c < N / 16; ++c) tmem_ld16(taddr + (uint32_t)c * 16, reinterpret_cast<uint32_t(&)[16]>(v[c * 16]));
    if constexpr (N % 16 != 0) tmem_ld8(taddr + (uint32_t)(N / 16) * 16, reinterpret_cast<uint32_t(&)[8]>(v[(N / 16) * 16]));
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// Named barriers of the softmax warpgroups: id 1 + wg over the 128 threads of warpgroup wg (the .red.or form returns
// the OR of `pred` over them), id 3 over all softmax threads (128 * NWG).
__device__ __forceinline__ void wg_sync(int wg) { asm volatile("bar.sync %0, 128;" ::"r"(1 + wg) : "memory"); }
template <int NWG>
__device__ __forceinline__ void sm_sync() {
    if constexpr (NWG == 1) asm volatile("bar.sync 1, 128;" ::: "memory");
    else asm volatile("bar.sync 3, 256;" ::: "memory");
}
__device__ __forceinline__ bool wg_any(bool pred, int wg) {
    uint32_t r;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t"
        "setp.ne.b32 q, %1, 0;\n\t"
        "bar.red.or.pred p, %2, 128, q;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(r)
        : "r"((uint32_t)pred), "r"(1 + wg)
        : "memory");
    return r != 0;
}

// UMMA shared-memory matrix descriptor (sm_100 format: version 1 in bits [46,48); offsets in 16-byte units).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
           (1ull << 46) | ((uint64_t)layout << 61);
}
constexpr uint32_t kLayoutNone = 0, kLayoutSw128 = 2;
// Instruction descriptor, kind::f16: fp32 accumulate (bit 4), bf16 A (bit 7) and B (bit 10), majors in bits 15/16
// (0 = K-major, 1 = MN-major), N >> 3 in bits [17,23), M >> 4 in bits [24,29).
__host__ __device__ constexpr uint32_t umma_idesc(int m, int n, int a_mn_major, int b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn_major << 15) | ((uint32_t)b_mn_major << 16) |
           ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}

__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Spin until *p != 0.  The writer is a CTA with a lower block index than the caller (see the kernel: range ids run
// against the block indices), i.e. one the hardware has dispatched no later than the caller, so the wait ends without
// the whole grid being co-resident.  A few quick polls, then back off so a long wait does not steal issue slots.
__device__ __forceinline__ void wait_flag(const int* p) {
    int v, polls = 0;
    for (;;) {
        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        if (v != 0) break;
        if (++polls > 16) __nanosleep(polls > 256 ? 256 : 64);
    }
}

// Order-preserving map float <-> int32 (for redux.sync.max.s32); its own inverse.
__device__ __forceinline__ int flip_f32(int b) { return b ^ ((b >> 31) & 0x7fffffff); }
__device__ __forceinline__ float warp_max_f32(float x) {
    const int k = __reduce_max_sync(0xffffffffu, flip_f32(__float_as_int(x)));
    return __int_as_float(flip_f32(k));
}

// Transposing warp reduction of N per-lane values: after it, lane L holds the warp-wide result of kFinal<N> rows,
// row_base(L) + i.  At lane bit B the lanes of a pair split the remaining rows between them (one shuffle per two
// rows); once the count is odd the remaining steps are plain butterflies.  N = 48 takes 48 shuffles instead of 240.
template <int N, int B>
struct TrFinal { static constexpr int value = B == 5 ? N : (N % 2 == 0 ? TrFinal<N / 2, B + 1>::value : TrFinal<N, B + 1>::value); };
template <int N>
struct TrFinal<N, 5> { static constexpr int value = N; };
template <bool MAX>
__device__ __forceinline__ float tr_op(float a, float b) { return MAX ? fmaxf(a, b) : a + b; }
template <bool MAX, int N, int B, int NV>
__device__ __forceinline__ void tr_reduce(float (&v)[NV], int lane, int& row_base) {
    if constexpr (B < 5) {
        if constexpr (N % 2 == 0) {
            constexpr int H = N / 2;
            const bool up = (lane >> B) & 1;
#pragma unroll
            for (int i = 0; i < H; ++i) {
                const float keep = up ? v[i + H] : v[i];
                const float send = up ? v[i] : v[i + H];
                v[i] = tr_op<MAX>(keep, __shfl_xor_sync(0xffffffffu, send, 1 << B));
            }
            if (up) row_base += H;
            tr_reduce<MAX, H, B + 1>(v, lane, row_base);
        } else {
#pragma unroll
            for (int i = 0; i < N; ++i) v[i] = tr_op<MAX>(v[i], __shfl_xor_sync(0xffffffffu, v[i], 1 << B));
            tr_reduce<MAX, N, B + 1>(v, lane, row_base);
        }
    }
}

// ---- shared-memory plan --------------------------------------------------------------------------------------------
template <int NQ>
struct TcCfg {
    static constexpr int kSlotsN = NQ <= 48 ? 6 : 5;
    static constexpr int kQBufs = NQ <= 32 ? 2 : 1;      // 48 rows and more: one Q buffer buys another K/V slot
    static constexpr int kQBytes = NQ * kD * 2;          // one Q buffer, [64-dim half][row][128 B] swizzled
    static constexpr int kPBytes = NQ * kTile * 2;       // P^T, [8-row block][token][16 B]
    static constexpr int kOffSlots = 0;
    static constexpr int kOffQ = kOffSlots + kSlotsN * kSlotBytes;
    static constexpr int kOffP = kOffQ + kQBufs * kQBytes;
    static constexpr int kOffPrefix = kOffP + kPBytes;                    // int [kMaxUnits + 1]
    static constexpr int kOffRef = kOffPrefix + (kMaxUnits + 4) * 4;      // float m_ref[NQ]
    static constexpr int kOffFac = kOffRef + NQ * 4;                      // float fac[NQ]
    static constexpr int kOffDlt = kOffFac + NQ * 4;                      // float dlt[NQ]: m_old - m_new of a reference move
    static constexpr int kOffWarp = kOffDlt + NQ * 4;                     // float [4][NQ]: per-warp maxima / sums
    static constexpr int kOffWgt = kOffWarp + 4 * NQ * 4;                 // float [kMergeFast][NQ]: merge weights
    static constexpr int kOffRowTab = (kOffWgt + kMergeFast * NQ * 4 + 15) & ~15;   // {K row, V row} addresses, 2 tiles
    static constexpr int kOffRowOff = kOffRowTab + 2 * kTile * 16;        // int row -> element offset inside out[b]
    static constexpr int kOffScan = kOffRowOff + NQ * 4;                  // int [16] warp totals / maxima of the scan
    static constexpr int kOffBar = (kOffScan + 16 * 4 + 8 + 7) & ~7;      // uint64 barriers
    static constexpr int kNumBar = 2 * kSlotsN + 14;
    static constexpr int kOffTmem = kOffBar + kNumBar * 8;                // uint32 TMEM base, uint32 combine flag
    static constexpr int kOffTs = kOffTmem + 16;                          // uint32 [64] timeline samples (trace knob)
    static constexpr int kSmemBytes = kOffTs + 256;
    static_assert(kSmemBytes <= 232448, "shared-memory plan exceeds 227 KB");
    static_assert(kOffQ % 1024 == 0 && kQBytes % 1024 == 0 && kOffP % 1024 == 0, "UMMA operands need 1 KB alignment");
};

// ---- segments ---------------------------------------------------------------------------------------------------
// Piece of one unit's token list that falls into this CTA's range of the concatenated token space.
struct Seg {
    int u, b, g, list;
    int cnt;              // cache rows of the unit.  Its token list: positions [0, kTile) = the tile of the T new rows
                          // (the rest of it padding), positions kTile + j = cache row j of the list
    int pos_lo, pos_hi;   // this piece: token positions [pos_lo, pos_hi) of the unit
    int n_tiles;
    int whole;            // the piece is the entire unit: the result goes straight to `out`
    int slot;             // partial slot of this CTA (0: the piece continues a unit begun earlier, 1: otherwise)
    int cta_first, cta_last;   // range ids (gridDim.x - 1 - blockIdx.x) of the CTAs that hold pieces of the unit
};

struct TileCursor {
    const int* prefix;
    int n_units, n_kv, n_lists, lo, hi, chunk;
    int ulen;      // >= 0: every unit is this long and prefix[] holds padded unit starts (even-pieces plan); -1: prefix[u + 1]
    int next_u;
    Seg s;
    int ti;        // tile index inside the segment
    int seg_no;    // running segment number of this CTA
    bool valid;

    __device__ __forceinline__ bool load_seg() {
        if (next_u >= n_units) return false;
        const int ps = prefix[next_u];
        if (ps >= hi) return false;
        const int pe = ulen >= 0 ? ps + ulen : prefix[next_u + 1];
        if (lo >= pe) return false;   // (even-pieces plan: a range in the padding behind the last unit piece)
        s.u = next_u;
        s.b = next_u / n_kv;
        s.g = next_u - s.b * n_kv;
        s.list = n_lists == 1 ? 0 : s.g;
        s.cnt = pe - ps - kTile;
        s.pos_lo = max(lo, ps) - ps;
        s.pos_hi = min(hi, pe) - ps;
        s.n_tiles = (s.pos_hi - s.pos_lo + kTile - 1) / kTile;
        s.whole = (s.pos_lo == 0 && s.pos_hi == pe - ps) ? 1 : 0;
        s.slot = ps <= lo ? 0 : 1;
        s.cta_first = (ps + kTile - 1) / chunk;   // cuts inside the new-row tile are moved to the unit's start (snap_cut)
        s.cta_last = (pe - 1) / chunk;
        ++next_u;
        return true;
    }
    __device__ __forceinline__ void init(const int* prefix_, int n_units_, int n_kv_, int n_lists_, int lo_, int hi_,
                                         int chunk_, int u0, int ulen_) {
        prefix = prefix_; n_units = n_units_; n_kv = n_kv_; n_lists = n_lists_;
        lo = lo_; hi = hi_; chunk = chunk_; next_u = u0; ulen = ulen_;
        ti = 0; seg_no = 0;
        valid = load_seg();
    }
    __device__ __forceinline__ bool last_tile() const { return ti == s.n_tiles - 1; }
    // The tile of the unit's new rows (positions [0, kTile)): no piece starts inside it (make_plan), so it is exactly the
    // first tile of a piece that starts its unit.  Every other tile holds gathered cache rows only.
    __device__ __forceinline__ bool new_tile() const { return s.pos_lo == 0 && ti == 0; }
    __device__ __forceinline__ void advance() {
        if (++ti >= s.n_tiles) {
            ti = 0;
            ++seg_no;
            valid = load_seg();
        }
    }
};

// ---- plan -------------------------------------------------------------------------------------------------------
// Range [lo, hi) of the concatenated token space that the CTA of range id `rid` works through, and the first unit in
// it.  prefix(u) = start of unit u (prefix(n_units) = total); unit_of(x) = largest u with prefix(u) <= x.
struct Plan {
    int lo, hi, u0, chunk;
    bool whole;   // every CTA takes one whole unit
};
template <class PrefixFn, class UnitOfFn>
__device__ __forceinline__ Plan make_plan(PrefixFn prefix, UnitOfFn unit_of, int n_units, int longest, int grid, int rid,
                                          bool force_stream) {
    Plan pl;
    const int total = prefix(n_units);
    pl.chunk = (((total + grid - 1) / grid) + 31) & ~31;
    // Few units of similar length (at most one per CTA, the longest not much above the even share): every CTA
    // takes one WHOLE unit -- no partials, no merge, one epilogue -- and the memory system, not the idle SMs, sets
    // the pace.  Otherwise: equal token ranges (stream-K).
    pl.whole = n_units <= grid && longest <= total / grid + 4 * kTile && !force_stream;
    pl.u0 = 0;
    if (pl.whole) {
        pl.lo = rid < n_units ? prefix(rid) : total;
        pl.hi = rid < n_units ? prefix(rid + 1) : total;
        pl.u0 = min(rid, n_units - 1);
    } else {
        // A cut that falls inside the new-row tile of a unit moves down to the unit's start, so that no piece begins in
        // the padding of that tile (its first tile would hold nothing visible to some query rows).  Seg::cta_first agrees.
        auto snap_cut = [&](long long x) -> int {
            if (x >= total) return total;
            const int ps = prefix(unit_of((int)x));
            return (int)x - ps < kTile ? ps : (int)x;
        };
        const long long c0 = (long long)rid * pl.chunk;
        pl.lo = snap_cut(c0);
        pl.hi = snap_cut(c0 + pl.chunk);
        if (pl.lo < pl.hi) pl.u0 = unit_of(pl.lo);
    }
    return pl;
}

// Even-pieces plan: CTAs per unit (>= 2), or 0 when it does not apply.  Units of one length `len` (new-row tile included),
// at most half as many as CTAs, at least two tiles per piece.
__device__ __forceinline__ int even_pieces_per_unit(int len, int n_units, int grid) {
    if (n_units <= 0 || n_units * 2 > grid) return 0;
    const int n_tiles = (len + kTile - 1) / kTile;
    const int ppu = min(grid / n_units, n_tiles / 2);
    return ppu >= 2 ? ppu : 0;
}

// ---- kernel -----------------------------------------------------------------------------------------------------
struct TcWs {
    int* flags;         // [grid, 2] "partial is in the workspace" flags, zeroed before the launch
    unsigned long long* dbg_ts;   // optional timeline (DUSTIN_DBG & 8): [grid][64] globaltimer samples
    float* part_o;      // [grid, 2, rows, 128] normalised partial outputs
    float* part_lse;    // [grid, 2, rows] log2-domain normalisers
};

__device__ __forceinline__ unsigned long long gtimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ uint32_t clock32() {
    uint32_t t;
    asm volatile("mov.u32 %0, %clock;" : "=r"(t));
    return t;
}
// Timeline samples (DUSTIN_KNOB_ATTN_TRACE & 8): SM clock into shared memory (a %globaltimer read is far too slow to sit on
// the paths it is meant to time), copied to the workspace tail when the CTA ends; slot 63 holds %globaltimer at the start.
#define TS(slot) do { if (p.dbg & 8) s_ts[(slot)] = clock32(); } while (0)

template <int NQ, int NWG, bool GATHER>
__global__ void __launch_bounds__(kTcThreads + 128 * (NWG - 1), 1) attn_tc_kernel(const AttnParams p, const TcWs ws) {
    using C = TcCfg<NQ>;
    constexpr int NS = C::kSlotsN;
    // Producer warpgroups: one (warps 4-7 copy the K and the V tiles).  A second one for the V tiles (warps 12-15 when
    // there is a single softmax warpgroup) was measured: the copies are bound by the SM's cp.async path (one 512-byte
    // warp instruction per ~20 cycles, whoever issues it), eight warps only contend for it -- 1.49 instead of 1.31 us a tile.
    constexpr int NPW = 1;
    extern __shared__ __align__(1024) unsigned char smem[];   // 128-byte-swizzled operands need 1 KB alignment
    const uint32_t sbase = smem_u32(smem);
    if (sbase & 1023u) __trap();
    int* s_prefix = reinterpret_cast<int*>(smem + C::kOffPrefix);
    float* s_ref = reinterpret_cast<float*>(smem + C::kOffRef);
    float* s_fac = reinterpret_cast<float*>(smem + C::kOffFac);
    float* s_dlt = reinterpret_cast<float*>(smem + C::kOffDlt);
    float* s_warp = reinterpret_cast<float*>(smem + C::kOffWarp);
    float* s_wgt = reinterpret_cast<float*>(smem + C::kOffWgt);
    int* s_rowoff = reinterpret_cast<int*>(smem + C::kOffRowOff);
    int* s_scan = reinterpret_cast<int*>(smem + C::kOffScan);
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(smem + C::kOffTmem);
    const uint32_t bar0 = sbase + C::kOffBar;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    // barrier indices
    constexpr int kSlotFull = 0, kSlotEmpty = NS, kQFull = 2 * NS, kQEmpty = 2 * NS + 2, kSFull = 2 * NS + 4,
                  kSEmpty = 2 * NS + 6, kPFull = 2 * NS + 8, kPvDone = 2 * NS + 9, kTabFull = 2 * NS + 10,
                  kTabEmpty = 2 * NS + 12;
    constexpr int kTabs = 2;   // tiles of row addresses in the table ring

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int T = p.n_new, r = p.group, rows = p.rows, Hkv = p.n_kv_heads, Hq = p.n_q_heads;
    const int n_units = p.batch * Hkv;
    // Range id of this CTA in the cut of the concatenated token space: it runs AGAINST the block index.  The CTA that
    // merges a unit (the one holding the unit's first piece, i.e. its lowest range id) then waits for CTAs with higher
    // range ids = LOWER block indices, which were dispatched no later than itself: no co-residency assumption.
    const int rid = (int)gridDim.x - 1 - (int)blockIdx.x;
    uint32_t* s_ts = reinterpret_cast<uint32_t*>(smem + C::kOffTs);
    if (p.dbg & 8) {
        if (tid < 64) s_ts[tid] = 0;
        __syncthreads();
        if (tid == 0 && ws.dbg_ts) ws.dbg_ts[(size_t)blockIdx.x * 64 + 63] = gtimer();
    }
    if (tid == 0) TS(0);
    // Let the next kernel's CTAs be scheduled from now on (they take an SM as soon as its CTA of this grid exits, run
    // their prologue and stop at their own dependency wait, which still waits for this whole grid to complete).  The
    // hardware holds them back until every CTA of this grid has started, so they cannot take an SM this grid needs.
    if (!(p.dbg & 64)) pdl_trigger();
    // ---- token-list lengths of all units -> exclusive prefix sums (threads 0..255) --------------------------------
    // A unit's token list is the tile of its T new rows (kTile virtual positions, see Seg) followed by its cache rows.
    // The new rows need no index list and come first: their tile is worked through while the first gathered rows are
    // still on their way, instead of costing a nearly empty tile at the end of the unit.
    auto unit_len = [&](int u) -> int {
        const int b = u / Hkv;
        int c;
        if (p.uniform_cnt >= 0) {
            c = p.uniform_cnt;
        } else if (GATHER) {
            const int list = p.n_lists == 1 ? 0 : u - b * Hkv;
            c = __ldg(p.cnt + b * p.n_lists + list);
            c = c < 0 ? 0 : (c > p.k_max ? p.k_max : c);
        } else {
            c = seq_len_of(p.kv.seq_lens, b, p.max_ctx);
        }
        return c + kTile;
    };
    // Barriers and TMEM need nothing from global memory: under programmatic dependent launch this part runs while the
    // previous kernel drains; pdl_wait() returns when that kernel has completed and its writes are visible.
    // Lengths known on the host (uniform budget over full-length sequences; the dense baseline without seq_lens): the
    // whole plan is arithmetic and is laid out before the dependency wait.  Otherwise the lengths are read after it.
    const bool uniform = p.uniform_cnt >= 0;
    Plan pl;
    // Uniform lengths, one whole unit per CTA, gathered rows (the shape of the headline workload): the resolver warps ask
    // for the index entries of the first two gathered tiles right here, in as few instructions as possible (at the
    // start of a launch every line of code is an instruction-cache miss), so that their trip overlaps the rest of the
    // prologue.  The conditions restate make_plan's for this case.
    int early_tok[4] = {-1, -1, -1, -1};
    bool early = false;
    if (GATHER && uniform && (warp == 9 || warp == 10) && rid < n_units && n_units <= (int)gridDim.x && !(p.dbg & 32) &&
        even_pieces_per_unit(p.uniform_cnt + kTile, n_units, (int)gridDim.x) == 0) {
        const int len = p.uniform_cnt + kTile;
        if (len <= (n_units * len) / (int)gridDim.x + 4 * kTile) {
            const int first = (warp - 9) * kTile + lane;   // cache position of this lane's first row
            const int* lrow = p.idx + (long long)(p.n_lists == 1 ? rid / Hkv : rid) * p.k_max + first;
            early = true;
            pdl_wait();
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (first + 32 * i < p.uniform_cnt) early_tok[i] = __ldg(lrow + 32 * i);
        }
    }
    if (tid == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(bar(kSlotFull + i), 128);
            mbar_init(bar(kSlotEmpty + i), 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar(kQFull + i), 128);
            mbar_init(bar(kQEmpty + i), 1);
            mbar_init(bar(kSFull + i), 1);
            mbar_init(bar(kSEmpty + i), 128 * NWG);
        }
        mbar_init(bar(kPFull), 128 * NWG);
        mbar_init(bar(kPvDone), 1);
        for (int i = 0; i < kTabs; ++i) {
            mbar_init(bar(kTabFull + i), 1);    // the resolver warp of the table
            mbar_init(bar(kTabEmpty + i), 4 * NPW);   // the producer warps
        }
        fence_mbar_init();
    }
    if (warp == 8) tmem_alloc(smem_u32(s_tmem), 512);
    if (!uniform) {
        pdl_wait();
        if (tid == 0) TS(57);
    }
    const int per = (n_units + 255) / 256;
    const int u_lo = min(tid * per, n_units), u_hi = tid < 256 ? min(u_lo + per, n_units) : u_lo;
    // Even-pieces plan (gathered rows, all units of one length, at most half as many units as CTAs: 64k / 128k contexts at
    // small batch): ppu CTAs per unit, every CTA ONE piece of tpp whole tiles of ONE unit; the CTAs beyond n_units * ppu
    // stay idle.  Equal token ranges over all 148 CTAs give some CTAs the tail of one unit and the head of the next: two
    // epilogues, a second Q load and 4.6 pieces per unit to merge instead of 4 (measured: 128k / B = 4 22.8 -> 19.7 us,
    // 64k / B = 8 25.8 -> 22.1 us, 128k / k = 8192 39.8 -> 37.5 us; the dense baseline, which streams far more per unit,
    // loses: 341 -> 372 us, hence gathered rows only).  The unit starts are padded to ppu * tpp tiles so that the cuts are
    // plain multiples of the chunk.  Whether the lengths are equal is a property of the data, not of how the kernel learnt
    // them: the same decomposition follows from the host's hint and from the lengths read below (bit-identical results).
    int ulen = uniform ? p.uniform_cnt + kTile : -1;                   // common unit length, -1: not (yet) known to be one
    int ppu = (GATHER && uniform && !(p.dbg & 32)) ? even_pieces_per_unit(ulen, n_units, (int)gridDim.x) : 0;
    int even_chunk = ppu >= 2 ? ((ulen + kTile - 1) / kTile + ppu - 1) / ppu * kTile : 0;
    if (uniform) {
        const int len = ppu >= 2 ? ppu * even_chunk : p.uniform_cnt + kTile;
        for (int u = u_lo; u < u_hi; ++u) s_prefix[u] = u * len;
        if (tid == 255) s_prefix[n_units] = n_units * len;
    } else {
        int sum = 0, longest = 0;
        for (int u = u_lo; u < u_hi; ++u) {
            const int l = unit_len(u);
            sum += l;
            longest = max(longest, l);
        }
        int inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += v;
        }
        longest = __reduce_max_sync(0xffffffffu, longest);
        const int wsum = __shfl_sync(0xffffffffu, inc, 31);   // stored from lane 0 (see block_excl_scan in select_impl.inl)
        if (lane == 0 && warp < 8) {
            s_scan[warp] = wsum;
            s_scan[8 + warp] = longest;
        }
        __syncthreads();
        int base = 0;
        for (int w = 0; w < warp && w < 8; ++w) base += s_scan[w];
        int run = base + inc - sum;
        for (int u = u_lo; u < u_hi; ++u) {
            s_prefix[u] = run;
            run += unit_len(u);
        }
        if (tid == 255) s_prefix[n_units] = run;
        if (GATHER && !(p.dbg & 32)) {
            // lengths read from memory: all equal?  (total == n_units * longest)  Then the even-pieces plan applies as above.
            __syncthreads();
            int longest_all = 0;
#pragma unroll
            for (int w = 0; w < 8; ++w) longest_all = max(longest_all, s_scan[8 + w]);
            if (s_prefix[n_units] == n_units * longest_all) {
                const int pp = even_pieces_per_unit(longest_all, n_units, (int)gridDim.x);
                if (pp >= 2) {   // (uniform over the CTA)
                    ulen = longest_all;
                    ppu = pp;
                    even_chunk = ((ulen + kTile - 1) / kTile + ppu - 1) / ppu * kTile;
                    __syncthreads();   // everybody has read the exact prefix
                    for (int u = u_lo; u < u_hi; ++u) s_prefix[u] = u * ppu * even_chunk;
                    if (tid == 255) s_prefix[n_units] = n_units * ppu * even_chunk;
                }
            }
        }
    }
    if (tid < NQ) {
        s_ref[tid] = kRefInit;
        s_rowoff[tid] = ((tid / r) * Hq + tid % r) * kD;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (tid == 0) TS(1);
    const uint32_t tmem = *s_tmem;
    constexpr uint32_t kColS = 0, kColO = 256;   // S buffers at columns 0 and 128, O^T at 256
    if (ppu >= 2) {
        pl.chunk = even_chunk;
        pl.whole = false;
        pl.u0 = min(rid / ppu, n_units - 1);
        pl.lo = rid < n_units * ppu ? rid * even_chunk : n_units * ppu * even_chunk;
        pl.hi = rid < n_units * ppu ? pl.lo + even_chunk : pl.lo;
        if (pl.lo >= pl.u0 * ppu * even_chunk + ulen) pl.hi = pl.lo;   // nothing of the unit left for this piece
    } else if (uniform) {
        const int len = p.uniform_cnt + kTile;
        pl = make_plan([&](int u) { return u * len; }, [&](int x) { return min(x / len, n_units - 1); }, n_units, len,
                       (int)gridDim.x, rid, (p.dbg & 32) != 0);
    } else {
        int longest_all = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) longest_all = max(longest_all, s_scan[8 + w]);
        pl = make_plan([&](int u) { return s_prefix[u]; },
                       [&](int x) {
                           int a = 0, bnd = n_units;
                           while (bnd - a > 1) {
                               const int m = (a + bnd) >> 1;
                               if (s_prefix[m] <= x) a = m; else bnd = m;
                           }
                           return a;
                       },
                       n_units, longest_all, (int)gridDim.x, rid, (p.dbg & 32) != 0);
    }
    const int lo = pl.lo, hi = pl.hi, u0 = pl.u0, chunk = pl.chunk;
    const bool active = lo < hi;   // a CTA past the end of the token space only takes part in the teardown
    if (tid == 0) TS(2);
    if (uniform) {
        pdl_wait();
        if (tid == 0) TS(57);
    }

    TileCursor cur;
    cur.init(s_prefix, n_units, Hkv, p.n_lists, lo, hi, chunk, u0, ppu >= 2 ? ulen : -1);
    if (!active) cur.valid = false;

    if ((warp >= 4 && warp < 8) || (NPW == 2 && warp >= 12)) {
        // ================= producers ===========================================================================
        if constexpr (NWG == 1) asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        const bool do_k = warp < 8, do_v = NPW == 1 || warp >= 12;
        const int pw = warp & 3, ptid = do_k ? tid - 128 : -1;
        // lane = 16-byte chunk c of rows 2i + h (h = lane / 16), i = 0..15, of this warp's 32 rows of the tile.
        // Destination inside a slot: [64-dim half c/8][row][128 B], chunk XOR (row & 7); rows 2i + h and
        // 2(i + 4) + h share the swizzle term and lie 1 KB apart.
        const int c = lane & 15, h = lane >> 4;
        uint32_t dsw[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int row = 32 * pw + 2 * q + h;
            dsw[q] = (uint32_t)(c >> 3) * (kTile * 128) + (uint32_t)row * 128 + (uint32_t)(((c & 7) ^ (row & 7)) << 4);
        }
        const ulonglong2* tab_rd = reinterpret_cast<const ulonglong2*>(smem + C::kOffRowTab) + 32 * pw + h;
        const unsigned long long coff = (unsigned long long)c * 16;
        const unsigned long long kdummy = (unsigned long long)p.kv.k;   // never read (src-size 0)
        // (An evict_first hint on these copies -- the rows are read once -- was measured: the attention kernel alone gains
        // 0.3 us, the fused layer loses 2.4: the dirty score rows of the selection kernel then stay in L2 until the next
        // layer's K stream has to write them back.)
        // K and V tiles of tile gj: items 2gj and 2gj+1 of the slot ring; row addresses from the resolver warps' table
        auto issue_tile = [&](int gj, int ord) {   // ord: ordinal of the tile among the CTA's gathered tiles
            const int ik = 2 * gj, iv = 2 * gj + 1, sk = ik % NS, sv = iv % NS, tb = ord % kTabs;
            mbar_wait(bar(kTabFull + tb), ((uint32_t)(ord / kTabs)) & 1u);
            if (do_k) mbar_wait(bar(kSlotEmpty + sk), (((uint32_t)(ik / NS)) & 1u) ^ 1u);
            if (do_v) mbar_wait(bar(kSlotEmpty + sv), (((uint32_t)(iv / NS)) & 1u) ^ 1u);
            const uint32_t dk = sbase + C::kOffSlots + (uint32_t)sk * kSlotBytes;
            const uint32_t dv = sbase + C::kOffSlots + (uint32_t)sv * kSlotBytes;
            const ulonglong2* trow = tab_rd + tb * kTile;
            // (unrolled by 4, not 16: the first pass through this code is an instruction-cache miss per line, and it sits
            // between the launch and the first request for cache rows)
#pragma unroll 1
            for (int i4 = 0; i4 < 4; ++i4) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const ulonglong2 a = trow[2 * (4 * i4 + q)];
                    const uint32_t d = dsw[q] + (uint32_t)i4 * 1024;
                    const int nb = a.x != 0ull ? 16 : 0;
                    if (NPW == 1 || do_k) cp_async16(dk + d, reinterpret_cast<const void*>((nb ? a.x : kdummy) + coff), nb);
                    if (NPW == 1 || do_v) cp_async16(dv + d, reinterpret_cast<const void*>((nb ? a.y : kdummy) + coff), nb);
                }
            }
            if (do_k) cp_async_mbar_arrive_noinc(bar(kSlotFull + sk));
            if (do_v) cp_async_mbar_arrive_noinc(bar(kSlotFull + sv));
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(kTabEmpty + tb));   // this warp has read its 32 entries
        };

        // The tile of a unit's new rows: row u < T of the tile is new row u; the rest is padding, zeroed with plain stores
        // (the copy path is the SM's scarcest resource: a tile of zero-filling copies would cost as much of it as a tile of
        // cache rows).  K padding only has to be there; V padding must be finite, since it meets P = 0 in the MMA.
        auto issue_new = [&](int gj) {
            const int ik = 2 * gj, iv = 2 * gj + 1, sk = ik % NS, sv = iv % NS;
            mbar_wait(bar(kSlotEmpty + sk), (((uint32_t)(ik / NS)) & 1u) ^ 1u);
            mbar_wait(bar(kSlotEmpty + sv), (((uint32_t)(iv / NS)) & 1u) ^ 1u);
            const uint32_t dk = sbase + C::kOffSlots + (uint32_t)sk * kSlotBytes;
            const uint32_t dv = sbase + C::kOffSlots + (uint32_t)sv * kSlotBytes;
            const long long o0 = (((long long)cur.s.b * T + (32 * pw + h)) * Hkv + cur.s.g) * kD + c * 8;   // row 32 pw + h
#pragma unroll 1
            for (int i4 = 0; i4 < 4; ++i4) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int i = 4 * i4 + q;
                    const uint32_t d = dsw[q] + (uint32_t)i4 * 1024;
                    if (32 * pw + 2 * i + h < T) {
                        const long long o = o0 + (long long)(2 * i) * Hkv * kD;
                        cp_async16(dk + d, p.k_new + o, 16);
                        cp_async16(dv + d, p.v_new + o, 16);
                    } else {
                        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(dk + d), "r"(0) : "memory");
                        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(dv + d), "r"(0) : "memory");
                    }
                }
            }
            fence_proxy_async();   // the plain stores, before the arrivals that hand the slots to the MMA
            cp_async_mbar_arrive_noinc(bar(kSlotFull + sk));
            cp_async_mbar_arrive_noinc(bar(kSlotFull + sv));
        };

        if (ptid == 0) TS(58);
        // The T*r query rows of the cursor's segment (zero-padded to NQ) into Q buffer seg_no % kQBufs.
        auto issue_q = [&]() {
            const int k = cur.seg_no, qb = k % C::kQBufs;
            mbar_wait(bar(kQEmpty + qb), (((uint32_t)(k / C::kQBufs)) & 1u) ^ 1u);
            const uint32_t qdst = sbase + C::kOffQ + (uint32_t)qb * C::kQBytes;
            const __nv_bfloat16* qsrc = p.q + ((long long)cur.s.b * T * Hq + (long long)cur.s.g * r) * kD;
#pragma unroll 1
            for (int x0 = 0; x0 < NQ * 16; x0 += 128) {
                const int x = x0 + ptid, rr = x >> 4, cc = x & 15;
                const bool ok = rr < rows;
                const __nv_bfloat16* src = ok ? qsrc + s_rowoff[rr] + cc * 8 : p.q;
                cp_async16(qdst + (uint32_t)(cc >> 3) * (NQ * 128) + (uint32_t)rr * 128 +
                               (uint32_t)(((cc & 7) ^ (rr & 7)) << 4), src, ok ? 16 : 0);
            }
            cp_async_mbar_arrive_noinc(bar(kQFull + qb));
        };
        int gj = 0, ord = 0;
#pragma unroll 1
        while (cur.valid) {
            if (cur.ti == 0 && do_k) issue_q();    // new segment: its query rows
            if (cur.new_tile()) {
                issue_new(gj);
            } else {
                issue_tile(gj, ord);
                ++ord;
            }
            if (ptid == 0 && gj < 3) TS(4 + gj);
            cur.advance();
            ++gj;
        }
    } else if (warp >= 8 && warp < 12) {
        // ================= MMA issuer (one thread of warp 8) =====================================================
        if constexpr (NWG == 1) asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp > 8) {
            // ================= resolver warps 9 and 10: warp 9 + w serves the gathered tiles of ordinal w, w + 2, ... ====
            // index entry -> (page table ->) absolute addresses of the K and the V row, for the 128 rows of a tile of
            // cache rows (4 per lane, all loads of a tile in flight together), into table w of two in shared memory, which
            // the producers read.  Each warp has two tile periods for its chain of dependent loads, so the producers do not
            // wait for an index in the steady state; in the whole-unit case the entries of the first two tiles were
            // requested at the top of the kernel.  (One warp per table: a warp then waits on consecutive phases of its
            // table's barrier and cannot run a phase ahead.)  The new-row tiles need no table: the producers address them.
            const int rw = warp - 9;
            if (rw < kTabs) {
                ulonglong2* tabw = reinterpret_cast<ulonglong2*>(smem + C::kOffRowTab) + rw * kTile;
                // cache rows (token indices) of rows lane + 32 i of the cursor's tile; -1 = past the end of the piece
                auto load4 = [&](const TileCursor& c, int (&tok)[4]) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) tok[i] = -1;
                    if (!c.valid) return;
                    const Seg& sg = c.s;
                    const int pos0 = sg.pos_lo + c.ti * kTile + lane;
                    const int* lrow = GATHER ? p.idx + ((long long)sg.b * p.n_lists + sg.list) * p.k_max - kTile : nullptr;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int pos = pos0 + 32 * i;
                        if (pos < sg.pos_hi) tok[i] = GATHER ? __ldg(lrow + pos) : pos - kTile;
                    }
                };
                if (rw == 0 && lane == 0) TS(62);
                TileCursor rc = cur;
                int ord = 0, want = rw;   // ord: gathered tiles before the cursor's; want: the ordinal this warp serves next
                auto seek = [&]() {
                    while (rc.valid) {
                        if (!rc.new_tile()) {
                            if (ord == want) return;
                            ++ord;
                        }
                        rc.advance();
                    }
                };
                seek();
                int tok[4];
                if (early) {   // whole unit: requested at the top of the kernel
#pragma unroll
                    for (int i = 0; i < 4; ++i) tok[i] = early_tok[i];
                } else {
                    load4(rc, tok);
                }
                int use = 0;   // how many times this warp has filled its table
#pragma unroll 1
                while (rc.valid) {
                    const int sb_ = rc.s.b, sg_ = rc.s.g;
                    ulonglong2 a[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        a[i].x = a[i].y = 0ull;   // past the end of the piece: zero-filled by the copy (src-size 0)
                        if (tok[i] >= 0) {
                            const long long off = kv_row_offset(p.kv, sb_, tok[i], sg_);
                            a[i].x = (unsigned long long)(p.kv.k + off);
                            a[i].y = (unsigned long long)(p.kv.v + off);
                        }
                    }
                    mbar_wait(bar(kTabEmpty + rw), ((uint32_t)use & 1u) ^ 1u);
#pragma unroll
                    for (int i = 0; i < 4; ++i) tabw[lane + 32 * i] = a[i];
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(kTabFull + rw));
                    if (rw == 0 && lane == 0 && use == 0) TS(50);
                    if (rw == 0 && lane == 0 && use == 1) TS(7);
                    want += kTabs;
                    seek();
                    load4(rc, tok);   // this warp's next tile
                    ++use;
                }
            }
        } else if (lane == 0) {
            constexpr uint32_t idesc_s = umma_idesc(kTile, NQ, 0, 0);    // S^T = K . Q^T : both K-major
            constexpr uint32_t idesc_pv = umma_idesc(kTile, NQ, 1, 1);   // O^T = V^T . P^T : both MN-major
            const uint32_t slots = sbase + C::kOffSlots, pbuf = sbase + C::kOffP;
            auto issue_pv = [&](int j, bool first_of_seg) {
                mbar_wait(bar(kPFull), (uint32_t)j & 1u);
                const int item = 2 * j + 1, slot = item % NS;
                mbar_wait(bar(kSlotFull + slot), ((uint32_t)(item / NS)) & 1u);
                fence_proxy_async();
                tc_fence_after();
                const uint32_t vb = slots + (uint32_t)slot * kSlotBytes;
#pragma unroll
                for (int ks = 0; ks < kTile / 16; ++ks) {
                    // A = V tile as [dim (M), token (K)], dim contiguous: 64-dim halves 16 KB apart (LBO), 8-token
                    // groups 1 KB apart (SBO);  B = P^T as [row (N), token (K)], row contiguous, no swizzle:
                    // 8-row blocks 2 KB apart (SBO), 8-token groups 128 B apart (LBO).
                    const uint64_t ad = umma_desc(vb + (uint32_t)ks * 2048, kTile * 128, 1024, kLayoutSw128);
                    const uint64_t bd = umma_desc(pbuf + (uint32_t)ks * 256, 128, 2048, kLayoutNone);
                    if (!DUSTIN_DBG_SKIP(p.dbg, 1)) umma_bf16(tmem + kColO, ad, bd, idesc_pv, (first_of_seg && ks == 0) ? 0u : 1u);
                }
                umma_commit(bar(kSlotEmpty + slot));
                umma_commit(bar(kPvDone));
            };
            int gj = 0;
            bool have_prev = false, prev_first = false;
            while (cur.valid) {
                const int k = cur.seg_no, qb = k % C::kQBufs;
                const uint32_t qpar = ((uint32_t)(k / C::kQBufs)) & 1u;
                const int item = 2 * gj, slot = item % NS, sb = gj & 1;
                // S of this tile first, then P.V of the previous one.  (Issuing whichever is ready first was measured on
                // the 4- and 5-slot rings: it only helps when the ring is too short to hold two tiles besides the one
                // in use, which no variant is any more.)
                if (cur.ti == 0) mbar_wait(bar(kQFull + qb), qpar);
                mbar_wait(bar(kSlotFull + slot), ((uint32_t)(item / NS)) & 1u);
                mbar_wait(bar(kSEmpty + sb), (((uint32_t)(gj >> 1)) & 1u) ^ 1u);
                fence_proxy_async();
                tc_fence_after();
                const uint32_t kb = slots + (uint32_t)slot * kSlotBytes;
                const uint32_t qbuf = sbase + C::kOffQ + (uint32_t)qb * C::kQBytes;
#pragma unroll
                for (int ks = 0; ks < kD / 16; ++ks) {
                    // both operands K-major, 128-byte swizzle: rows 128 B apart, 8-row groups 1 KB apart (SBO); the
                    // k-step moves 32 B inside the swizzled row, the second 64-dim half sits one [rows][128 B] on
                    const uint64_t ad = umma_desc(kb + (uint32_t)(ks >> 2) * (kTile * 128) + (uint32_t)(ks & 3) * 32, 16,
                                                  1024, kLayoutSw128);
                    const uint64_t bd = umma_desc(qbuf + (uint32_t)(ks >> 2) * (NQ * 128) + (uint32_t)(ks & 3) * 32, 16,
                                                  1024, kLayoutSw128);
                    if (!DUSTIN_DBG_SKIP(p.dbg, 2)) umma_bf16(tmem + kColS + (uint32_t)sb * 128, ad, bd, idesc_s, ks > 0 ? 1u : 0u);
                }
                umma_commit(bar(kSlotEmpty + slot));
                umma_commit(bar(kSFull + sb));
                if (gj < 4) TS(8 + gj);
                if (cur.last_tile()) umma_commit(bar(kQEmpty + qb));
                if (have_prev) issue_pv(gj - 1, prev_first);
                have_prev = true;
                prev_first = cur.ti == 0;
                cur.advance();
                ++gj;
            }
            if (have_prev) issue_pv(gj - 1, prev_first);
        }
        __syncwarp();
    } else {
        // ================= softmax warpgroup: thread = token of the tile = TMEM lane ==============================
        // NWG = 2 (T*r > 48): a second softmax warpgroup (warps 12-15) takes the query rows [NW, 2 NW); the two own
        // the same TMEM lanes (warp % 4) and disjoint columns, rows of s_ref / s_fac / P / partials, and meet only on
        // the mbarriers (S consumed, P ready: 128 arrivals each) and where a flag is published or cleared.
        if constexpr (NWG == 1) asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
        constexpr int NW = NQ / NWG;
        const int wg = (NWG == 2 && warp >= 12) ? 1 : 0;
        const int c_off = wg * NW, wq = warp & 3;
        const int t = tid - wg * 384;   // (warps 12-15 are the second softmax warpgroup only when NWG == 2)
        const int rows_w = min(max(rows - c_off, 0), NW);
        const uint32_t lane_base = tmem + ((uint32_t)(wq * 32) << 16) + (uint32_t)c_off;
        const float sl2 = p.scale_log2;
        float* s_ref_w = s_ref + c_off;
        float* s_fac_w = s_fac + c_off;
        float* s_dlt_w = s_dlt + c_off;
        float* s_wgt_w = s_wgt + c_off;
        const int* s_rowoff_w = s_rowoff + c_off;
        float* s_warp_w = s_warp + wg * 4 * NW;          // [4 warps][NW] per warpgroup
        const float4* ref4 = reinterpret_cast<const float4*>(s_ref_w);
        const float4* fac4 = reinterpret_cast<const float4*>(s_fac_w);
        float lpart[NW];   // this token lane's share of the running row sums
#pragma unroll
        for (int i = 0; i < NW; ++i) lpart[i] = 0.f;
        int gj = 0;
        while (cur.valid) {
            const Seg& s = cur.s;
            const int sb = gj & 1;
            mbar_wait(bar(kSFull + sb), ((uint32_t)(gj >> 1)) & 1u);
            tc_fence_after();
            if (t == 0 && gj < 20) TS(12 + gj);
            uint32_t xs[NW];
            tmem_ld_cols<NW>(lane_base + kColS + (uint32_t)sb * 128, xs);
            tmem_wait_ld();
            tc_fence_before();
            mbar_arrive(bar(kSEmpty + sb));

            // scale into the log2 domain; mask the tail of the piece, the padding of the new-row tile and, for a new row
            // u, the query rows of verify positions < u (row i belongs to position i / r, so those are the rows i < u * r)
            const int pos = s.pos_lo + cur.ti * kTile + t;
            const int thr = (pos >= s.pos_hi ? INT_MAX : (pos >= kTile ? 0 : (pos < T ? pos * r : INT_MAX))) - c_off;
            // x[i] = d_i = s_i * scale - m_ref[i] (one FFMA), the exponent that P needs; the masks cost nothing in the
            // tiles that have none (cache rows inside the piece: every tile but the last one or two).
            float x[NW];
            bool over = cur.ti == 0;   // the first tile of a piece always moves the reference to its row maxima
            if (__all_sync(0xffffffffu, thr <= 0)) {
#pragma unroll
                for (int i4 = 0; i4 < NW / 4; ++i4) {
                    const float4 m = ref4[i4];
                    x[i4 * 4 + 0] = fmaf(__uint_as_float(xs[i4 * 4 + 0]), sl2, -m.x);
                    x[i4 * 4 + 1] = fmaf(__uint_as_float(xs[i4 * 4 + 1]), sl2, -m.y);
                    x[i4 * 4 + 2] = fmaf(__uint_as_float(xs[i4 * 4 + 2]), sl2, -m.z);
                    x[i4 * 4 + 3] = fmaf(__uint_as_float(xs[i4 * 4 + 3]), sl2, -m.w);
                }
            } else {
#pragma unroll
                for (int i4 = 0; i4 < NW / 4; ++i4) {
                    const float4 m = ref4[i4];
                    const float mm[4] = {m.x, m.y, m.z, m.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int i = i4 * 4 + e;
                        x[i] = i < thr ? -INFINITY : fmaf(__uint_as_float(xs[i]), sl2, -mm[e]);
                    }
                }
            }
            {
                float mx = x[0];   // three-input maxima: half the instructions of one compare per score
#pragma unroll
                for (int i = 1; i + 1 < NW; i += 2) mx = fmaxf(mx, fmaxf(x[i], x[i + 1]));
                mx = fmaxf(mx, x[NW - 1]);
                over |= mx > kRefSlack;
            }
            if (wg_any(over, wg)) {
                // Move the reference exponents to the running row maxima (rare after the first tile).
                {
                    float red[NW];
#pragma unroll
                    for (int i = 0; i < NW; ++i) red[i] = x[i];
                    int rb = 0;
                    tr_reduce<true, NW, 0>(red, lane, rb);
#pragma unroll
                    for (int i = 0; i < TrFinal<NW, 0>::value; ++i) s_warp_w[wq * NW + rb + i] = red[i];
                }
                wg_sync(wg);
                if (t < NW) {
                    const float m_old = s_ref_w[t];
                    const float dmax = fmaxf(fmaxf(s_warp_w[t], s_warp_w[NW + t]), fmaxf(s_warp_w[2 * NW + t], s_warp_w[3 * NW + t]));
                    // first tile: the reference becomes the row maximum itself (nothing has been accumulated yet, so no
                    // factor); later: it only ever rises
                    const float m_new = cur.ti == 0 ? fmaxf(m_old + dmax, kRefFloor) : m_old + fmaxf(dmax, 0.f);
                    s_dlt_w[t] = m_old - m_new;
                    s_fac_w[t] = cur.ti == 0 ? 1.f : exp2f(m_old - m_new);
                    s_ref_w[t] = m_new;
                }
                wg_sync(wg);
                {
                    const float4* dlt4 = reinterpret_cast<const float4*>(s_dlt_w);
#pragma unroll
                    for (int i4 = 0; i4 < NW / 4; ++i4) {
                        const float4 d = dlt4[i4];
                        x[i4 * 4 + 0] += d.x;
                        x[i4 * 4 + 1] += d.y;
                        x[i4 * 4 + 2] += d.z;
                        x[i4 * 4 + 3] += d.w;
                    }
                }
#pragma unroll
                for (int i4 = 0; i4 < NW / 4; ++i4) {
                    const float4 f = fac4[i4];
                    lpart[i4 * 4 + 0] *= f.x;
                    lpart[i4 * 4 + 1] *= f.y;
                    lpart[i4 * 4 + 2] *= f.z;
                    lpart[i4 * 4 + 3] *= f.w;
                }
                if (cur.ti > 0) {   // O^T already holds earlier tiles of this piece: rescale it column by column
                    mbar_wait(bar(kPvDone), (uint32_t)(gj - 1) & 1u);
                    tc_fence_after();
#pragma unroll
                    for (int c = 0; c < NW / 16; ++c) {
                        uint32_t o[16];
                        tmem_ld16(lane_base + kColO + (uint32_t)c * 16, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 16; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * s_fac_w[c * 16 + e]);
                        tmem_st16(lane_base + kColO + (uint32_t)c * 16, o);
                    }
                    if constexpr (NW % 16 != 0) {
                        constexpr int c8 = (NW / 16) * 16;
                        uint32_t o[8];
                        tmem_ld8(lane_base + kColO + (uint32_t)c8, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 8; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * s_fac_w[c8 + e]);
                        tmem_st8(lane_base + kColO + (uint32_t)c8, o);
                    }
                    tmem_wait_st();
                    tc_fence_before();
                }
            }

            // P^T: this token's NW weights, bf16, row-contiguous -> 16-byte stores at [8-row block][token]
            if (gj > 0) mbar_wait(bar(kPvDone), (uint32_t)(gj - 1) & 1u);   // the previous P.V has read the buffer
            unsigned char* prow = smem + C::kOffP + (c_off / 8) * 2048 + t * 16;
#pragma unroll
            for (int jb = 0; jb < NW / 8; ++jb) {
                float pr[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    pr[e] = fast_exp2(x[jb * 8 + e]);
                    lpart[jb * 8 + e] += pr[e];
                }
                *reinterpret_cast<uint4*>(prow + jb * 2048) = make_uint4(pack_bf16(pr[0], pr[1]), pack_bf16(pr[2], pr[3]),
                                                                         pack_bf16(pr[4], pr[5]), pack_bf16(pr[6], pr[7]));
            }
            fence_proxy_async();
            mbar_arrive(bar(kPFull));
            if (t == 0 && gj < 8) TS(40 + gj);

            if (cur.last_tile()) {
                if (t == 0) TS(32 + 4 * (cur.seg_no & 3));
                // ---- the piece is complete ----------------------------------------------------------------------
                // whole unit: normalise, write `out`.  Piece that does not start its unit: leave a normalised partial
                // (o, lse) in the workspace and raise its flag.  Piece that starts a unit cut into several (the head;
                // it runs last in its CTA while the others run first in theirs): pull the other pieces -- normally
                // long finished -- and merge them with this CTA's accumulator, own piece first, then in CTA order.
                const bool merge = s.pos_lo == 0 && !s.whole;
                const int nseg = s.cta_last - s.cta_first + 1;
                const long long slot_id = (long long)rid * 2 + s.slot;
                float v1[NW];
                float lse1 = -INFINITY;
                if (merge) {   // second piece = slot 0 of the next CTA: loads in flight during the reductions below
                    const long long sid1 = (long long)(s.cta_first + 1) * 2;
                    wait_flag(ws.flags + sid1);
                    const float* src1 = ws.part_o + sid1 * NQ * kD + c_off * kD + t;
#pragma unroll
                    for (int i = 0; i < NW; ++i) v1[i] = __ldcg(src1 + i * kD);
                    if (t < rows_w) lse1 = __ldcg(ws.part_lse + sid1 * NQ + c_off + t);
                }
                if (t == 0) TS(56);
                {
                    int rb = 0;
                    tr_reduce<false, NW, 0>(lpart, lane, rb);
#pragma unroll
                    for (int i = 0; i < TrFinal<NW, 0>::value; ++i) s_warp_w[wq * NW + rb + i] = lpart[i];
#pragma unroll
                    for (int i = 0; i < NW; ++i) lpart[i] = 0.f;
                }
                wg_sync(wg);
                float M_row = 0.f, W_row = 0.f;   // thread t < rows: merged maximum and weight sum of row t
                if (t < NW) {
                    const float l = (s_warp_w[t] + s_warp_w[NW + t]) + (s_warp_w[2 * NW + t] + s_warp_w[3 * NW + t]);
                    const float lse_own = l > 0.f ? s_ref_w[t] + log2f(l) : -INFINITY;
                    float scale = l > 0.f ? 1.f / l : 0.f, lse_fin = lse_own;
                    if (merge && t < rows_w) {
                        float M = fmaxf(lse_own, lse1);
                        for (int j = 2; j < nseg; ++j) {
                            const long long sid = (long long)(s.cta_first + j) * 2;
                            wait_flag(ws.flags + sid);
                            M = fmaxf(M, __ldcg(ws.part_lse + sid * NQ + c_off + t));
                        }
                        const float e0 = lse_own == -INFINITY ? 0.f : exp2f(lse_own - M);
                        const float e1 = lse1 == -INFINITY ? 0.f : exp2f(lse1 - M);
                        float W = e0 + e1;
                        for (int j = 2; j < nseg; ++j) {
                            const float lj = __ldcg(ws.part_lse + ((long long)(s.cta_first + j) * 2) * NQ + c_off + t);
                            W += lj == -INFINITY ? 0.f : exp2f(lj - M);
                        }
                        const float invW = W > 0.f ? 1.f / W : 0.f;
                        scale *= e0 * invW;
                        s_wgt_w[t] = e1 * invW;
                        lse_fin = W > 0.f ? M + log2f(W) : -INFINITY;
                        M_row = M;
                        W_row = invW;
                    }
                    s_fac_w[t] = scale;
                    if (t < rows_w) {
                        if (s.pos_lo != 0) ws.part_lse[slot_id * NQ + c_off + t] = lse_own;
                        else if (p.lse_out)
                            p.lse_out[((long long)s.b * Hq + s.g * r + (c_off + t) % r) * T + (c_off + t) / r] = lse_fin * kLn2;
                    }
                }
                if (t == 0) TS(54);
                mbar_wait(bar(kPvDone), (uint32_t)gj & 1u);   // every P.V of the piece has completed
                tc_fence_after();
                if (t == 0) TS(55);
                uint32_t o[NW];
                tmem_ld_cols<NW>(lane_base + kColO, o);
                tmem_wait_ld();
                tc_fence_before();
                sm_sync<NWG>();
                if (merge && t == 0 && wg == 0)   // every thread is past its flag waits: leave the flags zero for the next launch
                    for (int j = 1; j < nseg; ++j) ws.flags[(long long)(s.cta_first + j) * 2] = 0;
                if (t == 0) TS(33 + 4 * (cur.seg_no & 3));
                if (s.pos_lo != 0) {
                    float* po = ws.part_o + slot_id * NQ * kD + c_off * kD + t;   // padded to NW rows: no predicate
#pragma unroll
                    for (int i = 0; i < NW; ++i) po[i * kD] = __uint_as_float(o[i]) * s_fac_w[i];
                    // publish: the barrier orders the stores of both warpgroups before thread 0's fence and flag
                    sm_sync<NWG>();
                    if (t == 0 && wg == 0) {
                        __threadfence();
                        st_release(ws.flags + slot_id, 1);
                    }
                } else {
                    float acc[NW];
#pragma unroll
                    for (int i = 0; i < NW; ++i) acc[i] = __uint_as_float(o[i]) * s_fac_w[i];
                    if (merge) {
#pragma unroll
                        for (int i = 0; i < NW; ++i) acc[i] = fmaf(s_wgt_w[i], v1[i], acc[i]);
                        for (int j = 2; j < nseg; ++j) {   // units cut into more than two pieces (very long sequences)
                            const long long sid = (long long)(s.cta_first + j) * 2;
                            wg_sync(wg);
                            if (t < rows_w) {
                                const float lj = __ldcg(ws.part_lse + sid * NQ + c_off + t);
                                s_wgt_w[t] = lj == -INFINITY ? 0.f : exp2f(lj - M_row) * W_row;
                            }
                            const float* src = ws.part_o + sid * NQ * kD + c_off * kD + t;
#pragma unroll
                            for (int i = 0; i < NW; ++i) v1[i] = __ldcg(src + i * kD);
                            wg_sync(wg);
#pragma unroll
                            for (int i = 0; i < NW; ++i) acc[i] = fmaf(s_wgt_w[i], v1[i], acc[i]);
                        }
                    }
                    if (t == 0) TS(53);
                    // bf16 rows staged in the P buffer (idle: every P.V of the piece has completed), then written
                    // with 16-byte stores: row x / 16, chunk x % 16
                    __nv_bfloat16* so = reinterpret_cast<__nv_bfloat16*>(smem + C::kOffP) + c_off * kD;
#pragma unroll
                    for (int i = 0; i < NW; ++i) so[i * kD + t] = __float2bfloat16_rn(acc[i]);
                    wg_sync(wg);
                    __nv_bfloat16* ob = p.out + ((long long)s.b * T * Hq + (long long)s.g * r) * kD;
#pragma unroll 1
                    for (int x = t; x < rows_w * 16; x += 128) {
                        const int rr = x >> 4, cc = x & 15;
                        *reinterpret_cast<uint4*>(ob + s_rowoff_w[rr] + cc * 8) =
                            *reinterpret_cast<const uint4*>(so + rr * kD + cc * 8);
                    }
                }
                if (t == 0) TS(34 + 4 * (cur.seg_no & 3));
                if (t == 0) TS(35 + 4 * (cur.seg_no & 3));
                wg_sync(wg);
                if (t < NW) s_ref_w[t] = kRefInit;
                wg_sync(wg);
            }
            cur.advance();
            ++gj;
        }
    }

    if (p.dbg & 64) pdl_trigger();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) TS(3);
    if ((p.dbg & 8) && ws.dbg_ts) {
        __syncthreads();
        if (tid < 62) ws.dbg_ts[(size_t)blockIdx.x * 64 + tid] = s_ts[tid];
        if (tid == 62) ws.dbg_ts[(size_t)blockIdx.x * 64 + 62] = gtimer();   // end of the CTA (slot 63: its start)
    }
    if (warp == 8) {
        tc_fence_after();
        tmem_dealloc(tmem, 512);
    }
}

constexpr int kMaxGrid = 256;   // workspace is sized for this many CTAs

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

template <int NQ, int NWG, bool GATHER>
cudaError_t launch_tc(const AttnParams& p, const TcWs& ws, int grid, cudaStream_t stream) {
    using C = TcCfg<NQ>;
    constexpr int smem = C::kSmemBytes;
    static DeviceOnce once;   // per instantiation
    {
        const cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(attn_tc_kernel<NQ, NWG, GATHER>), smem, once);
        if (e != cudaSuccess) return e;
    }
    ProfScope prof(kKernAttn, stream);
    return launch_pdl(attn_tc_kernel<NQ, NWG, GATHER>, dim3(grid), dim3(kTcThreads + 128 * (NWG - 1)), smem, stream, p, ws);
}

template <int NQ, int NWG = 1>
cudaError_t launch_tc_nq(const AttnParams& p, const TcWs& ws, int grid, cudaStream_t stream) {
    return p.idx ? launch_tc<NQ, NWG, true>(p, ws, grid, stream) : launch_tc<NQ, NWG, false>(p, ws, grid, stream);
}

}  // namespace

bool attn_tc_usable(int batch, int n_kv_heads, int head_dim, int rows, int max_tokens, int n_new) {
    if (head_dim != kD || rows > 96 || rows < 1) return false;
    const long long units = (long long)batch * n_kv_heads;
    if (units > kMaxUnits) return false;
    (void)n_new;   // the new rows of a unit take one whole tile of its token space
    return units * ((long long)max_tokens + kTile) < (1ll << 31) - (1 << 20);
}

size_t attn_tc_ws_bytes(int batch, int n_kv_heads, int rows) {
    static_assert(kMaxGrid * 2 * sizeof(int) <= kWsHeader, "the flags must fit the persistent header");
    const size_t nq = (size_t)((rows + 15) / 16) * 16;   // partials are padded to the kernel's NQ rows
    return kWsHeader + align256((size_t)kMaxGrid * 2 * nq * kD * sizeof(float)) +
           align256((size_t)kMaxGrid * 2 * nq * sizeof(float)) + (size_t)kMaxGrid * 64 * 8;
}

cudaError_t launch_attn_tc(const AttnParams& p_in, void* ws_base, cudaStream_t stream) {
    AttnParams p = p_in;
    p.dbg = knob(DUSTIN_KNOB_ATTN_TRACE);
    const size_t units = (size_t)p.batch * p.n_kv_heads;
    char* base = static_cast<char*>(ws_base);
    (void)stream;
    TcWs ws;
    // Persistent header (kernels.cuh kWsHeader): the flags.  Zero before the first use
    // (dustin.h); every launch leaves it zero again (the merging piece clears the flags it has consumed).
    ws.flags = reinterpret_cast<int*>(base);
    ws.part_o = reinterpret_cast<float*>(base + kWsHeader);
    const size_t nq = (size_t)((p.rows + 15) / 16) * 16;
    ws.part_lse = reinterpret_cast<float*>(base + kWsHeader + align256((size_t)kMaxGrid * 2 * nq * kD * sizeof(float)));
    ws.dbg_ts = (p.dbg & 8) ? reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(ws.part_lse) + align256((size_t)kMaxGrid * 2 * nq * sizeof(float))) : nullptr;
    const int max_tokens = (p.idx ? (p.k_max < p.max_ctx ? p.k_max : p.max_ctx) : p.max_ctx) + kTile;
    long long tiles = ((long long)units * max_tokens + kTile - 1) / kTile;
    const int sms = device_sm_count();
    int grid = sms < kMaxGrid ? sms : kMaxGrid;
    if (tiles < grid) grid = tiles < 1 ? 1 : (int)tiles;
    switch ((p.rows + 15) / 16) {
        case 1: return launch_tc_nq<16>(p, ws, grid, stream);
        case 2: return launch_tc_nq<32>(p, ws, grid, stream);
        case 3: return launch_tc_nq<48>(p, ws, grid, stream);
        // more than 48 query rows: padded to a multiple of 16, one softmax warpgroup per half (a single warpgroup needs
        // 2.3 us per tile for 80 rows and bounds the kernel; two need about half)
        case 4: return launch_tc_nq<64, 2>(p, ws, grid, stream);
        case 5: return launch_tc_nq<80, 2>(p, ws, grid, stream);   // Gamma = 8 on an 8-head group: 72 rows, 40 + 32
        case 6: return launch_tc_nq<96, 2>(p, ws, grid, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace dustin
