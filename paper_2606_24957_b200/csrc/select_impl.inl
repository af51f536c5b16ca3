// select_impl.inl -- device code of stage a3, included by select.cu once per CTA size (SEL_NT threads) inside a
// namespace of its own.  See select.cu for the description of the algorithm.

constexpr int kSelThreads = SEL_NT;   // threads per CTA: set by the including file (select.cu)
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kBins = 2048;
constexpr int kBinsPerThread = kBins / kSelThreads;

__device__ __forceinline__ uint32_t key_of(float s) { return s > 0.f ? __float_as_uint(s) : 0u; }

// DUSTIN_KNOB_SELECT_TRACE: thread 0 of every CTA samples %globaltimer at the phase boundaries.
__device__ __forceinline__ void sel_ts(unsigned long long* row, int slot) {
    if (row != nullptr && threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
        row[slot] = t;
    }
}

// Threshold bins of at most this many entries are ranked by brute force (list_select_ranged); fuller ones cost another
// histogram pass (two more block-wide barriers), which showed as the slow tail of the kernel at 32.
constexpr int kSmallList = 128;

struct SelShared {
    uint32_t hist[kBins];
    uint32_t warp_tot[kSelWarps + 1];
    uint32_t res_bin, res_rank, res_cnt;
    uint32_t list_n, res_total;
    // scratch of the sampled path: two copies used alternately (parity of a per-thread phase counter), so one barrier
    // between a write and its reads is enough
    uint32_t tot_db[2][kSelWarps], min_db[2][kSelWarps], max_db[2][kSelWarps], res_db[2][4];
    uint32_t small_n, small_key[kSmallList], small_idx[kSmallList];
    float2 stats[64];   // (M, 1/Z) of the heads feeding this row (row materialisation)
    unsigned long long* trace;   // this CTA's 64 timestamp slots, or nullptr (read and written by thread 0 only)
    int trace_base;              // first slot of the tier in progress
};

// Exclusive prefix of v over the block in thread order; *total (optional) receives the block sum.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, SelShared& sh, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += o;
    }
    __syncthreads();   // protects warp_tot against the previous use
    // The warp total travels to lane 0 before it is stored.  (Storing from lane 31 miscompiles with nvcc 12.9 in the 256-
    // and 512-thread instantiations: the address is formed as base + (tid >> 3), which is only warp * 4 when lane == 0.)
    const uint32_t wtot = __shfl_sync(0xffffffffu, inc, 31);
    if (lane == 0) sh.warp_tot[warp] = wtot;
    __syncthreads();
    const uint32_t t = lane < kSelWarps ? sh.warp_tot[lane] : 0u;   // every warp scans the warp totals redundantly
    uint32_t ti = t;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, ti, off);
        if (lane >= off) ti += o;
    }
    if (total) *total = __shfl_sync(0xffffffffu, ti, 31);
    return __shfl_sync(0xffffffffu, ti - t, warp) + inc - v;
}

// Test hook (dustin_debug_block_scan, dustin_debug.h): block_excl_scan on its own, twice in a row on different values
// (the second use must not see the first one's warp totals).  in: [gridDim.x][kSelThreads];  out: [2][gridDim.x][kSelThreads]
// exclusive prefixes of in and of in + 1;  total: [2][gridDim.x].
__global__ void __launch_bounds__(kSelThreads) scan_test_kernel(const uint32_t* __restrict__ in, uint32_t* __restrict__ out,
                                                                uint32_t* __restrict__ total) {
    __shared__ SelShared sh;
    const size_t i = (size_t)blockIdx.x * kSelThreads + threadIdx.x, n = (size_t)gridDim.x * kSelThreads;
    const uint32_t v = in[i];
    uint32_t t0, t1;
    out[i] = block_excl_scan(v, sh, &t0);
    out[n + i] = block_excl_scan(v + 1u, sh, &t1);
    if (threadIdx.x == kSelThreads - 1) {
        total[blockIdx.x] = t0;
        total[gridDim.x + blockIdx.x] = t1;
    }
}

// Key of descending rank `rank` (1-based) among the candidates n in [lo, hi) whose bit in `mem` is clear.
// Returns the key; need_eq = how many candidates equal to it must still be admitted (in index order);
// eq_total = how many candidates carry exactly that key.
__device__ uint32_t radix_select(const float* __restrict__ s, int lo, int hi, const uint32_t* mem, int rank,
                                 SelShared& sh, int& need_eq, int& eq_total) {
    uint32_t prefix = 0;
    const int shifts[3] = {21, 10, 0};
    const int widths[3] = {11, 11, 10};
#pragma unroll
    for (int pass = 0; pass < 3; ++pass) {
        const int shift = shifts[pass], nb = 1 << widths[pass];
        for (int i = threadIdx.x; i < kBins; i += kSelThreads) sh.hist[i] = 0;
        __syncthreads();
        const int hs = shift + widths[pass];   // bits above the digit
        for (int n = lo + threadIdx.x; n < hi; n += kSelThreads) {
            if ((mem[n >> 5] >> (n & 31)) & 1u) continue;
            const uint32_t key = key_of(__ldcg(s + n));
            if (pass > 0 && (key >> hs) != (prefix >> hs)) continue;
            const uint32_t digit = (key >> shift) & (nb - 1);
            atomicAdd(&sh.hist[nb - 1 - digit], 1u);   // reversed: bin 0 holds the largest digit
        }
        __syncthreads();
        uint32_t cb[kBinsPerThread], mine = 0;   // this thread's consecutive bins
#pragma unroll
        for (int i = 0; i < kBinsPerThread; ++i) {
            cb[i] = sh.hist[kBinsPerThread * threadIdx.x + i];
            mine += cb[i];
        }
        uint32_t run = block_excl_scan(mine, sh, nullptr);
        const uint32_t r = (uint32_t)rank;
#pragma unroll
        for (int i = 0; i < kBinsPerThread; ++i) {
            if (run < r && r <= run + cb[i]) {
                sh.res_bin = kBinsPerThread * threadIdx.x + i;
                sh.res_rank = r - run;
                sh.res_cnt = cb[i];
            }
            run += cb[i];
        }
        __syncthreads();
        prefix |= (uint32_t)(nb - 1 - sh.res_bin) << shift;
        rank = (int)sh.res_rank;
        eq_total = (int)sh.res_cnt;
        __syncthreads();
    }
    need_eq = rank;
    return prefix;
}

// Admit into `mem` every candidate with key > T and the first need_eq candidates (index order) with key == T.
__device__ void admit_tier(const float* __restrict__ s, int lo, int hi, uint32_t* mem, int n_words, uint32_t T,
                           int need_eq, int eq_total, SelShared& sh) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wpw = (n_words + kSelWarps - 1) / kSelWarps;
    const int w_lo = warp * wpw, w_hi = min(w_lo + wpw, n_words);
    uint32_t eq_before = 0;
    const bool ranked = need_eq < eq_total;   // otherwise every equal key is admitted and no order is needed
    if (ranked) {
        uint32_t mine = 0;
        for (int w = w_lo; w < w_hi; ++w) {
            const int n = w * 32 + lane;
            const bool cand = n >= lo && n < hi && !((mem[w] >> lane) & 1u);
            const bool eq = cand && key_of(__ldcg(s + n)) == T;
            mine += __popc(__ballot_sync(0xffffffffu, eq));
        }
        __syncthreads();
        if (lane == 0) sh.warp_tot[warp] = mine;
        __syncthreads();
        for (int w = 0; w < warp; ++w) eq_before += sh.warp_tot[w];
        __syncthreads();
    }
    for (int w = w_lo; w < w_hi; ++w) {
        const int n = w * 32 + lane;
        const uint32_t old = mem[w];
        const bool cand = n >= lo && n < hi && !((old >> lane) & 1u);
        const uint32_t key = cand ? key_of(__ldcg(s + n)) : 0u;
        const bool gt = cand && key > T, eq = cand && key == T;
        const uint32_t eqb = __ballot_sync(0xffffffffu, eq);
        bool take = gt;
        if (eq) take = !ranked || (int)(eq_before + __popc(eqb & ((1u << lane) - 1u))) < need_eq;
        const uint32_t add = __ballot_sync(0xffffffffu, take);
        eq_before += __popc(eqb);
        __syncwarp();
        if (lane == 0) mem[w] = old | add;
    }
    __syncthreads();
}

__device__ __noinline__ void full_scan_tier(const float* __restrict__ s, int lo, int hi, uint32_t* mem, int n_words,
                                            int rank, SelShared& sh) {
    int need_eq, eq_total;
    const uint32_t T = radix_select(s, lo, hi, mem, rank, sh, need_eq, eq_total);
    admit_tier(s, lo, hi, mem, n_words, T, need_eq, eq_total, sh);
}

// ---- fast path --------------------------------------------------------------------------------------------------
// One full scan builds the histogram of the top 11 key bits (R lane-interleaved replicas keep same-address shared
// atomics apart); a second full scan admits everything above the threshold bin and compacts the threshold bin
// itself into a short (key, index) list in shared memory; the remaining 21 key bits -- and, when equal keys
// straddle the threshold, the index order among them -- are resolved on that list alone.  A threshold bin that
// does not fit the list (massive ties) takes the full-scan path above instead.
struct SelLayout {
    uint32_t* mem;        // membership bitmask
    uint32_t* hist;       // kBins * R counters
    uint32_t* list_key;   // cap
    uint32_t* list_idx;   // cap
    int R, cap;
};

// Key of a score: the uint32 image of max(s, 0) (order-preserving for s >= 0; negatives and -0 tie at 0).
__device__ __forceinline__ uint32_t key_max0(float s) { return __float_as_uint(fmaxf(s, 0.f)); }

// Scan 1: histogram of the top 11 key bits over the candidates.  A candidate is an index of [lo, hi) whose bit in
// `mem` is clear; every non-candidate index that a 16-byte load can touch (sink, window, tail of the last word)
// has its bit set, so the bitmask alone decides.  hist_rep = hist + replica; bin 0 holds the largest keys.
template <bool VEC>
__device__ __forceinline__ void scan_hist(const float* __restrict__ s, int lo, int hi, const uint32_t* mem,
                                          uint32_t* hist_rep, int R) {
    uint32_t* top = hist_rep + (size_t)(kBins - 1) * R;
    if (VEC) {
        const float4* s4 = reinterpret_cast<const float4*>(s);
        const int v_end = (hi + 3) >> 2;
        for (int v = (lo >> 2) + threadIdx.x; v < v_end; v += 4 * kSelThreads) {
            float4 x[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int vv = v + u * kSelThreads;
                x[u] = vv < v_end ? __ldcg(s4 + vv) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int n = (v + u * kSelThreads) << 2;
                const uint32_t nib = n < hi ? mem[n >> 5] >> (n & 31) : 0xfu;
                if (!(nib & 1u)) atomicAdd(top - (key_max0(x[u].x) >> 21) * R, 1u);
                if (!(nib & 2u)) atomicAdd(top - (key_max0(x[u].y) >> 21) * R, 1u);
                if (!(nib & 4u)) atomicAdd(top - (key_max0(x[u].z) >> 21) * R, 1u);
                if (!(nib & 8u)) atomicAdd(top - (key_max0(x[u].w) >> 21) * R, 1u);
            }
        }
    } else {
        for (int n = lo + threadIdx.x; n < hi; n += kSelThreads)
            if (!((mem[n >> 5] >> (n & 31)) & 1u)) atomicAdd(top - (key_max0(__ldcg(s + n)) >> 21) * R, 1u);
    }
}

// Scan 2: candidates whose top key bits exceed t1 are admitted (their bits set in mem); those equal to t1 are
// appended, in any order, to the (key, index) list.
struct ListAppender {
    uint32_t* key;
    uint32_t* idx;
    uint32_t* count;
    uint32_t cap;   // entries beyond cap are counted but not stored (the caller then takes another path)
    // One lane, any time (divergent callers): lanes that arrive together share one counter update.
    __device__ __forceinline__ void operator()(uint32_t k, int i) const {
        const uint32_t peers = __activemask();   // lanes appending together (any subset is correct)
        const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if (lane == leader) base = atomicAdd(count, (uint32_t)__popc(peers));
        base = __shfl_sync(peers, base, leader);
        const uint32_t pos = base + __popc(peers & ((1u << lane) - 1u));
        if (pos < cap) {
            key[pos] = k;
            idx[pos] = (uint32_t)i;
        }
    }
    // Whole warp, converged: lane holds 4 consecutive elements n..n+3, bit e of `hit` says element e is appended.
    // One shared-memory counter update per warp call (only when some lane has a hit).
    __device__ __forceinline__ void warp4(uint32_t hit, uint32_t k0, uint32_t k1, uint32_t k2, uint32_t k3,
                                          int n) const {
        const int lane = threadIdx.x & 31;
        const uint32_t mine = __popc(hit & 0xfu);
        if (!__any_sync(0xffffffffu, mine != 0)) return;
        uint32_t inc = mine;   // inclusive prefix of the per-lane counts
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t o = __shfl_up_sync(0xffffffffu, inc, off);
            if (lane >= off) inc += o;
        }
        uint32_t base = 0;
        if (lane == 31) base = atomicAdd(count, inc);
        base = __shfl_sync(0xffffffffu, base, 31);
        uint32_t pos = base + inc - mine;
        if (hit & 1u) { if (pos < cap) { key[pos] = k0; idx[pos] = (uint32_t)n; } ++pos; }
        if (hit & 2u) { if (pos < cap) { key[pos] = k1; idx[pos] = (uint32_t)(n + 1); } ++pos; }
        if (hit & 4u) { if (pos < cap) { key[pos] = k2; idx[pos] = (uint32_t)(n + 2); } ++pos; }
        if (hit & 8u) { if (pos < cap) { key[pos] = k3; idx[pos] = (uint32_t)(n + 3); } ++pos; }
    }
};

template <bool VEC>
__device__ __forceinline__ void scan_admit(const float* __restrict__ s, int lo, int hi, uint32_t* mem, uint32_t t1,
                                           const ListAppender& app) {
    if (VEC) {
        const float4* s4 = reinterpret_cast<const float4*>(s);
        const int v_end = (hi + 3) >> 2;
        // warp-uniform trip count: the list append below needs the whole warp converged
        for (int vb = (lo >> 2) + (threadIdx.x & ~31); vb < v_end; vb += 4 * kSelThreads) {
            const int v = vb + (threadIdx.x & 31);
            float4 x[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int vv = v + u * kSelThreads;
                x[u] = vv < v_end ? __ldcg(s4 + vv) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int n = (v + u * kSelThreads) << 2;
                const uint32_t nib = n < hi ? mem[n >> 5] >> (n & 31) : 0xfu;
                const uint32_t k0 = key_max0(x[u].x), k1 = key_max0(x[u].y), k2 = key_max0(x[u].z),
                               k3 = key_max0(x[u].w);
                uint32_t add = 0;
                add |= ((k0 >> 21) > t1) ? 1u : 0u;
                add |= ((k1 >> 21) > t1) ? 2u : 0u;
                add |= ((k2 >> 21) > t1) ? 4u : 0u;
                add |= ((k3 >> 21) > t1) ? 8u : 0u;
                add &= ~nib;
                if (add) atomicOr(&mem[n >> 5], add << (n & 31));
                uint32_t eq = 0;
                eq |= ((k0 >> 21) == t1) ? 1u : 0u;
                eq |= ((k1 >> 21) == t1) ? 2u : 0u;
                eq |= ((k2 >> 21) == t1) ? 4u : 0u;
                eq |= ((k3 >> 21) == t1) ? 8u : 0u;
                app.warp4(eq & ~nib, k0, k1, k2, k3, n);
            }
        }
    } else {
        for (int n = lo + threadIdx.x; n < hi; n += kSelThreads) {
            if ((mem[n >> 5] >> (n & 31)) & 1u) continue;
            const uint32_t k = key_max0(__ldcg(s + n));
            if ((k >> 21) > t1) atomicOr(&mem[n >> 5], 1u << (n & 31));
            if ((k >> 21) == t1) app(k, n);
        }
    }
}

// hist layout: [bin][R] (the R replicas of a bin are contiguous); kBins * R words, 16-byte aligned.
__device__ __forceinline__ void clear_hist(uint32_t* hist, int R) {
    uint4* h4 = reinterpret_cast<uint4*>(hist);
    for (int i = threadIdx.x; i < kBins * R / 4; i += kSelThreads) h4[i] = make_uint4(0, 0, 0, 0);
}

// Bin holding rank `rank` (1-based, bins in ascending bin order); leaves (bin, rank inside the bin, bin count)
// in sh.res_*.  Thread t owns bins 2t and 2t + 1 (2R contiguous words).  R in {1, 4, 8}.  Ends with a barrier.
__device__ __forceinline__ void find_bin(const uint32_t* hist, int R, uint32_t rank, SelShared& sh) {
    uint32_t cb[kBinsPerThread], mine = 0;   // this thread's consecutive bins, summed over the R replicas
#pragma unroll
    for (int i = 0; i < kBinsPerThread; ++i) {
        const uint32_t* h = hist + (size_t)(kBinsPerThread * threadIdx.x + i) * R;
        uint32_t c = 0;
        if (R == 1) {
            c = h[0];
        } else {
            const uint4* h4 = reinterpret_cast<const uint4*>(h);
            for (int r = 0; r < R / 4; ++r) {
                const uint4 a = h4[r];
                c += a.x + a.y + a.z + a.w;
            }
        }
        cb[i] = c;
        mine += c;
    }
    uint32_t total;
    uint32_t run = block_excl_scan(mine, sh, &total);
    if (threadIdx.x == 0) sh.res_total = total;
#pragma unroll
    for (int i = 0; i < kBinsPerThread; ++i) {
        if (run < rank && rank <= run + cb[i]) {
            sh.res_bin = kBinsPerThread * threadIdx.x + i;
            sh.res_rank = rank - run;
            sh.res_cnt = cb[i];
        }
        run += cb[i];
    }
    __syncthreads();
}

__device__ __forceinline__ void set_member(uint32_t* mem, int idx) { atomicOr(&mem[idx >> 5], 1u << (idx & 31)); }

// Scan of the sampled path: every candidate whose top 11 key bits are >= tau_top is appended to the list.
template <bool VEC>
__device__ __forceinline__ void scan_collect(const float* __restrict__ s, int lo, int hi, const uint32_t* mem,
                                             uint32_t tau_top, const ListAppender& app) {
    if (VEC) {
        const float4* s4 = reinterpret_cast<const float4*>(s);
        const int v_end = (hi + 3) >> 2;
        // warp-uniform trip count: the list append below needs the whole warp converged
        for (int vb = (lo >> 2) + (threadIdx.x & ~31); vb < v_end; vb += 4 * kSelThreads) {
            const int v = vb + (threadIdx.x & 31);
            float4 x[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int vv = v + u * kSelThreads;
                x[u] = vv < v_end ? __ldcg(s4 + vv) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int n = (v + u * kSelThreads) << 2;
                const uint32_t k0 = key_max0(x[u].x), k1 = key_max0(x[u].y), k2 = key_max0(x[u].z),
                               k3 = key_max0(x[u].w);
                uint32_t hit = 0;
                hit |= ((k0 >> 21) >= tau_top) ? 1u : 0u;
                hit |= ((k1 >> 21) >= tau_top) ? 2u : 0u;
                hit |= ((k2 >> 21) >= tau_top) ? 4u : 0u;
                hit |= ((k3 >> 21) >= tau_top) ? 8u : 0u;
                if (hit) hit &= n < hi ? ~(mem[n >> 5] >> (n & 31)) : 0u;
                app.warp4(hit, k0, k1, k2, k3, n);
            }
        }
    } else {
        for (int n = lo + threadIdx.x; n < hi; n += kSelThreads) {
            const uint32_t k = key_max0(__ldcg(s + n));
            if ((k >> 21) >= tau_top && !((mem[n >> 5] >> (n & 31)) & 1u)) app(k, n);
        }
    }
}

// Exact selection on the candidate list: admits the `rank` best of the n_list entries (key descending, ties toward
// the lower index).  first_pass = 0: all 32 key bits are resolved here; 1: the entries share their top 11 bits.
__device__ void list_select(const SelLayout& L, int n_list, uint32_t rank, int first_pass, uint32_t prefix,
                            SelShared& sh) {
    uint32_t* hist = L.hist;
    uint32_t eq_total = 0;
#pragma unroll 1
    for (int pass = first_pass; pass < 3; ++pass) {
        const int shift = pass == 0 ? 21 : (pass == 1 ? 10 : 0);
        const uint32_t nb = pass == 2 ? 1024u : 2048u;
        const int hs = pass == 1 ? 21 : 10;   // bits above the digit (pass 0 has none)
        clear_hist(hist, 1);
        __syncthreads();
        for (int j = threadIdx.x; j < n_list; j += kSelThreads) {
            const uint32_t key = L.list_key[j];
            if (pass == 0 || (key >> hs) == (prefix >> hs)) atomicAdd(&hist[nb - 1 - ((key >> shift) & (nb - 1))], 1u);
        }
        __syncthreads();
        find_bin(hist, 1, rank, sh);
        prefix |= (nb - 1 - sh.res_bin) << shift;
        rank = sh.res_rank;
        eq_total = sh.res_cnt;
        __syncthreads();
    }
    const uint32_t T = prefix, need_eq = rank;
    if (need_eq == eq_total) {   // every key equal to T is admitted: no order needed
        for (int j = threadIdx.x; j < n_list; j += kSelThreads)
            if (L.list_key[j] >= T) set_member(L.mem, (int)L.list_idx[j]);
        __syncthreads();
        return;
    }
    // Equal keys straddle the threshold: admit the need_eq lowest indices among them (indices < 2^20).
    clear_hist(hist, 1);
    __syncthreads();
    for (int j = threadIdx.x; j < n_list; j += kSelThreads) {
        const uint32_t key = L.list_key[j];
        if (key > T) set_member(L.mem, (int)L.list_idx[j]);
        if (key == T) atomicAdd(&hist[L.list_idx[j] >> 10], 1u);
    }
    __syncthreads();
    find_bin(hist, 1, need_eq, sh);
    const uint32_t i_hi = sh.res_bin, rank_lo = sh.res_rank;
    __syncthreads();
    clear_hist(hist, 1);
    __syncthreads();
    for (int j = threadIdx.x; j < n_list; j += kSelThreads)
        if (L.list_key[j] == T && (L.list_idx[j] >> 10) == i_hi) atomicAdd(&hist[L.list_idx[j] & 0x3ffu], 1u);
    __syncthreads();
    find_bin(hist, 1, rank_lo, sh);
    const uint32_t i_star = (i_hi << 10) | sh.res_bin;
    __syncthreads();
    for (int j = threadIdx.x; j < n_list; j += kSelThreads)
        if (L.list_key[j] == T && L.list_idx[j] <= i_star) set_member(L.mem, (int)L.list_idx[j]);
    __syncthreads();
}

// ---- building blocks of the sampled path: one barrier each (double-buffered scratch, use counters in `ph`) ----------
struct Phase {
    int scan = 0, mm = 0, res = 0;   // uses so far of tot_db / min_db+max_db / res_db (block-uniform)
};
// Block-wide minimum of `tmin` and maximum of `tmax` over the threads with `valid` set (kmin > kmax when none is).
__device__ __forceinline__ void block_minmax(uint32_t tmin, uint32_t tmax, bool valid, SelShared& sh, Phase& ph,
                                             uint32_t& kmin, uint32_t& kmax) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, b = ph.mm++ & 1;
    const uint32_t lo = __reduce_min_sync(0xffffffffu, valid ? tmin : 0xffffffffu);
    const uint32_t hi = __reduce_max_sync(0xffffffffu, valid ? tmax : 0u);
    if (lane == 0) {
        sh.min_db[b][warp] = lo;
        sh.max_db[b][warp] = hi;
    }
    __syncthreads();
    kmin = __reduce_min_sync(0xffffffffu, lane < kSelWarps ? sh.min_db[b][lane] : 0xffffffffu);
    kmax = __reduce_max_sync(0xffffffffu, lane < kSelWarps ? sh.max_db[b][lane] : 0u);
}

// Exclusive prefix of v over the block in thread order; *total receives the block sum.
__device__ __forceinline__ uint32_t block_excl_scan_db(uint32_t v, SelShared& sh, Phase& ph, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, b = ph.scan++ & 1;
    uint32_t inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += o;
    }
    const uint32_t wtot = __shfl_sync(0xffffffffu, inc, 31);   // stored from lane 0: see block_excl_scan
    if (lane == 0) sh.tot_db[b][warp] = wtot;
    __syncthreads();
    const uint32_t t = lane < kSelWarps ? sh.tot_db[b][lane] : 0u;   // every warp scans the warp totals redundantly
    uint32_t ti = t;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, ti, off);
        if (lane >= off) ti += o;
    }
    *total = __shfl_sync(0xffffffffu, ti, 31);
    return __shfl_sync(0xffffffffu, ti - t, warp) + inc - v;
}

// Bin of the single-replica histogram that holds rank `rank` (1-based, ascending bin order).  Leaves the histogram
// ZEROED for its next use.  Returns {bin, rank inside the bin, bin count, total}; bin is valid when rank <= total.
__device__ __forceinline__ uint4 find_bin_db(uint32_t* hist, uint32_t rank, SelShared& sh, Phase& ph) {
    uint32_t cb[kBinsPerThread], mine = 0;
#pragma unroll
    for (int i = 0; i < kBinsPerThread; ++i) {
        cb[i] = hist[kBinsPerThread * threadIdx.x + i];
        mine += cb[i];
    }
    uint32_t total;
    uint32_t run = block_excl_scan_db(mine, sh, ph, &total);
#pragma unroll
    for (int i = 0; i < kBinsPerThread; ++i) hist[kBinsPerThread * threadIdx.x + i] = 0u;   // every thread is past its read
    const int b = ph.res++ & 1;
#pragma unroll
    for (int i = 0; i < kBinsPerThread; ++i) {
        if (run < rank && rank <= run + cb[i]) {
            sh.res_db[b][0] = kBinsPerThread * threadIdx.x + i;
            sh.res_db[b][1] = rank - run;
            sh.res_db[b][2] = cb[i];
        }
        run += cb[i];
    }
    __syncthreads();
    return make_uint4(sh.res_db[b][0], sh.res_db[b][1], sh.res_db[b][2], total);
}

// Digit position that spreads the key range [kmin, kmax] over the kBins bins: bucket = (key - kmin) >> shift.
__device__ __forceinline__ int range_shift(uint32_t kmin, uint32_t kmax) {
    const int bits = kmax > kmin ? 32 - __clz(kmax - kmin) : 0;
    return bits > 11 ? bits - 11 : 0;
}

// Exact selection on the candidate list by an OFFSET radix select: a pass spreads the current key range
// [klo, khi] (first pass: the list's own minimum and maximum) over the 2048 bins, so the scores of one row -- which
// share their leading exponent bits -- do not pile up in a handful of bins (same-address shared atomics serialise).
// A threshold bin of <= kSmallList entries is then ranked by brute force ((key desc, index asc) order, which also settles
// ties); a fuller one becomes the range of the next pass.  Admits the `rank` best of the n_list entries.
template <int kPer>   // entries per thread: n_list <= kPer * kSelThreads
__device__ void list_select_ranged(const float* __restrict__ s, const SelLayout& L, int n_list, uint32_t rank,
                                   SelShared& sh, Phase& ph) {
    // On entry: list_idx[0, n_list) filled, hist (replica 0) all zero, a barrier since both.  Leaves hist zero.
    uint32_t* hist = L.hist;
    uint32_t key[kPer], idx[kPer];
    uint32_t part = 0;        // bit e: entry threadIdx.x + e * kSelThreads is still inside the key range
    uint32_t lmin = 0xffffffffu, lmax = 0u;
#pragma unroll
    for (int e = 0; e < kPer; ++e) {   // the keys come straight from the score row: independent loads, all in flight
        const int j = threadIdx.x + e * kSelThreads;
        idx[e] = j < n_list ? L.list_idx[j] : 0u;
        key[e] = j < n_list ? key_max0(__ldcg(s + idx[e])) : 0u;
    }
#pragma unroll
    for (int e = 0; e < kPer; ++e)
        if (threadIdx.x + e * kSelThreads < n_list) {
            part |= 1u << e;
            lmin = min(lmin, key[e]);
            lmax = max(lmax, key[e]);
        }
    if (threadIdx.x == 0) sh.small_n = 0;
    uint32_t klo, khi;
    block_minmax(lmin, lmax, part != 0, sh, ph, klo, khi);
    if (threadIdx.x == 0) sel_ts(sh.trace, sh.trace_base + 2);   // list keys gathered, range known
    uint32_t eq_total = (uint32_t)n_list;
    uint32_t T = klo, i_star = 0xffffffffu;   // admitted: key > T, or key == T and index <= i_star
    bool settled = false;
#pragma unroll 1
    while (khi > klo) {
        const int shift = range_shift(klo, khi);
#pragma unroll
        for (int e = 0; e < kPer; ++e)
            if ((part >> e) & 1u) atomicAdd(&hist[kBins - 1 - ((key[e] - klo) >> shift)], 1u);
        __syncthreads();
        const uint4 fb = find_bin_db(hist, rank, sh, ph);
        const uint32_t bucket = (uint32_t)(kBins - 1) - fb.x;
        rank = fb.y;
        eq_total = fb.z;
        // entries above the bucket are in, entries below are out; the bucket itself is what is left to rank
        const uint32_t nlo = klo + (bucket << shift);
        const uint32_t nhi = shift == 0 ? nlo : min(khi, nlo + ((1u << shift) - 1u));
#pragma unroll
        for (int e = 0; e < kPer; ++e)
            if (((part >> e) & 1u) && (key[e] < nlo || key[e] > nhi)) part &= ~(1u << e);
        klo = nlo;
        khi = nhi;
        if (eq_total <= (uint32_t)kSmallList) {
#pragma unroll
            for (int e = 0; e < kPer; ++e)
                if ((part >> e) & 1u) {
                    const uint32_t at = atomicAdd(&sh.small_n, 1u);
                    sh.small_key[at] = key[e];
                    sh.small_idx[at] = idx[e];
                }
            __syncthreads();
            const int b = ph.res++ & 1;
            if (threadIdx.x < eq_total) {
                const uint32_t mk = sh.small_key[threadIdx.x], mi = sh.small_idx[threadIdx.x];
                uint32_t ahead = 0;
                for (uint32_t i = 0; i < eq_total; ++i) {
                    const uint32_t ok = sh.small_key[i], oi = sh.small_idx[i];
                    ahead += (ok > mk || (ok == mk && oi < mi)) ? 1u : 0u;
                }
                if (ahead == rank - 1u) {
                    sh.res_db[b][0] = mk;
                    sh.res_db[b][1] = mi;
                }
            }
            __syncthreads();
            T = sh.res_db[b][0];
            i_star = sh.res_db[b][1];
            settled = true;
            break;
        }
    }
    if (!settled) {
        T = klo;
        const uint32_t need_eq = rank;
        if (need_eq < eq_total) {
            // More than 32 equal keys straddle the threshold: i_star = the need_eq-th lowest index among them
            // (indices < 2^21), by two histogram passes over the index bits.
#pragma unroll
            for (int e = 0; e < kPer; ++e)
                if (((part >> e) & 1u) && key[e] == T) atomicAdd(&hist[idx[e] >> 10], 1u);
            __syncthreads();
            const uint4 f1 = find_bin_db(hist, need_eq, sh, ph);
#pragma unroll
            for (int e = 0; e < kPer; ++e)
                if (((part >> e) & 1u) && key[e] == T && (idx[e] >> 10) == f1.x) atomicAdd(&hist[idx[e] & 0x3ffu], 1u);
            __syncthreads();
            const uint4 f2 = find_bin_db(hist, f1.y, sh, ph);
            i_star = (f1.x << 10) | f2.x;
        }
    }
    if (threadIdx.x == 0) sel_ts(sh.trace, sh.trace_base + 3);   // threshold (T, i_star) settled
#pragma unroll
    for (int e = 0; e < kPer; ++e)
        if (threadIdx.x + e * kSelThreads < n_list && (key[e] > T || (key[e] == T && idx[e] <= i_star)))
            set_member(L.mem, (int)idx[e]);
    __syncthreads();
}

__device__ __noinline__ void list_select_ranged_big(const float* __restrict__ s, const SelLayout& L, int n_list,
                                                    uint32_t rank, SelShared& sh, Phase& ph) {
    list_select_ranged<8192 / kSelThreads>(s, L, n_list, rank, sh, ph);   // cap <= 8192 entries
}
// Entries per thread: 2048 / 3072 / 8192 entries in all, whatever the CTA size.
__device__ __forceinline__ void select_from_list(const float* __restrict__ s, const SelLayout& L, int n_list,
                                                 uint32_t rank, SelShared& sh, Phase& ph) {
    if (n_list <= 2048)
        list_select_ranged<2048 / kSelThreads>(s, L, n_list, rank, sh, ph);
    else if (n_list <= 3072)   // the tail of the list-length distribution at rank ~900: not worth the 8192-entry variant
        list_select_ranged<3072 / kSelThreads>(s, L, n_list, rank, sh, ph);
    else
        list_select_ranged_big(s, L, n_list, rank, sh, ph);
}

// ---- sampled path on 16-byte loads ---------------------------------------------------------------------------------
// Thread t holds the vectors v0 + (8c + u) * 1024 + t of the row (chunk c = 32768 elements, u = 0..7).  A row of one
// chunk stays in registers from the threshold estimate to the compaction; longer rows are re-read from L2 per phase.
//  (a) 1024 samples spread over the row -> their minimum / maximum -> offset-radix histogram -> the key tau that
//      the true rank-th key exceeds with overwhelming probability (the sample only decides which path runs);
//  (b) every candidate with key >= tau goes to the (key, index) list: per-thread counts, one block scan per chunk,
//      no atomics;  (c) exact selection on the list (list_select_ranged).
// Returns false (nothing admitted) when the list came out too short or too long; the caller then takes path (2).
// On entry hist (replica 0) must be all zero; it is left all zero.
constexpr int kVecPerChunk = 8;
__device__ bool sampled_tier_vec(const float* __restrict__ s, int lo, int hi, int rank, const SelLayout& L,
                                 SelShared& sh, Phase& ph) {
    const float4* s4 = reinterpret_cast<const float4*>(s);
    const int t = threadIdx.x;
    const int v0 = lo >> 2, v_end = (hi + 3) >> 2;
    const int n_chunks = (v_end - v0 + kVecPerChunk * kSelThreads - 1) / (kVecPerChunk * kSelThreads);
    const bool one = n_chunks == 1;
    const int n_cand = hi - lo;
    float4 x[kVecPerChunk];
    auto load_chunk = [&](int c) {
#pragma unroll
        for (int u = 0; u < kVecPerChunk; ++u) {
            const int vv = v0 + (c * kVecPerChunk + u) * kSelThreads + t;
            x[u] = vv < v_end ? __ldcg(s4 + vv) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    // candidate nibble of a vector: bit e clear <=> element 4 * vv + e is a candidate
    auto nib_of = [&](int vv) -> uint32_t {
        const int n = vv << 2;
        return vv < v_end ? (L.mem[n >> 5] >> (n & 31)) & 0xfu : 0xfu;
    };
    // ---- (a) threshold from ~1024 samples ----
    // One chunk: one sample per thread, out of the registers.  Longer rows: 1024 strided samples whatever the CTA size
    // (kSampPer per thread): the estimate, and with it the length of the candidate list, must not degrade in the small-CTA
    // instantiation.
    constexpr int kSampPer = kSelThreads >= 1024 ? 1 : 1024 / kSelThreads;
    uint32_t skey[kSampPer];
    bool svalid[kSampPer];
#pragma unroll
    for (int i = 0; i < kSampPer; ++i) {
        skey[i] = 0;
        svalid[i] = false;
    }
    int n_slots;
    if (one) {
        load_chunk(0);
        const int u_s = t & 7, e_s = (t >> 3) & 3;
        float4 xv = x[0];
#pragma unroll
        for (int u = 1; u < kVecPerChunk; ++u)
            if (u_s == u) xv = x[u];
        const float f = e_s == 0 ? xv.x : (e_s == 1 ? xv.y : (e_s == 2 ? xv.z : xv.w));
        skey[0] = key_max0(f);
        svalid[0] = !((nib_of(v0 + u_s * kSelThreads + t) >> e_s) & 1u);
        n_slots = min(kSelThreads, (v_end - v0));   // threads whose sampled vector can exist at all (upper bound)
    } else {
        constexpr int kSamples = kSampPer * kSelThreads;
        const int stride = max(1, n_cand / kSamples);
        n_slots = min(kSamples, (n_cand + stride - 1) / stride);
#pragma unroll
        for (int i = 0; i < kSampPer; ++i) {
            const int slot = t + i * kSelThreads;
            const int pos = lo + slot * stride;
            if (slot < n_slots) {
                skey[i] = key_max0(__ldcg(s + pos));
                svalid[i] = !((L.mem[pos >> 5] >> (pos & 31)) & 1u);
            }
        }
    }
    uint32_t kmin, kmax;
    {
        uint32_t tmin = 0xffffffffu, tmax = 0u;
        bool any = false;
#pragma unroll
        for (int i = 0; i < kSampPer; ++i)
            if (svalid[i]) {
                tmin = min(tmin, skey[i]);
                tmax = max(tmax, skey[i]);
                any = true;
            }
        block_minmax(tmin, tmax, any, sh, ph, kmin, kmax);
    }
    uint32_t tau = 0;   // 0: every candidate goes to the list
    if (kmin <= kmax) {
        const int shift = range_shift(kmin, kmax);
#pragma unroll
        for (int i = 0; i < kSampPer; ++i)
            if (svalid[i]) atomicAdd(&L.hist[kBins - 1 - ((skey[i] - kmin) >> shift)], 1u);
        __syncthreads();
        // sample rank that the true rank-th key exceeds with overwhelming probability (mean * 1.25 + 3.5 sigma + 4)
        const float mean = (float)n_slots * (float)rank / (float)n_cand;
        const uint32_t j = (uint32_t)(mean * 1.25f + 3.5f * sqrtf(mean) + 4.f);
        const uint4 fb = find_bin_db(L.hist, j, sh, ph);
        if (j <= fb.w) tau = kmin + (((uint32_t)(kBins - 1) - fb.x) << shift);
    }
    if (threadIdx.x == 0) sel_ts(sh.trace, sh.trace_base + 0);   // threshold estimate done
    // ---- (b) compaction: candidates with key >= tau ----
    // Signed compare on the raw bits: for s >= 0 it is the key order; negative scores (key 0, reading A15) pass
    // only when tau == 0, i.e. when every candidate is taken.
    const int tau_s = tau == 0u ? INT_MIN : (int)tau;
    const int wsh = ((v0 + t) & 7) * 4;                      // this thread's nibble inside its bitmask words
    uint32_t base = 0;
#pragma unroll 1
    for (int c = 0; c < n_chunks; ++c) {
        if (!one) load_chunk(c);
        const int vc = v0 + c * kVecPerChunk * kSelThreads + t;   // vector of u = 0
        // vectors u < nv of this thread exist; the bitmask words of the others are padding (select_plan), ignored
        const int nv = min(max((v_end - vc + kSelThreads - 1) / kSelThreads, 0), kVecPerChunk);
        const uint32_t exist = nv >= 8 ? 0xffffffffu : (1u << (4 * nv)) - 1u;
        const uint32_t* mrow = L.mem + (vc >> 3);                 // word of vector u: mrow[u * kSelThreads / 8], same nibble
        uint32_t hits = 0, taken = 0;   // bit 4u + e: element e of vector u
#pragma unroll
        for (int u = 0; u < kVecPerChunk; ++u) {
            if (__float_as_int(x[u].x) >= tau_s) hits |= 1u << (4 * u);
            if (__float_as_int(x[u].y) >= tau_s) hits |= 2u << (4 * u);
            if (__float_as_int(x[u].z) >= tau_s) hits |= 4u << (4 * u);
            if (__float_as_int(x[u].w) >= tau_s) hits |= 8u << (4 * u);
            taken |= ((mrow[(kSelThreads / 8) * u] >> wsh) & 0xfu) << (4 * u);
        }
        hits &= exist;
        hits &= ~taken;
        uint32_t total;
        uint32_t pos = base + block_excl_scan_db((uint32_t)__popc(hits), sh, ph, &total);
        base += total;
        const uint32_t n0 = (uint32_t)vc << 2;
        while (hits) {   // ~6 % of the elements; only the index is kept, list_select_ranged gathers the keys
            const uint32_t bit = (uint32_t)__ffs(hits) - 1u;
            hits &= hits - 1u;
            if (pos < (uint32_t)L.cap) L.list_idx[pos] = n0 + (bit >> 2) * (4u * kSelThreads) + (bit & 3u);
            ++pos;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) sel_ts(sh.trace, sh.trace_base + 1);   // compaction done
    const uint32_t n_list = base;
    if (n_list < (uint32_t)rank || n_list > (uint32_t)L.cap) return false;
    select_from_list(s, L, (int)n_list, (uint32_t)rank, sh, ph);
    return true;
}

// One tier of Eq. 6: admits into `mem` the `rank` best candidates of [lo, hi) by s (ties -> lower index).
//  (1) sampled path: 1024 strided samples give a conservative threshold on the top 11 key bits; one scan compacts
//      every candidate at or above it into the list; if the list holds >= rank entries (and fits) the exact answer
//      is selected from the list alone.  The sample only decides which path runs, never the result.
//  (2) histogram path: full histogram of the top 11 bits, second scan admits / compacts the threshold bin.
//  (3) full-scan path for a threshold bin larger than the list (massive ties).
// The slower paths of a tier, out of line so that the common path stays compact in the instruction cache.
template <bool VEC>
__device__ __noinline__ void fallback_tier(const float* __restrict__ s, int lo, int hi, int rank, const SelLayout& L,
                                           int n_words, SelShared& sh);

template <bool VEC>
__device__ __forceinline__ void select_tier(const float* __restrict__ s, int lo, int hi, int rank, const SelLayout& L,
                                            int n_words, SelShared& sh, Phase& ph, bool& hist_clean) {
    if (VEC) {
        if (!hist_clean) {
            clear_hist(L.hist, 1);
            __syncthreads();
        }
        hist_clean = true;
        if (sampled_tier_vec(s, lo, hi, rank, L, sh, ph)) return;
        hist_clean = false;   // the paths below leave their counts behind
        __syncthreads();
    }
    fallback_tier<VEC>(s, lo, hi, rank, L, n_words, sh);
}

template <bool VEC>
__device__ __noinline__ void fallback_tier(const float* __restrict__ s, int lo, int hi, int rank, const SelLayout& L,
                                           int n_words, SelShared& sh) {
    const int R = L.R, rep = threadIdx.x & (R - 1);
    uint32_t* hist = L.hist;
    const ListAppender app{L.list_key, L.list_idx, &sh.list_n, (uint32_t)L.cap};
    const int n_cand = hi - lo;
    // ---- (1) sampled threshold ----
    if (!VEC) {
        clear_hist(hist, 1);
        if (threadIdx.x == 0) sh.list_n = 0;
        __syncthreads();
        const int stride = max(1, n_cand / kSelThreads);
        const int n_slots = min(kSelThreads, (n_cand + stride - 1) / stride);
        const int pos = lo + threadIdx.x * stride;
        if (threadIdx.x < n_slots && !((L.mem[pos >> 5] >> (pos & 31)) & 1u))
            atomicAdd(&hist[kBins - 1 - (key_max0(__ldcg(s + pos)) >> 21)], 1u);
        __syncthreads();
        // sample rank that the true rank-th key exceeds with overwhelming probability (mean * 1.25 + 3.5 sigma + 4)
        const float mean = (float)n_slots * (float)rank / (float)n_cand;
        const uint32_t j = (uint32_t)(mean * 1.25f + 3.5f * sqrtf(mean) + 4.f);
        uint32_t tau_top = 0;
        find_bin(hist, 1, j, sh);
        if (j <= sh.res_total) tau_top = (uint32_t)(kBins - 1) - sh.res_bin;
        __syncthreads();
        scan_collect<VEC>(s, lo, hi, L.mem, tau_top, app);
        __syncthreads();
        const uint32_t n_list = sh.list_n;
        if (n_list >= (uint32_t)rank && n_list <= (uint32_t)L.cap) {
            list_select(L, (int)n_list, (uint32_t)rank, 0, 0u, sh);
            return;
        }
        __syncthreads();
    }
    // ---- (2) histogram of the top 11 key bits ----
    clear_hist(hist, R);
    if (threadIdx.x == 0) sh.list_n = 0;
    __syncthreads();
    scan_hist<VEC>(s, lo, hi, L.mem, hist + rep, R);
    __syncthreads();
    find_bin(hist, R, (uint32_t)rank, sh);
    const uint32_t bin1 = sh.res_bin, rank1 = sh.res_rank, cnt1 = sh.res_cnt;
    __syncthreads();
    if (cnt1 > (uint32_t)L.cap) {   // ---- (3) threshold bin too large for the list ----
        full_scan_tier(s, lo, hi, L.mem, n_words, rank, sh);
        return;
    }
    // scan 2: admit above the threshold bin, compact the threshold bin (warp-aggregated append, any order)
    const uint32_t t1 = (uint32_t)(kBins - 1) - bin1;
    scan_admit<VEC>(s, lo, hi, L.mem, t1, app);
    __syncthreads();
    list_select(L, (int)sh.list_n, rank1, 1, t1 << 21, sh);
}

// Row materialisation (fused entry point): a1's softmax normalisation summed over the heads of list l, and Eq. 5
// (PAPER.md:161-164), for this CTA's own target row -- the same arithmetic as score_stats_kernel +
// score_normalize_kernel (common.cuh helpers), so the result is bit-identical to the staged calls.  Ends with a
// barrier; the row is then re-read with ld.cg (L2, where this CTA's stores have landed).
__device__ __forceinline__ void materialize_row(const SelectParams& p, int b, int l, int N, SelShared& sh) {
    const int first = p.norm.list_first[l], nh = p.norm.list_cnt[l];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int j = warp; j < nh; j += kSelWarps) {
        const float2 st = fold_stats_warp(p.norm.part + ((long long)b * p.norm.nsel + first + j) * p.norm.n_chunks,
                                          p.norm.n_chunks, lane);
        if (lane == 0) sh.stats[j] = st;
    }
    __syncthreads();
    if (threadIdx.x == 0) sel_ts(sh.trace, 7);   // softmax statistics folded
    float4* hrow = reinterpret_cast<float4*>(const_cast<float*>(p.s_target) +
                                             ((long long)b * p.n_lists + l) * p.max_ctx);
    const float* lg = p.norm.logits + ((long long)b * p.norm.nsel + first) * p.norm.logit_stride;
    const float alpha = p.norm.alpha;
    const int nvec = (N + 3) >> 2;
    constexpr int kU = 4;   // vectors in flight per thread
#pragma unroll 1
    for (int v0 = threadIdx.x; v0 < nvec; v0 += kU * kSelThreads) {
        float4 h[kU];
        float a[kU][4];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int v = v0 + u * kSelThreads;
            h[u] = v < nvec ? hrow[v] : make_float4(0.f, 0.f, 0.f, 0.f);
            a[u][0] = a[u][1] = a[u][2] = a[u][3] = 0.f;
        }
#pragma unroll 1
        for (int j = 0; j < nh; ++j) {
            const float2 st = sh.stats[j];
            const float4* lj = reinterpret_cast<const float4*>(lg + (long long)j * p.norm.logit_stride);
            float4 x[kU];
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const int v = v0 + u * kSelThreads;
                x[u] = v < nvec ? __ldcg(lj + v) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int u = 0; u < kU; ++u) prob_accumulate4(a[u], x[u], st);
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int v = v0 + u * kSelThreads, n = v << 2;
            if (v < nvec) {
                float4 r = h[u];
                r.x = __fmaf_rn(alpha, r.x, a[u][0]);
                if (n + 1 < N) r.y = __fmaf_rn(alpha, r.y, a[u][1]);
                if (n + 2 < N) r.z = __fmaf_rn(alpha, r.z, a[u][2]);
                if (n + 3 < N) r.w = __fmaf_rn(alpha, r.w, a[u][3]);
                hrow[v] = r;
            }
        }
    }
    __syncthreads();   // the row is re-read below (ld.cg: L2, where these stores have landed for this CTA)
}

// MODE kSelBoth: both tiers of Eq. 6 and the list (the staged call).  The fused call splits the work so that the
// draft tier -- which needs nothing from stage a1 -- runs while a1 streams K:
//   kSelDraft   I_prot and I_draft = TopK(S_Draft \ I_prot, m) only; the membership bitmask goes to p.draft_mask.
//               Launched BEFORE the scoring kernel, it releases it at once (pdl_trigger right after its own dependency
//               wait) and works beside it: gridDim.x CTAs walk the rows blockIdx.x, blockIdx.x + gridDim.x, ...
//               (select.cu picks 256-thread CTAs, one per row, when many rows are in flight).
//   kSelTarget  picks the bitmask up, (materialises its target row,) runs the target tier and emits the list.
constexpr int kSelBoth = 0, kSelDraft = 1, kSelTarget = 2;

// One (sequence b, list l) row.  Returns early (uniformly over the CTA) on rows that need no selection.
template <bool VEC, int MODE>
__device__ __forceinline__ void select_row(const SelectParams& p, int b, int l, uint32_t* smem_dyn, SelShared& sh,
                                           Phase& ph, unsigned long long* tr) {
    const int N = seq_len_of(p.seq_lens, b, p.max_ctx);
    const int k = p.budgets ? p.budgets[b] : p.budget;
    int* out = p.idx_out + ((long long)b * p.n_lists + l) * p.k_max;
    int* cnt_out = p.cnt_out + (long long)b * p.n_lists + l;

    const bool invalid = k > p.k_max || k < p.n_sink + p.n_recent;   // argument error on this row (dustin.h)
    const bool all = k >= N;                                          // everything is selected (reading A12)
    const int S = min(p.n_sink, N), W = min(p.n_recent, N - S);
    const int lo = S, hi = N - W;                       // candidate range [lo, hi)
    const int c = k - S - W;
    const int m = (int)min((long long)c * p.m_num / p.m_den, (long long)c);
    const int n_words = (N + 31) >> 5;
    const float* sd = p.s_draft + (long long)b * p.draft_batch_stride + (long long)l * p.draft_list_stride;
    const float* st = p.s_target + ((long long)b * p.n_lists + l) * p.max_ctx;
    SelLayout L;
    L.mem = smem_dyn;
    L.hist = smem_dyn + p.mask_words;
    L.list_key = L.hist + (size_t)kBins * p.replicas;
    L.list_idx = L.list_key + p.list_cap;
    L.R = p.replicas;
    L.cap = p.list_cap;
    uint32_t* mem = L.mem;
    uint32_t* gmask = p.draft_mask + ((long long)b * p.n_lists + l) * p.draft_mask_stride;
    if (!invalid && !all) {
        if (MODE == kSelTarget) {
            // I_prot U I_draft as the draft-tier kernel left it (plain loads: that grid has completed and flushed); requested
            // before the row is materialised, so the trip overlaps it
            for (int w = threadIdx.x; w < n_words; w += kSelThreads) mem[w] = gmask[w];
        } else {
            // I_prot = I_sink U I_window
            for (int w = threadIdx.x; w < n_words; w += kSelThreads) {
                uint32_t bits = 0;
                const int n0 = w * 32;
                if (n0 < S) bits |= (S - n0 >= 32) ? 0xffffffffu : ((1u << (S - n0)) - 1u);
                if (n0 + 32 > hi) {   // window [hi, N) and, for now, the tail [N, 32 * n_words) of the last word
                    const int from = max(hi - n0, 0);
                    bits |= ~((1u << from) - 1u);
                }
                mem[w] = bits;
            }
        }
        if (VEC) clear_hist(L.hist, 1);
    }
    // Fused call: this CTA computes its target row itself (a1's normalisation + Eq. 5), for every row -- also those
    // that need no selection.
    const bool own_row = MODE != kSelDraft && VEC && p.norm.logits != nullptr;
    if (own_row) materialize_row(p, b, l, N, sh);
    sel_ts(tr, 2);
    if (invalid) {
        if (MODE == kSelDraft) return;
        for (int i = threadIdx.x; i < p.k_max; i += kSelThreads) out[i] = -1;
        if (threadIdx.x == 0) *cnt_out = 0;
        return;
    }
    if (all) {
        if (MODE == kSelDraft) return;
        for (int i = threadIdx.x; i < p.k_max; i += kSelThreads) out[i] = i < N ? i : -1;
        if (threadIdx.x == 0) *cnt_out = N;
        return;
    }
    bool hist_clean = VEC;
    __syncthreads();

    // tier 0: I_draft = TopK(S_Draft \ I_prot, m);  tier 1: I_target = TopK(S_Target \ (I_prot U I_draft), k-m-|I_prot|)
#pragma unroll 1
    for (int tier = (MODE == kSelTarget ? 1 : 0); tier < (MODE == kSelDraft ? 1 : 2); ++tier) {
        const int want = tier == 0 ? m : c - m;
        if (threadIdx.x == 0) sh.trace_base = 16 + 16 * tier;
        if (want > 0)
            select_tier<VEC>(tier == 0 ? sd : st, lo, hi, want, L, n_words, sh, ph, hist_clean);
        sel_ts(tr, 3 + tier);
    }
    if (MODE == kSelDraft) {
        for (int w = threadIdx.x; w < n_words; w += kSelThreads) gmask[w] = mem[w];
        return;
    }
    if (threadIdx.x == 0 && (N & 31)) mem[n_words - 1] &= (1u << (N & 31)) - 1u;   // drop the tail bits >= N
    __syncthreads();
    // I_verify in ascending order: prefix sum over the popcounts of the bitmask words.
    const int wpt = (n_words + kSelThreads - 1) / kSelThreads;   // consecutive words per thread
    const int w_lo = threadIdx.x * wpt, w_hi = min(w_lo + wpt, n_words);
    uint32_t mine = 0;
    for (int w = w_lo; w < w_hi; ++w) mine += __popc(mem[w]);
    uint32_t total;
    uint32_t pos = block_excl_scan(mine, sh, &total);
    sel_ts(tr, 5);
    // The list is assembled in shared memory (the candidate-list area is free now) and leaves in 16-byte stores; lists
    // that do not fit there, or unaligned output rows, are written entry by entry.
    const bool staged = VEC && (uint32_t)p.k_max <= 2u * (uint32_t)L.cap && (p.k_max & 3) == 0 &&
                        (reinterpret_cast<uintptr_t>(out) & 15) == 0;
    int* dst = staged ? reinterpret_cast<int*>(L.list_key) : out;
    for (int w = w_lo; w < w_hi; ++w) {
        uint32_t bits = mem[w];
        if (bits == 0xffffffffu) {   // sink and window words: 32 independent stores instead of a dependent bit chain
#pragma unroll 8
            for (int j = 0; j < 32; ++j)
                if (pos + j < (uint32_t)p.k_max) dst[pos + j] = w * 32 + j;
            pos += 32;
            continue;
        }
        while (bits) {
            const int bit = __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < (uint32_t)p.k_max) dst[pos] = w * 32 + bit;
            ++pos;
        }
    }
    for (int i = (int)total + threadIdx.x; i < p.k_max; i += kSelThreads) dst[i] = -1;
    if (staged) {
        __syncthreads();
        const int4* src4 = reinterpret_cast<const int4*>(dst);
        int4* out4 = reinterpret_cast<int4*>(out);
        for (int i = threadIdx.x; i < p.k_max / 4; i += kSelThreads) out4[i] = src4[i];
    }
    if (threadIdx.x == 0) *cnt_out = (int)total;
    // The logits of the heads that feed this row are scratch nobody reads again (one reader per logits row, whole lines:
    // api.cu): drop them from L2, or their dirty lines are written back to HBM while the attention kernel gathers.  Every
    // thread of the CTA is long past its last read of them (the barrier that ends materialize_row).
    if (own_row && p.norm.discard_logits) {
        const int first = p.norm.list_first[l], nh = p.norm.list_cnt[l];
        const int lines = (int)(p.norm.logit_stride >> 5);
        for (int j = 0; j < nh; ++j) {
            const float* row = p.norm.logits + ((long long)b * p.norm.nsel + first + j) * p.norm.logit_stride;
            for (int i = threadIdx.x; i < lines; i += kSelThreads) l2_discard128(row + (long long)i * 32);
        }
    }
}

template <bool VEC, int MODE>
__global__ void __launch_bounds__(kSelThreads, kSelThreads <= 256 ? 3 : (kSelThreads <= 512 ? 2 : 1))
    select_kernel(const SelectParams p) {
    extern __shared__ __align__(16) uint32_t smem_dyn[];
    __shared__ SelShared sh;
    unsigned long long* const tr =
        p.trace ? p.trace + ((size_t)blockIdx.y * gridDim.x + blockIdx.x + (MODE == kSelDraft ? (size_t)p.n_lists * p.batch : 0)) * 64
                : nullptr;
    sel_ts(tr, 0);
    // PDL chain invariant ("PDL chain invariant"): WAIT FIRST, THEN TRIGGER -- never the other way round.
    // The scoring kernel released here (ScoreParams::defer_wait) writes the logits scratch before any dependency wait of
    // its own, and that scratch shares the front of the workspace with the stream-K partials of the PREVIOUS call's
    // attention kernel, which released this kernel at its very start.  This wait (previous attention kernel complete and
    // visible) is therefore the only thing that orders the scoring kernel behind it.
    pdl_wait();
    if (MODE == kSelDraft) pdl_trigger();   // the scoring kernel may start now: it needs nothing from this one
    sel_ts(tr, 1);
    if (threadIdx.x == 0) {
        sh.trace = tr;
        sh.trace_base = 8;
    }
    Phase ph;
    if (MODE == kSelDraft) {
        // a few CTAs walk all rows (grid = (n_ctas, 1)); the trace shows the CTA's first row and its end
        const int n_rows = p.n_lists * p.batch;
#pragma unroll 1
        for (int row = blockIdx.x; row < n_rows; row += gridDim.x) {
            select_row<VEC, MODE>(p, row / p.n_lists, row % p.n_lists, smem_dyn, sh, ph, row == (int)blockIdx.x ? tr : nullptr);
            __syncthreads();   // the next row reuses the shared-memory state
            if (threadIdx.x == 0) sh.trace = nullptr;
        }
        sel_ts(tr, 6);
        return;
    }
    select_row<VEC, MODE>(p, blockIdx.y, blockIdx.x, smem_dyn, sh, ph, tr);
    sel_ts(tr, 6);
    pdl_trigger();
}
