// select_cluster.cu -- the target tier of Eq. 6 for FEW LONG ROWS: one thread-block cluster per
// (sequence, list) row instead of one CTA.
//
// With one CTA per row, 16 rows (the paper's one global list per sequence, at batch 16) or 32 rows (128k
// context at batch 4) leave most of the 148 SMs idle while each busy SM pushes a whole row -- and, in the one-shot call,
// the logits of all heads that feed it -- through its own L2 port.  Here a row is cut into C contiguous slices (C = 2, 4
// or 8 CTAs of one cluster); every CTA
//   1. materialises its slice of the target row (a1's normalisation summed over the heads of the list + Eq. 5, the same
//      arithmetic as score_normalize_kernel: bit-identical to the staged calls) and keeps it in shared memory,
//   2. takes part in an exact cluster-wide selection of the `want` best candidates: offset-radix passes whose 2048-bin
//      histograms are built per CTA in shared memory and summed by every CTA through distributed shared memory (each CTA
//      reads all C copies and arrives at the same bin), until the threshold bin is small enough to be ranked by brute
//      force ((key desc, index asc) order, which settles ties; every CTA gathers the C partial lists and ranks them
//      itself) -- or, when more equal keys than that straddle the threshold, two more passes over the index bits find
//      the last admitted index,
//   3. emits its part of the ascending index list at the offset given by the popcounts of the slices before it.
// No sampling, no candidate list, no fallback path: every step is exact, and the only state is the slice (values + a
// 4 KB mask) and two histograms in shared memory.  The draft tier has been taken beforehand by the draft-tier kernel (select.cu); its
// membership bitmask arrives in SelectParams::draft_mask.
#include "kernels.cuh"

#include "../../include/dustin_debug.h"

#include <cooperative_groups.h>

#include <map>
#include <mutex>
#include <tuple>

namespace dustin {

namespace cg = cooperative_groups;

namespace {

constexpr int kMaxC = 8;               // largest cluster
constexpr int kCT = 1024;             // threads per CTA
constexpr int kCWarps = kCT / 32;
constexpr int kCBins = 2048;
constexpr int kCVec = 8;              // a slice holds at most kCVec * kCT * 4 = 32768 elements (one mask word per thread)
constexpr int kCSmall = 128;          // threshold bins up to this size are ranked by brute force

struct ClShared {
    uint32_t hist[2][kCBins];         // double-buffered local histograms (peers read them through DSMEM)
    uint32_t minmax_all[2 * kMaxC];   // (min, max) of the candidate keys of every CTA (each pushes its pair to all)
    uint32_t total_all[kMaxC];        // popcount of the finished mask slice of every CTA (pushed likewise)
    uint32_t small_n;                 // this CTA's entries of the threshold bin (peers gather them through DSMEM)
    uint32_t small_key[kCSmall], small_idx[kCSmall];
    uint32_t all_key[kCSmall], all_idx[kCSmall];   // the whole threshold bin, gathered from the C CTAs
    uint32_t result[2];               // (T, i_star)
    uint32_t warp_a[kCWarps], warp_b[kCWarps];   // block reductions
    uint32_t res[4];                  // find_bin result
    float2 stats[64];                 // (M, 1/Z) of the heads feeding this row
};

__device__ __forceinline__ uint32_t key_max0(float s) { return __float_as_uint(fmaxf(s, 0.f)); }

__device__ __forceinline__ int range_shift(uint32_t kmin, uint32_t kmax) {
    const int bits = kmax > kmin ? 32 - __clz(kmax - kmin) : 0;
    return bits > 11 ? bits - 11 : 0;
}

// Block-wide (min, max) of the per-thread values; two barriers.
__device__ __forceinline__ void block_minmax(uint32_t tmin, uint32_t tmax, ClShared& sh, uint32_t& kmin, uint32_t& kmax) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lo = __reduce_min_sync(0xffffffffu, tmin), hi = __reduce_max_sync(0xffffffffu, tmax);
    __syncthreads();
    if (lane == 0) {
        sh.warp_a[warp] = lo;
        sh.warp_b[warp] = hi;
    }
    __syncthreads();
    kmin = __reduce_min_sync(0xffffffffu, sh.warp_a[lane]);
    kmax = __reduce_max_sync(0xffffffffu, sh.warp_b[lane]);
}

// Exclusive prefix of v over the block in thread order; *total = block sum.  Two barriers.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, ClShared& sh, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += o;
    }
    const uint32_t wtot = __shfl_sync(0xffffffffu, inc, 31);
    __syncthreads();
    if (lane == 0) sh.warp_a[warp] = wtot;
    __syncthreads();
    const uint32_t t = sh.warp_a[lane];
    uint32_t ti = t;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, ti, off);
        if (lane >= off) ti += o;
    }
    *total = __shfl_sync(0xffffffffu, ti, 31);
    return __shfl_sync(0xffffffffu, ti - t, warp) + inc - v;
}

// The histograms hist[buf] of all C CTAs hold one digit pass: sums them (every CTA reads all copies and computes the
// same thing), finds the bin that holds rank `rank` (1-based, ascending bin order) and returns {bin, rank inside the
// bin, bin count, total}.  Clears this CTA's OTHER buffer for the pass after.  Cluster barrier first (all copies
// complete), block barriers inside.
__device__ __forceinline__ uint4 cluster_find_bin(cg::cluster_group& cluster, ClShared& sh, int C, int buf, uint32_t rank) {
    cluster.sync();
    const int t = threadIdx.x;
    uint32_t c0 = 0, c1 = 0;
    for (int r = 0; r < C; ++r) {
        const uint2 v = *reinterpret_cast<const uint2*>(cluster.map_shared_rank(&sh.hist[buf][2 * t], r));
        c0 += v.x;
        c1 += v.y;
    }
    sh.hist[buf ^ 1][2 * t] = 0u;       // nobody reads that copy any more (its readers have passed the barrier above)
    sh.hist[buf ^ 1][2 * t + 1] = 0u;
    uint32_t total;
    const uint32_t run = block_excl_scan(c0 + c1, sh, &total);
    if (run < rank && rank <= run + c0) {
        sh.res[0] = 2 * t;
        sh.res[1] = rank - run;
        sh.res[2] = c0;
    } else if (run + c0 < rank && rank <= run + c0 + c1) {
        sh.res[0] = 2 * t + 1;
        sh.res[1] = rank - run - c0;
        sh.res[2] = c1;
    }
    __syncthreads();
    return make_uint4(sh.res[0], sh.res[1], sh.res[2], total);
}

__global__ void __launch_bounds__(kCT, 1) select_cluster_kernel(const SelectParams p, const int C) {
    extern __shared__ __align__(16) uint32_t mask[];   // this CTA's slice of the membership bitmask
    __shared__ ClShared sh;
    cg::cluster_group cluster = cg::this_cluster();
    const int rank_c = (int)cluster.block_rank();
    const int l = blockIdx.x / C, b = blockIdx.y;
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
    unsigned long long* const tr = p.trace ? p.trace + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 64 : nullptr;
    auto ts = [&](int slot) {
        if (tr != nullptr && t == 0) {
            unsigned long long v;
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(v));
            tr[slot] = v;
        }
    };
    ts(0);
    sh.hist[0][2 * t] = sh.hist[0][2 * t + 1] = 0u;
    sh.hist[1][2 * t] = sh.hist[1][2 * t + 1] = 0u;
    if (t == 0) sh.small_n = 0u;
    pdl_wait();
    ts(1);

    const int N = seq_len_of(p.seq_lens, b, p.max_ctx);
    const int k = p.budgets ? p.budgets[b] : p.budget;
    int* out = p.idx_out + ((long long)b * p.n_lists + l) * p.k_max;
    int* cnt_out = p.cnt_out + (long long)b * p.n_lists + l;
    const bool invalid = k > p.k_max || k < p.n_sink + p.n_recent;   // argument error on this row (dustin.h)
    const bool all = k >= N;                                          // everything is selected (reading A12)
    const bool selecting = !invalid && !all;
    const int S = min(p.n_sink, N), W = min(p.n_recent, N - S);
    const int c = k - S - W;
    const int m = (int)min((long long)c * p.m_num / p.m_den, (long long)c);
    uint32_t rank = selecting ? (uint32_t)(c - m) : 0u;   // candidates still to admit (the draft tier took m)

    // this CTA's slice [a, e) of the row: a multiple of 128 elements per CTA (whole mask words, whole vectors)
    const int per = (((N + C - 1) / C) + 127) & ~127;
    const int a = min(rank_c * per, N), e = min(a + per, N);
    const int va = a >> 2, ve = a < e ? (e + 3) >> 2 : va;   // vectors [va, ve)
    const int wa = a >> 5, we = a < e ? (e + 31) >> 5 : wa;   // mask words [wa, we); none for an empty slice
    float* row = const_cast<float*>(p.s_target) + ((long long)b * p.n_lists + l) * p.max_ctx;
    const int mask_words = per / 32 + 4;
    if (selecting) {
        const uint32_t* gmask = p.draft_mask + ((long long)b * p.n_lists + l) * p.draft_mask_stride;
        for (int w = wa + t; w < we; w += kCT) mask[w - wa] = gmask[w];   // I_prot U I_draft (tail bits >= N are set)
    }

    // ---- 1. the slice of the target row: a1's normalisation over the heads of the list + Eq. 5, kept in shared memory ----
    // Element j of mask word w (slice-relative) lives at vals[33 * w + j]: a thread later walks the 32 elements of ITS word,
    // and the odd pitch keeps the lanes of a warp on different banks while they do.
    float* vals = reinterpret_cast<float*>(mask + mask_words);
    {
        const int first = p.norm.list_first[l], nh = p.norm.list_cnt[l];
        for (int j = warp; j < nh; j += kCWarps) {
            const float2 st = fold_stats_warp(p.norm.part + ((long long)b * p.norm.nsel + first + j) * p.norm.n_chunks,
                                              p.norm.n_chunks, lane);
            if (lane == 0) sh.stats[j] = st;
        }
        __syncthreads();
        ts(7);
        float4* hrow = reinterpret_cast<float4*>(row);
        const float* lg = p.norm.logits + ((long long)b * p.norm.nsel + first) * p.norm.logit_stride;
        const float alpha = p.norm.alpha;
#pragma unroll 2
        for (int v = va + t; v < ve; v += kCT) {
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            float4 r = hrow[v];
            // the logits of four heads at a time: their loads in flight together, accumulated in head order
#pragma unroll 1
            for (int j0 = 0; j0 < nh; j0 += 4) {
                float4 lgv[4];
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (j0 + j < nh)
                        lgv[j] = __ldcg(reinterpret_cast<const float4*>(lg + (long long)(j0 + j) * p.norm.logit_stride) + v);
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (j0 + j < nh) prob_accumulate4(acc, lgv[j], sh.stats[j0 + j]);
            }
            const int n = v << 2;
            r.x = __fmaf_rn(alpha, r.x, acc[0]);
            if (n + 1 < N) r.y = __fmaf_rn(alpha, r.y, acc[1]);
            if (n + 2 < N) r.z = __fmaf_rn(alpha, r.z, acc[2]);
            if (n + 3 < N) r.w = __fmaf_rn(alpha, r.w, acc[3]);
            hrow[v] = r;
            float* dst = vals + 33 * ((n - a) >> 5) + ((n - a) & 31);
            dst[0] = r.x;
            dst[1] = r.y;
            dst[2] = r.z;
            dst[3] = r.w;
        }
    }
    ts(2);
    __syncthreads();   // mask slice and values are in shared memory

    // ---- 2. cluster-wide exact selection of the `rank` best candidates ------------------------------------------------
    // Thread t owns the mask words t, t + kCT ... of the slice (at most one: a slice has <= 1024 words) and with them the
    // 32 elements of each; `part` = its candidates still inside the key range under consideration.
    const int w_own = wa + t;
    const bool has_word = selecting && w_own < we;
    uint32_t part = has_word ? ~mask[t] : 0u;
    const float* myvals = vals + 33 * t;
    auto key_at = [&](int bit) -> uint32_t { return key_max0(myvals[bit]); };
    auto idx_at = [&](int bit) -> uint32_t { return (uint32_t)(w_own * 32 + bit); };
    uint32_t admitted = 0;   // bits this thread adds to its own mask word (no atomics: the word is its own)
    if (rank > 0) {   // cluster-uniform
        // key range of all candidates
        uint32_t tmin = 0xffffffffu, tmax = 0u;
        for (uint32_t pb = part; pb; pb &= pb - 1) {
            const uint32_t key = key_at(__ffs(pb) - 1);
            tmin = min(tmin, key);
            tmax = max(tmax, key);
        }
        uint32_t lmin, lmax;
        block_minmax(tmin, tmax, sh, lmin, lmax);
        if (t < C) {   // pushed to every peer: after the barrier each CTA reads its own copy
            uint32_t* mm = cluster.map_shared_rank(sh.minmax_all, t);
            mm[2 * rank_c] = lmin;
            mm[2 * rank_c + 1] = lmax;
        }
        cluster.sync();
        uint32_t klo = 0xffffffffu, khi = 0u;
        for (int r = 0; r < C; ++r) {
            klo = min(klo, sh.minmax_all[2 * r]);
            khi = max(khi, sh.minmax_all[2 * r + 1]);
        }
        ts(16);
        // offset-radix passes: the current key range [klo, khi] is spread over the 2048 bins (bin 0 = largest keys)
        int buf = 0;
        uint32_t T = klo, i_star = 0xffffffffu, eq_total = 0;
        bool settled = false;
#pragma unroll 1
        for (int pass = 0; pass < 4 && !settled; ++pass) {
            const int shift = range_shift(klo, khi);
            for (uint32_t pb = part; pb; pb &= pb - 1)
                atomicAdd(&sh.hist[buf][kCBins - 1 - ((key_at(__ffs(pb) - 1) - klo) >> shift)], 1u);
            const uint4 fb = cluster_find_bin(cluster, sh, C, buf, rank);
            buf ^= 1;
            const uint32_t bucket = (uint32_t)(kCBins - 1) - fb.x;
            rank = fb.y;
            eq_total = fb.z;
            const uint32_t nlo = klo + (bucket << shift);
            const uint32_t nhi = shift == 0 ? nlo : min(khi, nlo + ((1u << shift) - 1u));
            // above the bucket: in; below: out; the bucket itself stays under consideration
            for (uint32_t pb = part; pb; pb &= pb - 1) {
                const int bit = __ffs(pb) - 1;
                const uint32_t key = key_at(bit);
                if (key > nhi) admitted |= 1u << bit;
                if (key < nlo || key > nhi) part &= ~(1u << bit);
            }
            klo = nlo;
            khi = nhi;
            if (eq_total <= (uint32_t)kCSmall || khi == klo) settled = true;
        }
        ts(17);
        if (eq_total <= (uint32_t)kCSmall) {
            // Every CTA lists its own entries of the threshold bin, then gathers the C lists (in CTA order: the same array
            // everywhere) and ranks them by brute force in (key desc, index asc) order.
            for (uint32_t pb = part; pb; pb &= pb - 1) {
                const int bit = __ffs(pb) - 1;
                const uint32_t at = atomicAdd(&sh.small_n, 1u);
                sh.small_key[at] = key_at(bit);
                sh.small_idx[at] = idx_at(bit);
            }
            cluster.sync();
            if (t < kCSmall) {
                int r = 0, off = t;   // entry t of the concatenation of the C lists
                uint32_t nr = *cluster.map_shared_rank(&sh.small_n, 0);
                while (r < C - 1 && (uint32_t)off >= nr) {
                    off -= (int)nr;
                    ++r;
                    nr = *cluster.map_shared_rank(&sh.small_n, r);
                }
                if ((uint32_t)t < eq_total) {
                    sh.all_key[t] = cluster.map_shared_rank(sh.small_key, r)[off];
                    sh.all_idx[t] = cluster.map_shared_rank(sh.small_idx, r)[off];
                }
            }
            __syncthreads();
            if ((uint32_t)t < eq_total) {
                const uint32_t mk = sh.all_key[t], mi = sh.all_idx[t];
                uint32_t ahead = 0;
                for (uint32_t i = 0; i < eq_total; ++i) {
                    const uint32_t ok = sh.all_key[i], oi = sh.all_idx[i];
                    ahead += (ok > mk || (ok == mk && oi < mi)) ? 1u : 0u;
                }
                if (ahead == rank - 1u) {
                    sh.result[0] = mk;
                    sh.result[1] = mi;
                }
            }
            __syncthreads();
            T = sh.result[0];
            i_star = sh.result[1];
        } else {
            // more than kCSmall EQUAL keys straddle the threshold (khi == klo): the `rank` lowest indices among them
            // are admitted; i_star = the rank-th lowest, found by two passes over the index bits (indices < 2^20:
            // digit 1 = index >> 10, digit 2 = index & 1023; ascending bin order)
            T = klo;
            if (rank < eq_total) {
                for (uint32_t pb = part; pb; pb &= pb - 1) atomicAdd(&sh.hist[buf][idx_at(__ffs(pb) - 1) >> 10], 1u);
                const uint4 f1 = cluster_find_bin(cluster, sh, C, buf, rank);
                buf ^= 1;
                for (uint32_t pb = part; pb; pb &= pb - 1) {
                    const uint32_t i = idx_at(__ffs(pb) - 1);
                    if ((i >> 10) == f1.x) atomicAdd(&sh.hist[buf][i & 0x3ffu], 1u);
                }
                const uint4 f2 = cluster_find_bin(cluster, sh, C, buf, f1.y);
                buf ^= 1;
                i_star = (f1.x << 10) | f2.x;
            }
        }
        for (uint32_t pb = part; pb; pb &= pb - 1) {
            const int bit = __ffs(pb) - 1;
            const uint32_t key = key_at(bit);
            if (key > T || (key == T && idx_at(bit) <= i_star)) admitted |= 1u << bit;
        }
        ts(19);
    }

    // ---- 3. the ascending list: this slice's members at the offset given by the slices before it ----------------------
    uint32_t mine = 0, bits = 0;
    const int w = wa + t;   // one mask word per thread (a slice has at most 1024 words)
    if (selecting && w < we) {
        bits = mask[t] | admitted;
        if (w == ((N + 31) >> 5) - 1 && (N & 31)) bits &= (1u << (N & 31)) - 1u;   // drop the tail bits >= N
        mine = (uint32_t)__popc(bits);
    }
    uint32_t total_local;
    uint32_t pos = block_excl_scan(mine, sh, &total_local);
    if (t < C) cluster.map_shared_rank(sh.total_all, t)[rank_c] = total_local;   // pushed to every peer
    cluster.sync();   // also the last access to a peer's shared memory: no CTA is read after it has gone past this point
    uint32_t base = 0, grand = 0;
    for (int r = 0; r < C; ++r) {
        const uint32_t tr_ = sh.total_all[r];
        if (r < rank_c) base += tr_;
        grand += tr_;
    }
    ts(5);
    if (selecting) {
        pos += base;
        while (bits) {
            const int bit = __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < (uint32_t)p.k_max) out[pos] = w * 32 + bit;
            ++pos;
        }
        for (int i = (int)grand + rank_c * kCT + t; i < p.k_max; i += C * kCT) out[i] = -1;
        if (rank_c == 0 && t == 0) *cnt_out = (int)grand;
    } else {
        // rows that need no selection: argument error (all -1, cnt 0) or k >= N (everything)
        for (int i = rank_c * kCT + t; i < p.k_max; i += C * kCT) out[i] = (all && !invalid && i < N) ? i : -1;
        if (rank_c == 0 && t == 0) *cnt_out = invalid ? 0 : N;
    }
    ts(6);
    pdl_trigger();
}

size_t cluster_smem_bytes(int max_ctx, int C) {
    const int per = (((max_ctx + C - 1) / C) + 127) & ~127;
    return (size_t)(per / 32 + 4) * sizeof(uint32_t) + (size_t)(per / 32) * 33 * sizeof(float);   // mask slice + values
}

cudaError_t raise_cluster_smem() {
    static DeviceOnce once;
    return ensure_dyn_smem(reinterpret_cast<const void*>(select_cluster_kernel), 200 * 1024, once);
}

// Clusters of C CTAs of this kernel that the current device can hold at once (cudaOccupancyMaxActiveClusters; a
// cluster is gang-scheduled inside one GPC, so this is less than SMs / C).  0 on error.
int max_active_clusters(int C, size_t smem) {
    static std::mutex mu;
    static std::map<std::tuple<int, int, size_t>, int> cache;   // (device, C, smem) -> clusters
    const auto key = std::make_tuple(current_device(), C, smem);
    {
        std::lock_guard<std::mutex> lk(mu);
        const auto it = cache.find(key);
        if (it != cache.end()) return it->second;
    }
    if (raise_cluster_smem() != cudaSuccess) return 0;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C * 64, 1);
    cfg.blockDim = dim3(kCT);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, select_cluster_kernel, &cfg) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    std::lock_guard<std::mutex> lk(mu);
    cache[key] = n;
    return n;
}

}  // namespace

// CTAs per row for the cluster kernel, or 0 when one CTA per row (select.cu) serves better: enough rows to fill the GPU,
// rows too long for the shared-memory slices, or rows whose 16-byte alignment the kernel relies on is missing.  The
// largest cluster size whose clusters for ALL rows are resident at once is taken (a second wave would double the time).
int select_cluster_size(const SelectParams& p) {
    const int forced = knob(DUSTIN_KNOB_SELECT_SPLIT);
    if (forced == 1) return 0;
    const long long rows = (long long)p.n_lists * p.batch;
    const bool vec = (p.max_ctx & 3) == 0 && ((uintptr_t)p.s_target & 15) == 0;
    if (!vec || p.norm.logits == nullptr || p.draft_mask == nullptr || p.max_ctx < 1) return 0;
    auto fits = [&](int C) { return ((((p.max_ctx + C - 1) / C) + 127) & ~127) <= kCVec * kCT * 4; };
    if (forced == 2 || forced == 4 || forced == 8) return fits(forced) ? forced : 0;
    if (rows * 2 > device_sm_count()) return 0;       // one CTA per row already covers at least half the SMs
    for (int C = kMaxC; C >= 2; C >>= 1)
        if (fits(C) && rows <= max_active_clusters(C, cluster_smem_bytes(p.max_ctx, C))) return C;
    return 0;
}

cudaError_t launch_select_cluster(const SelectParams& p_in, int C, cudaStream_t stream) {
    SelectParams p = p_in;
    p.trace = nullptr;
    if (knob(DUSTIN_KNOB_SELECT_TRACE)) {
        size_t bytes = 0;
        void* buf = trace_buffer(&bytes);
        if (buf && bytes >= (size_t)C * p.n_lists * p.batch * 64 * sizeof(unsigned long long))
            p.trace = static_cast<unsigned long long*>(buf);
    }
    const size_t smem = cluster_smem_bytes(p.max_ctx, C);
    {
        const cudaError_t e = raise_cluster_smem();
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.n_lists * C, p.batch);
    cfg.blockDim = dim3(kCT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl_enabled() ? 2 : 1;
    ProfScope prof(kKernSelectCluster, stream);
    return cudaLaunchKernelEx(&cfg, select_cluster_kernel, p, C);
}

}  // namespace dustin
