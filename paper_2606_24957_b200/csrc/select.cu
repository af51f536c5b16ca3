// select.cu -- stage a3: tiered top-k of Eq. 6 with the protected sink + recent window counted
// inside the budget.  One CTA per (sequence, list) row.
//
// No sort.  Each tier is an exact radix select (11/11/10-bit digits, shared-memory histograms) over the ordered
// uint32 image of max(score, 0); ties at the threshold are admitted in index order through warp ballots; the
// membership set is a bitmask in shared memory (N/8 bytes) and the ascending index list falls out of a prefix
// sum over its popcounts.  The score rows (<= 512 KB) are re-read from L2 a handful of times; HBM sees them once.
#include "kernels.cuh"

namespace dustin {

namespace {

constexpr int kSelThreads = 1024;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kBins = 2048;

__device__ __forceinline__ uint32_t key_of(float s) { return s > 0.f ? __float_as_uint(s) : 0u; }

struct SelShared {
    uint32_t hist[kBins];
    uint32_t warp_tot[kSelWarps];
    uint32_t res_bin, res_rank, res_cnt;
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
    if (lane == 31) sh.warp_tot[warp] = inc;
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < kSelWarps; ++w) {
        const uint32_t t = sh.warp_tot[w];
        if (w < warp) base += t;
        tot += t;
    }
    if (total) *total = tot;
    return base + inc - v;
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
        const uint32_t c0 = sh.hist[2 * threadIdx.x], c1 = sh.hist[2 * threadIdx.x + 1];
        const uint32_t excl = block_excl_scan(c0 + c1, sh, nullptr);
        const uint32_t r = (uint32_t)rank;
        if (excl < r && r <= excl + c0) {
            sh.res_bin = 2 * threadIdx.x;
            sh.res_rank = r - excl;
            sh.res_cnt = c0;
        } else if (excl + c0 < r && r <= excl + c0 + c1) {
            sh.res_bin = 2 * threadIdx.x + 1;
            sh.res_rank = r - excl - c0;
            sh.res_cnt = c1;
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

__global__ void __launch_bounds__(kSelThreads) select_kernel(const SelectParams p) {
    extern __shared__ uint32_t mem[];   // membership bitmask, ceil(max_ctx / 32) words
    __shared__ SelShared sh;
    const int l = blockIdx.x, b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = seq_len_of(p.seq_lens, b, p.max_ctx);
    const int k = p.budgets ? p.budgets[b] : p.budget;
    int* out = p.idx_out + ((long long)b * p.n_lists + l) * p.k_max;
    int* cnt_out = p.cnt_out + (long long)b * p.n_lists + l;

    if (k > p.k_max || k < p.n_sink + p.n_recent) {   // argument error on this row (dustin.h)
        for (int i = threadIdx.x; i < p.k_max; i += kSelThreads) out[i] = -1;
        if (threadIdx.x == 0) *cnt_out = 0;
        return;
    }
    if (k >= N) {   // everything is selected (reading A12)
        for (int i = threadIdx.x; i < p.k_max; i += kSelThreads) out[i] = i < N ? i : -1;
        if (threadIdx.x == 0) *cnt_out = N;
        return;
    }
    const int S = min(p.n_sink, N), W = min(p.n_recent, N - S);
    const int lo = S, hi = N - W;                       // candidate range [lo, hi)
    const int c = k - S - W;
    const int m = (int)min((long long)c * p.m_num / p.m_den, (long long)c);
    const int n_words = (N + 31) >> 5;
    const float* sd = p.s_draft + (long long)b * p.draft_batch_stride + (long long)l * p.draft_list_stride;
    const float* st = p.s_target + ((long long)b * p.n_lists + l) * p.max_ctx;

    // I_prot = I_sink U I_window
    for (int w = threadIdx.x; w < n_words; w += kSelThreads) {
        uint32_t bits = 0;
        const int n0 = w * 32;
        if (n0 < S) bits |= (S - n0 >= 32) ? 0xffffffffu : ((1u << (S - n0)) - 1u);
        if (n0 + 32 > hi) {
            const int from = max(hi - n0, 0), to = min(N - n0, 32);   // bits [from, to)
            const uint32_t upto = to >= 32 ? 0xffffffffu : ((1u << to) - 1u);
            bits |= upto & ~((1u << from) - 1u);
        }
        mem[w] = bits;
    }
    __syncthreads();

    int need_eq, eq_total;
    if (m > 0) {        // I_draft = TopK(S_Draft \ I_prot, m)
        const uint32_t T = radix_select(sd, lo, hi, mem, m, sh, need_eq, eq_total);
        admit_tier(sd, lo, hi, mem, n_words, T, need_eq, eq_total, sh);
    }
    if (c - m > 0) {    // I_target = TopK(S_Target \ (I_prot U I_draft), k - m - |I_prot|)
        const uint32_t T = radix_select(st, lo, hi, mem, c - m, sh, need_eq, eq_total);
        admit_tier(st, lo, hi, mem, n_words, T, need_eq, eq_total, sh);
    }

    // I_verify in ascending order: prefix sum over the popcounts of the bitmask words.
    const int wpt = (n_words + kSelThreads - 1) / kSelThreads;   // consecutive words per thread
    const int w_lo = threadIdx.x * wpt, w_hi = min(w_lo + wpt, n_words);
    uint32_t mine = 0;
    for (int w = w_lo; w < w_hi; ++w) mine += __popc(mem[w]);
    uint32_t total;
    uint32_t pos = block_excl_scan(mine, sh, &total);
    for (int w = w_lo; w < w_hi; ++w) {
        uint32_t bits = mem[w];
        while (bits) {
            const int bit = __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < (uint32_t)p.k_max) out[pos] = w * 32 + bit;
            ++pos;
        }
    }
    for (int i = (int)total + threadIdx.x; i < p.k_max; i += kSelThreads) out[i] = -1;
    if (threadIdx.x == 0) *cnt_out = (int)total;
    (void)lane;
    (void)warp;
}

}  // namespace

size_t select_smem_bytes(int max_ctx) { return (size_t)((max_ctx + 31) / 32) * 4; }

cudaError_t launch_select(const SelectParams& p, cudaStream_t stream) {
    const size_t smem = select_smem_bytes(p.max_ctx);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    ProfScope prof(kKernSelect, stream);
    select_kernel<<<dim3(p.n_lists, p.batch), kSelThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace dustin
