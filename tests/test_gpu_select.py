"""GPU parity of stage a3 alone (dustin_topk_select, Eq. 6): fed identical fp32 scores the CUDA radix select and
the oracle's stable sort must agree bit for bit -- including heavy ties, zeros, negatives, ragged lengths,
degenerate budgets and the largest supported rows."""
import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import api

pytestmark = pytest.mark.gpu


def run_gpu(sd, st, budget, S, W, m_num, m_den, k_max=None, seq_lens=None, budgets=None):
    B, G, N = st.shape
    if k_max is None:
        k_max = int(budgets.max()) if budgets is not None else budget
    idx = torch.full((B, G, k_max), -9, dtype=torch.int32, device="cuda")
    cnt = torch.full((B, G), -9, dtype=torch.int32, device="cuda")
    sel = api.Select(budget, S, W, m_num, m_den, G, None if budgets is None else budgets.cuda())
    api.topk_select(sel, sd.cuda(), st.cuda(), idx, cnt, None if seq_lens is None else seq_lens.cuda())
    torch.cuda.synchronize()
    return idx.cpu(), cnt.cpu()


def both(sd, st, budget, S, W, m_num, m_den, k_max=None, seq_lens=None, budgets=None):
    want = ref.topk_select(sd, st, budget, S, W, m_num, m_den, k_max, seq_lens, budgets)
    got = run_gpu(sd, st, budget, S, W, m_num, m_den, k_max, seq_lens, budgets)
    assert torch.equal(got[1], want[1]), "cnt differs"
    assert torch.equal(got[0], want[0]), "idx differs"
    return got


def gen(seed):
    return torch.Generator().manual_seed(seed)


@pytest.mark.parametrize("N,k,S,W", [(1024, 128, 4, 32), (1000, 333, 0, 0), (33, 20, 3, 5), (31, 8, 1, 1),
                                     (5000, 2048, 64, 256), (70001, 4096, 64, 256), (4097, 4096, 64, 256)])
@pytest.mark.parametrize("m", [(0, 1), (1, 2), (1, 1), (3, 7)])
def test_random_scores(N, k, S, W, m):
    g = gen(N * 7 + k)
    st = torch.rand(2, 3, N, generator=g) ** 8           # skewed like attention mass
    sd = torch.rand(2, N, generator=g) ** 8
    both(sd, st, k, S, W, *m)
    sd3 = torch.rand(2, 3, N, generator=g)
    both(sd3, st, k, S, W, *m)                           # per-list draft scores


@pytest.mark.parametrize("levels", [1, 2, 5, 40])
def test_heavy_ties_break_toward_lower_index(levels):
    g = gen(levels)
    N = 3000
    st = torch.randint(0, levels, (2, 2, N), generator=g).float() / 7.0
    sd = torch.randint(0, levels, (2, N), generator=g).float() / 3.0
    for k in (100, 1500, 2999):
        both(sd, st, k, 10, 50, 1, 2)
        both(sd, st, k, 10, 50, 0, 1)


def test_zeros_negatives_and_denormals_compare_as_max_s_0():
    g = gen(11)
    N = 2000
    st = torch.randn(1, 1, N, generator=g)               # half negative -> all tie at 0
    st[0, 0, ::7] = 0.0
    st[0, 0, 1::7] = -0.0
    st[0, 0, 2::7] = 1e-42                               # denormal, still > 0
    sd = torch.randn(1, N, generator=g).clamp_max(0.0)   # every draft score <= 0: pure index order
    both(sd, st, 1200, 4, 16, 1, 2)
    both(sd, st, 300, 4, 16, 1, 2)


def test_ragged_lengths_budgets_and_degenerate_rows():
    g = gen(5)
    N = 2500
    st = torch.rand(6, 2, N, generator=g)
    sd = torch.rand(6, N, generator=g)
    seq_lens = torch.tensor([2500, 0, 1, 37, 321, 1999], dtype=torch.int32)
    budgets = torch.tensor([300, 40, 64, 36, 320, 1998], dtype=torch.int32)   # k >= N rows, k = S + W rows
    idx, cnt = both(sd, st, 0, 4, 32, 1, 2, k_max=2048, seq_lens=seq_lens, budgets=budgets)
    assert cnt[1].tolist() == [0, 0] and cnt[2].tolist() == [1, 1] and cnt[3].tolist() == [36, 36]
    # k = S + W: only the protected set
    idx, cnt = both(sd, st, 36, 4, 32, 1, 2)
    assert idx[0, 0].tolist() == list(range(4)) + list(range(N - 32, N))


@pytest.mark.parametrize("N", [131072, 1 << 20])
def test_largest_rows(N):
    g = gen(N)
    st = torch.rand(1, 2, N, generator=g)
    st[0, 1] = (st[0, 1] * 64).floor() / 64              # ties at scale
    sd = torch.rand(1, N, generator=g)
    both(sd, st, 8192, 64, 256, 1, 2)


def test_scale_invariance():
    g = gen(2)
    st = torch.rand(1, 1, 4000, generator=g)
    sd = torch.rand(1, 4000, generator=g)
    a = run_gpu(sd, st, 512, 4, 16, 1, 2)
    b = run_gpu(sd * 4.0, st * 0.125, 512, 4, 16, 1, 2)  # power-of-two rescale is exact in fp32
    assert torch.equal(a[0], b[0])


@pytest.mark.parametrize("threads", [256, 512, 1024])
def test_block_excl_scan_of_every_cta_size(threads):
    """The block-wide exclusive prefix sum of the selection kernels, alone, in each of its three instantiations (the 256-
    and 512-thread ones carry a work-around for a lane-31 store that nvcc 12.9 mis-addressed): against torch.cumsum in
    int64, on random counts, all-ones, a single non-zero and values that wrap 2^32; two scans in a row per CTA."""
    g = torch.Generator(device="cpu").manual_seed(1234 + threads)
    rows = [torch.randint(0, 5000, (threads,), generator=g), torch.ones(threads, dtype=torch.int64),
            torch.zeros(threads, dtype=torch.int64), torch.randint(0, 2, (threads,), generator=g),
            torch.randint(0, 1 << 31, (threads,), generator=g)]
    rows[2][threads - 1] = 7
    for k in range(11):
        rows.append(torch.randint(0, 40000, (threads,), generator=g))
    v = torch.stack(rows)                                          # int64 [n_blocks, threads], values < 2^31
    out, total = api.debug_block_scan(threads, v.to(torch.int32).cuda())
    torch.cuda.synchronize()
    out, total = out.cpu().to(torch.int64) & 0xFFFFFFFF, total.cpu().to(torch.int64) & 0xFFFFFFFF
    for j, vv in enumerate((v, v + 1)):
        inc = torch.cumsum(vv, dim=1)
        assert torch.equal(out[j], (inc - vv) & 0xFFFFFFFF), f"threads={threads} scan {j}: prefixes differ"
        assert torch.equal(total[j], inc[:, -1] & 0xFFFFFFFF), f"threads={threads} scan {j}: totals differ"
