"""Pins of the oracle's tiered top-k (Eq. 6; protected-set rule :443) -- SURVEY.md §8c O3.
CPU only."""
import itertools

import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import synth


def brute_select(sd, st, k, S, W, m):
    """Eq. 6 by exhaustive argmax, written independently of the oracle (no sort): repeatedly take the best
    remaining candidate (ties -> lower index, reading A11)."""
    N = len(sd)
    if k >= N:
        return list(range(N))
    S2 = min(S, N)
    W2 = min(W, N - S2)
    prot = set(range(S2)) | set(range(N - W2, N))
    c = k - len(prot)
    m = min(m, c)
    chosen = set(prot)
    for scores, quota in ((sd, m), (st, c - m)):
        for _ in range(quota):
            best = None
            for n in range(N):
                if n in chosen:
                    continue
                if best is None or max(scores[n], 0.0) > max(scores[best], 0.0):
                    best = n
            if best is None:
                break
            chosen.add(best)
    return sorted(chosen)


@pytest.mark.parametrize("seed", range(6))
def test_select_brute_force_tiny(seed):
    g = torch.Generator().manual_seed(seed)
    N = 12
    for k, S, W, (mn, md) in itertools.product((5, 7, 12, 20), (0, 1, 2), (0, 2, 3), ((0, 1), (1, 2), (1, 1), (1, 3))):
        if S + W > k:
            continue
        # quantised scores so that ties are frequent
        sd = (torch.randint(0, 4, (1, N), generator=g).float() / 4).contiguous()
        st = (torch.randint(0, 4, (1, 1, N), generator=g).float() / 4).contiguous()
        idx, cnt = ref.topk_select(sd, st, k, S, W, mn, md, k_max=k)
        c = k - min(S, N) - min(W, N - min(S, N))
        want = brute_select(sd[0].tolist(), st[0, 0].tolist(), k, S, W, (c * mn) // md)
        got = idx[0, 0, :cnt[0, 0]].tolist()
        assert got == want, (k, S, W, mn, md)
        assert (idx[0, 0, cnt[0, 0]:] == -1).all()


def test_select_invariants_and_thresholds():
    g = torch.Generator().manual_seed(11)
    B, G, N, k, S, W = 3, 2, 500, 64, 4, 16
    sd = torch.rand(B, N, generator=g)
    st = torch.rand(B, G, N, generator=g)
    idx, cnt = ref.topk_select(sd, st, k, S, W, 1, 2)
    c, m = k - S - W, (k - S - W) // 2
    for b in range(B):
        for l in range(G):
            sel = idx[b, l].tolist()
            assert cnt[b, l] == k and len(set(sel)) == k and sel == sorted(sel)
            assert min(sel) >= 0 and max(sel) < N
            assert set(range(S)) <= set(sel) and set(range(N - W, N)) <= set(sel)       # :166, :443
            cand = [n for n in range(S, N - W)]
            # tier 1 = the m best draft scores among the candidates (library sort as the textbook definition)
            order = sorted(cand, key=lambda n: (-sd[b, n].item(), n))
            tier1 = set(order[:m])
            assert tier1 <= set(sel)
            rest = [n for n in cand if n not in tier1]
            order2 = sorted(rest, key=lambda n: (-st[b, l, n].item(), n))
            tier2 = set(order2[:c - m])
            assert set(sel) == set(range(S)) | set(range(N - W, N)) | tier1 | tier2
            # threshold invariant: no unselected candidate beats the weakest admitted tier-2 score
            thr = min(st[b, l, n].item() for n in tier2)
            assert all(st[b, l, n].item() <= thr for n in cand if n not in set(sel))


@pytest.mark.parametrize("mn,md,which", [(0, 1, "target"), (1, 1, "draft")])
def test_select_single_tier_reduces_to_plain_topk(mn, md, which):
    """Dustin-T (m = 0) and Dustin-D (m = k - |prot|): one plain top-k == torch.topk."""
    g = torch.Generator().manual_seed(4)
    N, k, S, W = 1000, 100, 4, 16
    sd = torch.rand(2, N, generator=g)
    st = torch.rand(2, 1, N, generator=g)
    idx, cnt = ref.topk_select(sd, st, k, S, W, mn, md)
    src = st[:, 0] if which == "target" else sd
    for b in range(2):
        top = torch.topk(src[b, S:N - W], k - S - W).indices + S           # distinct random values: no ties
        want = sorted(list(range(S)) + top.tolist() + list(range(N - W, N)))
        assert idx[b, 0].tolist() == want


def test_select_all_equal_scores_take_lowest_indices():
    N, k, S, W = 100, 20, 2, 3
    idx, cnt = ref.topk_select(torch.ones(1, N), torch.ones(1, 1, N), k, S, W, 1, 2)
    assert idx[0, 0].tolist() == list(range(0, 2 + 15)) + [97, 98, 99]


def test_select_scale_invariance_and_degenerate_sizes():
    g = torch.Generator().manual_seed(8)
    N = 300
    sd, st = torch.rand(1, N, generator=g), torch.rand(1, 1, N, generator=g)
    a, _ = ref.topk_select(sd, st, 50, 4, 8, 1, 2)
    b, _ = ref.topk_select(sd * 4.0, st * 0.125, 50, 4, 8, 1, 2)                  # reading A7
    assert torch.equal(a, b)
    # k >= N selects everything (A12)
    idx, cnt = ref.topk_select(sd, st, 400, 4, 8, 1, 2, k_max=400)
    assert cnt.item() == N and idx[0, 0, :N].tolist() == list(range(N)) and (idx[0, 0, N:] == -1).all()
    # ragged: per-sequence lengths and budgets
    sd2, st2 = torch.rand(2, N, generator=g), torch.rand(2, 2, N, generator=g)
    sl = torch.tensor([300, 120], dtype=torch.int32)
    bud = torch.tensor([40, 24], dtype=torch.int32)
    idx, cnt = ref.topk_select(sd2, st2, 0, 4, 8, 1, 2, k_max=40, seq_lens=sl, budgets=bud)
    assert cnt.tolist() == [[40, 40], [24, 24]]
    assert idx[1, :, :24].max() < 120 and (idx[1, :, 24:] == -1).all()
    assert set(range(112, 120)) <= set(idx[1, 0].tolist())                         # window follows N_b
    # S + W > k is an argument error
    with pytest.raises(ValueError):
        ref.topk_select(sd, st, 10, 4, 8, 1, 2)
    # N < S + W <= k: k >= N, everything is selected (A12)
    idx, cnt = ref.topk_select(torch.rand(1, 10), torch.rand(1, 1, 10), 14, 6, 8, 1, 2)
    assert cnt.item() == 10 and idx[0, 0, :10].tolist() == list(range(10))


def test_select_draft_list_stride_broadcast_vs_per_list():
    g = torch.Generator().manual_seed(21)
    N = 200
    sd = torch.rand(2, N, generator=g)
    st = torch.rand(2, 3, N, generator=g)
    a, _ = ref.topk_select(sd, st, 32, 4, 8, 1, 2)
    b, _ = ref.topk_select(sd.view(2, 1, N).expand(2, 3, N).contiguous(), st, 32, 4, 8, 1, 2)
    assert torch.equal(a, b)


def test_select_arr_maximal_for_target_only():
    """Eq. 1: with m = 0 the selected set maximises the recovered mass of S_tgt among all sets
    of that size that contain the protected set (exhaustive on a tiny case)."""
    g = torch.Generator().manual_seed(2)
    N, k, S, W = 10, 5, 1, 1
    st = torch.rand(1, 1, N, generator=g)
    idx, _ = ref.topk_select(torch.zeros(1, N), st, k, S, W, 0, 1)
    got = st[0, 0, idx[0, 0].long()].sum().item()
    best = max(st[0, 0, list(c) + [0, N - 1]].sum().item() for c in itertools.combinations(range(1, N - 1), k - 2))
    assert abs(got - best) < 1e-6


def test_config1_planted_heavy_hitters_selected():
    cfg = synth.config_tiny()
    L = synth.make_layer(cfg)
    kv = ref.KV.contiguous_nhd(L.k, L.v)
    a = ref.score_heads(kv, L.q[:, 0], cfg.head_mask, 1, 1, cfg.ctx)
    h = ref.fuse_scores(a, L.hist, 1.0)
    idx, cnt = ref.topk_select(L.s_draft, h, cfg.budget, cfg.n_sink, cfg.n_recent, 1, 2)
    assert cnt.item() == 128
    planted = L.planted[0, 0].nonzero().flatten().tolist()
    assert len(planted) == 8 and set(planted) <= set(idx[0, 0].tolist())


def test_eq7_overhead_ratio_printed_value():
    """PAPER.md:397 prints (4*3*4 + 4*1*1) / (14*24*4 + 64*80*1) = 52/6464 ~ 0.8 %  (tests/golden/eq7.txt)."""
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "eq7.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                key, val = line.split("=")
                vals[key.strip()] = float(val)
    num = vals["Hd_sel"] * vals["Ld_sel"] * vals["Gamma"] + vals["Ht_sel"] * vals["Lt_sel"] * 1
    den = vals["Hd"] * vals["Ld"] * vals["Gamma"] + vals["Ht"] * vals["Lt"] * 1
    assert num == vals["numerator"] and den == vals["denominator"]
    assert abs(100 * num / den - vals["percent"]) < 0.05
