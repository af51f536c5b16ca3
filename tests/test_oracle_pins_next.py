"""Pins of the oracle functions of the widened path: Attention Recovery Rate (Eq. 1-4),
KV append after verification and the draft-side lookahead aggregation (Eq. 5).
CPU only; every expected value comes from the paper's definitions, brute force or a torch fp64 library routine."""
import itertools
import math

import pytest
import torch

from oracle import ref


def bf16(*shape, seed=0, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return (torch.randn(*shape, generator=g) * scale).to(torch.bfloat16)


def full_lists(B, G, N, k_max=None):
    k_max = k_max or N
    idx = torch.full((B, G, k_max), -1, dtype=torch.int32)
    idx[:, :, :N] = torch.arange(N, dtype=torch.int32)
    return idx, torch.full((B, G), N, dtype=torch.int32)


# ---- O5: Attention Recovery Rate ------------------------------------------------------------------------------------
def test_arr_is_one_when_everything_is_selected_and_zero_for_the_empty_set():
    """PAPER.md:92 "an ARR of 1 means that the selected positions cover all attention mass"."""
    a = torch.rand(2, 3, 40, generator=torch.Generator().manual_seed(1))
    idx, cnt = full_lists(2, 3, 40)
    assert torch.allclose(ref.arr(a, idx, cnt), torch.ones(2, 3, dtype=torch.float64), atol=1e-12)
    assert torch.equal(ref.arr(a, idx, torch.zeros(2, 3, dtype=torch.int32)), torch.zeros(2, 3, dtype=torch.float64))


def test_arr_matches_eq1_by_hand_and_is_scale_invariant_and_additive():
    g = torch.Generator().manual_seed(2)
    a = torch.rand(1, 1, 12, generator=g)
    p = (a.double() / a.double().sum()).flatten()                     # Eq. 1: normalised over the valid positions
    k1, k2 = [0, 3, 7], [2, 11]
    def run(ks, aa=a):
        idx = torch.full((1, 1, 6), -1, dtype=torch.int32)
        idx[0, 0, :len(ks)] = torch.tensor(ks, dtype=torch.int32)
        return float(ref.arr(aa, idx, torch.tensor([[len(ks)]], dtype=torch.int32)))
    assert run(k1) == pytest.approx(float(sum(p[j] for j in k1)), abs=1e-12)
    assert run(k1 + k2) == pytest.approx(run(k1) + run(k2), abs=1e-12)   # disjoint sets add up
    assert run(k1, a * 7.5) == pytest.approx(run(k1), abs=1e-7)           # only the normalised weights matter
    assert 0.0 <= run(k2) <= 1.0


def test_topk_of_the_scores_maximises_arr_eq3_eq4():
    """Eq. 3-4: the top-k of the (window-averaged) attention is the ARR upper bound.  Brute force
    over every subset of that size on a tiny row."""
    g = torch.Generator().manual_seed(3)
    N, k = 9, 4
    a = torch.rand(1, 1, N, generator=g)
    idx, cnt = ref.topk_select(a[:, 0], a, k, 0, 0, 0, 1)             # m = 0, S = W = 0: plain TopK_k
    best = float(ref.arr(a, idx, cnt))
    for sub in itertools.combinations(range(N), k):
        i2 = torch.tensor(sub, dtype=torch.int32).view(1, 1, k)
        assert float(ref.arr(a, i2, torch.tensor([[k]], dtype=torch.int32))) <= best + 1e-12


def test_windowed_arr_eq2_equals_arr_of_the_window_mean():
    """Eq. 2 averages per-step ARRs; Eq. 3-4 evaluate the same set on the window mean A-bar: the two agree when every
    step's A is normalised (sum over V = 1)."""
    g = torch.Generator().manual_seed(4)
    w, N = 5, 30
    steps = torch.rand(w, 1, 1, N, generator=g)
    steps = (steps / steps.sum(-1, keepdim=True)).float()
    idx = torch.tensor([1, 4, 9, 16, 25], dtype=torch.int32).view(1, 1, 5)
    cnt = torch.tensor([[5]], dtype=torch.int32)
    per_step = sum(float(ref.arr(steps[s], idx, cnt)) for s in range(w)) / w
    a_bar = steps.double().mean(0).float()
    assert float(ref.arr(a_bar, idx, cnt)) == pytest.approx(per_step, abs=1e-6)
    assert float(ref.arr(steps.double().sum(0).float(), idx, cnt)) == pytest.approx(per_step, abs=1e-6)


def test_arr_ignores_positions_beyond_the_sequence_length():
    a = torch.ones(2, 1, 10)
    lens = torch.tensor([10, 4], dtype=torch.int32)
    idx = torch.tensor([[[0, 1]], [[0, 1]]], dtype=torch.int32)
    cnt = torch.tensor([[2], [2]], dtype=torch.int32)
    got = ref.arr(a, idx, cnt, lens)
    assert got[0, 0] == pytest.approx(0.2) and got[1, 0] == pytest.approx(0.5)


# ---- O6: KV append ----------------------------------------------------------------------------------------------------
def test_append_places_the_accepted_rows_behind_each_sequence_and_nothing_else():
    B, cap, Hkv, d, T = 3, 20, 2, 8, 4
    k, v = bf16(B, cap, Hkv, d, seed=5), bf16(B, cap, Hkv, d, seed=6)
    kn, vn = bf16(B, T, Hkv, d, seed=7), bf16(B, T, Hkv, d, seed=8)
    lens = torch.tensor([5, 18, 0], dtype=torch.int32)
    na = torch.tensor([3, 4, 0], dtype=torch.int32)                    # sequence 1 only has room for 2 more rows
    hist = torch.full((B, 2, cap), 9.0)
    k0, v0 = k.clone(), v.clone()
    new_lens = ref.append_kv(ref.KV.contiguous_nhd(k, v), lens, kn, vn, na, cap, hist)
    assert new_lens.tolist() == [8, 20, 0]
    for b, (n0, a) in enumerate([(5, 3), (18, 2), (0, 0)]):
        assert torch.equal(k[b, n0:n0 + a], kn[b, :a]) and torch.equal(v[b, n0:n0 + a], vn[b, :a])
        keep = torch.ones(cap, dtype=torch.bool)
        keep[n0:n0 + a] = False
        assert torch.equal(k[b, keep], k0[b, keep]) and torch.equal(v[b, keep], v0[b, keep])
        assert torch.all(hist[b, :, n0:n0 + a] == 0) and torch.all(hist[b][:, keep] == 9.0)


def test_append_then_dense_attention_equals_attention_with_the_rows_still_in_the_block():
    """Pins the placement against O4: verify position a of the block [r_0..r_a] over the old cache sees
    exactly what a one-row block r_a sees over the cache with r_0..r_{a-1} appended."""
    B, N, cap, Hq, Hkv, d, a = 2, 11, 16, 4, 2, 16, 3
    k, v = bf16(B, cap, Hkv, d, seed=9), bf16(B, cap, Hkv, d, seed=10)
    q, kn, vn = bf16(B, a + 1, Hq, d, seed=11), bf16(B, a + 1, Hkv, d, seed=12), bf16(B, a + 1, Hkv, d, seed=13)
    lens = torch.full((B,), N, dtype=torch.int32)
    before, _ = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k, v, lens), q, kn, vn, None, None, cap)
    new_lens = ref.append_kv(ref.KV.contiguous_nhd(k, v), lens, kn, vn, torch.full((B,), a, dtype=torch.int32), cap)
    after, _ = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k, v, new_lens), q[:, a:].contiguous(),
                                      kn[:, a:].contiguous(), vn[:, a:].contiguous(), None, None, cap)
    assert torch.allclose(after[:, 0], before[:, a], atol=1e-12)


def test_append_paged_equals_contiguous():
    B, cap, Hkv, d, T, page = 2, 32, 2, 8, 3, 4
    k, v = bf16(B, cap, Hkv, d, seed=14), bf16(B, cap, Hkv, d, seed=15)
    kn, vn = bf16(B, T, Hkv, d, seed=16), bf16(B, T, Hkv, d, seed=17)
    lens = torch.tensor([7, 13], dtype=torch.int32)
    na = torch.tensor([3, 2], dtype=torch.int32)
    n_pages = B * cap // page
    perm = torch.randperm(n_pages, generator=torch.Generator().manual_seed(18)).to(torch.int32)
    table = perm.view(B, cap // page).contiguous()
    kp, vp = torch.zeros(n_pages, page, Hkv, d, dtype=torch.bfloat16), torch.zeros(n_pages, page, Hkv, d, dtype=torch.bfloat16)
    for b in range(B):
        for pg in range(cap // page):
            kp[table[b, pg]] = k[b, pg * page:(pg + 1) * page]
            vp[table[b, pg]] = v[b, pg * page:(pg + 1) * page]
    ref.append_kv(ref.KV.contiguous_nhd(k, v), lens, kn, vn, na, cap)
    paged = ref.KV(kp, vp, page * Hkv * d, Hkv * d, d, table, page)
    ref.append_kv(paged, lens, kn, vn, na, cap)
    for b in range(B):
        for pg in range(cap // page):
            assert torch.equal(kp[table[b, pg]], k[b, pg * page:(pg + 1) * page])
            assert torch.equal(vp[table[b, pg]], v[b, pg * page:(pg + 1) * page])


# ---- O7: draft-side lookahead aggregation -----------------------------------------------------------------------------
def draft_case(seed, B=2, N=24, Hq=4, Hkv=2, d=16, gamma=3, L=2):
    ks = [bf16(B, N, Hkv, d, seed=seed + l) for l in range(L)]
    qs = [bf16(B, gamma, Hq, d, seed=seed + 50 + l) for l in range(L)]
    return ks, qs


def test_draft_aggregate_matches_torch_softmax_summed_over_heads_layers_and_lookahead_tokens():
    """Eq. 5: S_Draft[n] = sum_{h,l,gamma} A^Draft; library cross-check in fp64."""
    B, N, Hq, Hkv, d, gamma, L = 2, 24, 4, 2, 16, 3, 2
    ks, qs = draft_case(20, B, N, Hq, Hkv, d, gamma, L)
    mask = 0b1011
    lens = torch.tensor([24, 17], dtype=torch.int32)
    got = ref.draft_aggregate(ks, qs, mask, Hkv, N, N * Hkv * d, Hkv * d, d, seq_lens=lens)
    want = torch.zeros(B, N, dtype=torch.float64)
    for b in range(B):
        n_b = int(lens[b])
        for l in range(L):
            for h in range(Hq):
                if not (mask >> h) & 1:
                    continue
                logits = qs[l][b, :, h].double() @ ks[l][b, :n_b, h // (Hq // Hkv)].double().T / math.sqrt(d)
                want[b, :n_b] += torch.softmax(logits, dim=-1).sum(0)
    assert torch.allclose(got.double(), want, rtol=1e-6, atol=1e-9)
    assert torch.all(got[1, 17:] == 0)


def test_draft_aggregate_mass_counts_the_terms_of_eq5_and_zero_keys_give_the_uniform_row():
    B, N, Hq, Hkv, d, gamma, L = 1, 16, 4, 1, 8, 4, 3
    ks, qs = draft_case(30, B, N, Hq, Hkv, d, gamma, L)
    got = ref.draft_aggregate(ks, qs, 0b0110, Hkv, N, N * Hkv * d, Hkv * d, d)
    assert float(got.sum()) == pytest.approx(2 * L * gamma, rel=1e-6)          # every softmax row sums to 1
    zero = [torch.zeros_like(k) for k in ks]
    got0 = ref.draft_aggregate(zero, qs, 0b0110, Hkv, N, N * Hkv * d, Hkv * d, d)
    assert torch.allclose(got0, torch.full((B, N), 2 * L * gamma / N), rtol=1e-6)


def test_draft_aggregate_is_the_sum_of_single_query_scorings():
    """Consistency with O1 (itself pinned in test_oracle_pins.py): one scoring call per (layer, lookahead token)."""
    B, N, Hq, Hkv, d, gamma, L = 2, 20, 4, 2, 16, 2, 2
    ks, qs = draft_case(40, B, N, Hq, Hkv, d, gamma, L)
    got = ref.draft_aggregate(ks, qs, 0b1111, Hkv, N, N * Hkv * d, Hkv * d, d)
    acc = torch.zeros(B, N, dtype=torch.float64)
    for l in range(L):
        for gam in range(gamma):
            acc += ref.score_heads(ref.KV.contiguous_nhd(ks[l], None), qs[l][:, gam], 0b1111, 1, Hkv, N)[:, 0].double()
    assert torch.allclose(got.double(), acc, rtol=1e-6, atol=1e-9)
