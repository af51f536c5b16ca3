"""Pins of the oracle's Quest-16 estimator (O8 page min/max metadata, O9 page scores; PAPER.md:51, :297-299, :401;
DESIGN.md readings A20 / A21) against things other than itself: pure-Python brute force on tiny pages, the bound
property that defines the estimate (a page's upper bound is never below an exact logit of a token inside it, with
equality when the page holds one distinct key), closed forms for sign-definite queries, and the special case page
size 1, where the estimator must reduce to the exact head-subset scores of O1 (itself pinned in test_oracle_pins.py)."""
import math

import torch

from oracle import ref


def _case(B=2, N=50, Hq=4, Hkv=2, d=8, seed=0, ragged=False):
    g = torch.Generator().manual_seed(seed)
    k = torch.randn(B, N, Hkv, d, generator=g).to(torch.bfloat16)
    q = torch.randn(B, Hq, d, generator=g).to(torch.bfloat16)
    lens = torch.tensor([N - 7 * b - 3 for b in range(B)], dtype=torch.int32) if ragged else None
    return k, q, lens


def test_page_minmax_brute_force_and_empty_pages():
    k, q, lens = _case(B=2, N=37, ragged=True)          # lengths 34 and 27: ragged last pages, one empty page for b = 1
    P = 5
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, lens), 2, 37, P)
    assert kmin.shape == (2, 8, 2, 8)
    for b in range(2):
        n_b = int(lens[b])
        for p in range(8):
            toks = [n for n in range(p * P, (p + 1) * P) if n < n_b]
            for g in range(2):
                for c in range(8):
                    vals = [float(k[b, n, g, c]) for n in toks]
                    lo, hi = (min(vals), max(vals)) if vals else (0.0, 0.0)
                    assert kmin[b, p, g, c].item() == lo and kmax[b, p, g, c].item() == hi
    assert int(lens[1]) == 27 and (kmin[1, 6:] == 0).all() and (kmax[1, 6:] == 0).all()


def test_page_minmax_is_layout_independent_paged_equals_contiguous():
    k, q, lens = _case(B=2, N=48, ragged=True, seed=3)
    ps, Hkv, d = 4, 2, 8
    n_phys = 2 * 12
    perm = torch.randperm(n_phys, generator=torch.Generator().manual_seed(9)).to(torch.int32)
    table = perm.view(2, 12).contiguous()
    pool = torch.zeros(n_phys, ps, Hkv, d, dtype=torch.bfloat16)
    for b in range(2):
        for lp in range(12):
            pool[int(table[b, lp])] = k[b, lp * ps:(lp + 1) * ps]
    a = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, lens), Hkv, 48, 16)
    paged = ref.KV(pool, None, ps * Hkv * d, Hkv * d, d, table, ps, lens)
    b_ = ref.quest_page_minmax(paged, Hkv, 48, 16)
    assert torch.equal(a[0], b_[0]) and torch.equal(a[1], b_[1])


def test_upper_bound_brute_force_python():
    k, q, lens = _case(B=1, N=23, Hq=4, Hkv=2, d=8, seed=5)
    P, scale = 4, 0.375          # exactly representable in the float the ABI carries
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, None), 2, 23, P)
    mask = 0b1011
    scores, ub = ref.quest_score_pages(kmin, kmax, q, mask, 1, 23, P, None, scale, want_ub=True)
    n_pages = 6
    tot = [0.0] * n_pages
    for h in range(4):
        if not (mask >> h) & 1:
            assert (ub[0, h] == 0).all()
            continue
        g = h // 2
        U = []
        for p in range(n_pages):
            toks = range(p * P, min((p + 1) * P, 23))
            acc = 0.0
            for c in range(8):
                qc = float(q[0, h, c])
                lo = min(float(k[0, n, g, c]) for n in toks)
                hi = max(float(k[0, n, g, c]) for n in toks)
                acc += max(qc * lo, qc * hi)
            U.append(acc * scale)
            assert abs(ub[0, h, p].item() - U[p]) <= 1e-12 * max(1.0, abs(U[p]))
        M = max(U)
        Z = sum(math.exp(u - M) for u in U)
        for p in range(n_pages):
            tot[p] += math.exp(U[p] - M) / Z
    for p in range(n_pages):
        assert abs(scores[0, 0, p].item() - tot[p]) <= 1e-6 * tot[p] + 1e-12
    assert abs(scores[0, 0].double().sum().item() - 3.0) < 1e-5          # three subset heads, each a distribution


def test_bound_property_no_exact_logit_above_its_pages_bound():
    k, q, lens = _case(B=2, N=200, Hq=8, Hkv=2, d=16, seed=11, ragged=True)
    P = 16
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, lens), 2, 200, P)
    _, ub = ref.quest_score_pages(kmin, kmax, q, 0xFF, 2, 200, P, lens, 0.0, want_ub=True)
    scale = 1.0 / math.sqrt(16)
    kd, qd = k.double(), q.double()
    tight = 0
    for b in range(2):
        for h in range(8):
            logits = (kd[b, :, h // 4, :] @ qd[b, h]) * scale                     # exact, by a library matmul
            for n in range(int(lens[b])):
                assert logits[n].item() <= ub[b, h, n // P].item() + 1e-12
            # the bound is not vacuous: it stays within the spread of the page's keys
            page_max = torch.stack([logits[p * P:min((p + 1) * P, int(lens[b]))].max()
                                    for p in range((int(lens[b]) + P - 1) // P)])
            tight += int((ub[b, h, :page_max.numel()] - page_max < 8.0).all())
    assert tight == 16


def test_single_key_pages_and_sign_definite_queries_closed_forms():
    B, N, Hkv, d, P = 1, 32, 1, 8, 8
    g = torch.Generator().manual_seed(2)
    base = torch.randn(B, N // P, Hkv, d, generator=g).to(torch.bfloat16)
    k = base.repeat_interleave(P, dim=1)                 # every page holds ONE distinct key: the bound is exact
    q = torch.randn(B, 2, d, generator=g).to(torch.bfloat16)
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, None), Hkv, N, P)
    assert torch.equal(kmin, kmax)
    _, ub = ref.quest_score_pages(kmin, kmax, q, 0b11, 1, N, P, None, 1.0, want_ub=True)
    exact = torch.einsum("bphc,bqc->bqp", base.double(), q.double())
    assert torch.allclose(ub, exact, rtol=0, atol=1e-12)
    # q >= 0: the bound is q . kmax;  q <= 0: q . kmin
    k2 = torch.randn(B, N, Hkv, d, generator=g).to(torch.bfloat16)
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k2, None, None), Hkv, N, P)
    qpos = q.abs()
    qq = torch.stack([qpos[:, 0], -qpos[:, 1]], dim=1).contiguous()
    _, ub = ref.quest_score_pages(kmin, kmax, qq, 0b11, 1, N, P, None, 1.0, want_ub=True)
    assert torch.allclose(ub[0, 0], kmax[0, :, 0].double() @ qq[0, 0].double(), atol=1e-12, rtol=0)
    assert torch.allclose(ub[0, 1], kmin[0, :, 0].double() @ qq[0, 1].double(), atol=1e-12, rtol=0)


def test_page_size_one_reduces_to_the_exact_head_subset_scores():
    """P = 1: min = max = the key itself, so the page score is O1's exact attention probability (both list modes,
    an empty KV group included, ragged lengths)."""
    k, q, lens = _case(B=2, N=61, Hq=8, Hkv=4, d=16, seed=21, ragged=True)
    kv = ref.KV.contiguous_nhd(k, None, lens)
    kmin, kmax = ref.quest_page_minmax(kv, 4, 61, 1)
    mask = 0b00110101                                   # groups 0, 1, 2 scored; group 3 empty (reading A2)
    for n_lists in (1, 4):
        got = ref.quest_score_pages(kmin, kmax, q, mask, n_lists, 61, 1, lens, 0.0)
        want = ref.score_heads(kv, q, mask, n_lists, 4, 61, 0.0)
        assert torch.allclose(got.double(), want.double(), rtol=1e-6, atol=1e-12)
        for b in range(2):
            assert (got[b, :, int(lens[b]):] == 0).all()


def test_uniform_when_all_pages_alike_and_row_sums():
    B, N, P = 1, 64, 16
    k = torch.ones(B, N, 1, 8).to(torch.bfloat16)
    q = torch.randn(B, 2, 8, generator=torch.Generator().manual_seed(4)).to(torch.bfloat16)
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, None), 1, N, P)
    s = ref.quest_score_pages(kmin, kmax, q, 0b11, 1, N, P)
    assert torch.allclose(s, torch.full_like(s, 2.0 / 4))           # two heads, four identical pages
    lens = torch.tensor([40], dtype=torch.int32)                    # three live pages
    kmin, kmax = ref.quest_page_minmax(ref.KV.contiguous_nhd(k, None, lens), 1, N, P)
    s = ref.quest_score_pages(kmin, kmax, q, 0b11, 1, N, P, lens)
    assert torch.allclose(s[0, 0, :3], torch.full((3,), 2.0 / 3)) and s[0, 0, 3] == 0
