"""Pins of the CPU oracle (oracle/dustin_ref.cpp) against things OTHER than itself (SURVEY.md §8c "what pins each
part"): brute force written independently in pure Python on tiny inputs, closed forms, invariants, special cases
that reduce to a library routine (torch fp64 softmax / SDPA / sort), and the one value PAPER.md prints (Eq. 7).
CPU only; none of these tests touches the CUDA path.
"""
import itertools
import math

import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import synth


def bf16(t):
    return t.to(torch.bfloat16)


def rand_case(B=2, N=37, Hq=4, Hkv=2, d=16, T=3, seed=0):
    g = torch.Generator().manual_seed(seed)
    q = bf16(torch.randn(B, T, Hq, d, generator=g))
    k = bf16(torch.randn(B, N, Hkv, d, generator=g))
    v = bf16(torch.randn(B, N, Hkv, d, generator=g))
    kn = bf16(torch.randn(B, T, Hkv, d, generator=g))
    vn = bf16(torch.randn(B, T, Hkv, d, generator=g))
    return q, k, v, kn, vn


# ----------------------------------------------------------------------------------------------------------------
# O1 scoring  (readings A2-A5)
# ----------------------------------------------------------------------------------------------------------------
def brute_scores(q0, k, heads, n_lists):
    """Independent pure-Python triple loop.  q0 [B,Hq,d], k [B,N,Hkv,d] (python floats via .double())."""
    B, Hq, d = q0.shape
    N, Hkv = k.shape[1], k.shape[2]
    r = Hq // Hkv
    out = [[[0.0] * N for _ in range(n_lists)] for _ in range(B)]
    qd, kd = q0.double().tolist(), k.double().tolist()
    for b in range(B):
        per_head = {}
        for h in heads:
            g = h // r
            lg = [sum(qd[b][h][c] * kd[b][n][g][c] for c in range(d)) / math.sqrt(d) for n in range(N)]
            mx = max(lg)
            ex = [math.exp(x - mx) for x in lg]
            z = sum(ex)
            per_head[h] = [e / z for e in ex]
        for l in range(n_lists):
            if n_lists == 1:
                hs = list(heads)
            else:
                hs = [h for h in heads if h // r == l] or list(heads)      # empty group -> global sum (A2)
            for n in range(N):
                out[b][l][n] = sum(per_head[h][n] for h in hs)
    return torch.tensor(out, dtype=torch.float64)


@pytest.mark.parametrize("n_lists,heads", [(1, (0, 3)), (2, (0, 1)), (2, (1, 2, 3)), (1, (2,))])
def test_score_brute_force(n_lists, heads):
    q, k, v, _, _ = rand_case(B=2, N=13, Hq=4, Hkv=2, d=8, T=1, seed=3)
    cfg_mask = sum(1 << h for h in heads)
    got = ref.score_heads(ref.KV.contiguous_nhd(k, v), q[:, 0], cfg_mask, n_lists, 2, 13)
    want = brute_scores(q[:, 0], k, heads, n_lists)
    assert torch.allclose(got.double(), want, rtol=2e-7, atol=1e-9)


def test_score_rows_sum_to_head_count():
    q, k, v, _, _ = rand_case(B=3, N=301, Hq=8, Hkv=4, d=32, T=1, seed=5)
    heads = (0, 1, 5)                                  # groups 0,0,2 ; groups 1 and 3 empty -> global sum
    a = ref.score_heads(ref.KV.contiguous_nhd(k, v), q[:, 0], sum(1 << h for h in heads), 4, 4, 301)
    sums = a.double().sum(-1)
    want = torch.tensor([2.0, 3.0, 1.0, 3.0]).expand(3, 4)
    assert torch.allclose(sums, want.double(), atol=1e-5)
    a1 = ref.score_heads(ref.KV.contiguous_nhd(k, v), q[:, 0], sum(1 << h for h in heads), 1, 4, 301)
    assert torch.allclose(a1.double().sum(-1), torch.full((3, 1), 3.0, dtype=torch.float64), atol=1e-5)
    assert (a >= 0).all()


def test_score_zero_keys_uniform():
    q, k, v, _, _ = rand_case(B=1, N=50, Hq=2, Hkv=1, d=8, T=1)
    a = ref.score_heads(ref.KV.contiguous_nhd(torch.zeros_like(k), v), q[:, 0], 0b11, 1, 1, 50)
    assert torch.equal(a, torch.full_like(a, float(2.0 / 50)))     # 2 heads * 1/N, exactly representable sum


def test_score_one_planted_key_closed_form():
    # K all zero except K[n*] = c * q_hat  =>  p[n*] = e^{c |q| / sqrt(d)} / (e^{...} + N - 1)
    d, N, nstar = 16, 64, 17
    q = torch.zeros(1, 1, 1, d)
    q[..., 0] = 3.0                                      # |q| = 3, exactly representable in bf16
    k = torch.zeros(1, N, 1, d)
    k[0, nstar, 0, 0] = 2.0                              # c = 2 along q_hat
    a = ref.score_heads(ref.KV.contiguous_nhd(bf16(k), bf16(k)), bf16(q)[:, 0], 1, 1, 1, N).double()
    e = math.exp(2.0 * 3.0 / math.sqrt(d))
    assert abs(a[0, 0, nstar].item() - e / (e + N - 1)) < 1e-7
    assert abs(a[0, 0, 0].item() - 1.0 / (e + N - 1)) < 1e-8


def test_score_permutation_equivariance_and_torch_softmax():
    q, k, v, _, _ = rand_case(B=2, N=200, Hq=4, Hkv=2, d=64, T=1, seed=9)
    kv = ref.KV.contiguous_nhd(k, v)
    a = ref.score_heads(kv, q[:, 0], 0b0101, 2, 2, 200)
    perm = torch.randperm(200, generator=torch.Generator().manual_seed(1))
    kp = k[:, perm].contiguous()
    ap = ref.score_heads(ref.KV.contiguous_nhd(kp, v), q[:, 0], 0b0101, 2, 2, 200)
    assert torch.allclose(ap, a[:, :, perm], rtol=1e-6, atol=0)
    # library cross-check (test-only): heads 0 and 2 sit in KV groups 0 and 1
    for l, h in ((0, 0), (1, 2)):
        lg = torch.einsum("bc,bnc->bn", q[:, 0, h].double(), k[:, :, l].double()) / math.sqrt(64)
        assert torch.allclose(a[:, l].double(), torch.softmax(lg, -1), rtol=2e-7, atol=1e-12)


def test_score_sm_scale_and_strided_query_and_seq_lens():
    q, k, v, _, _ = rand_case(B=2, N=40, Hq=2, Hkv=1, d=8, T=3, seed=2)
    kv = ref.KV.contiguous_nhd(k, v, seq_lens=torch.tensor([40, 25], dtype=torch.int32))
    a = ref.score_heads(kv, q[:, 1], 0b01, 1, 1, 40, sm_scale=0.25)           # strided view, position 1
    assert (a[1, 0, 25:] == 0).all()
    lg = torch.einsum("c,nc->n", q[1, 1, 0].double(), k[1, :25, 0].double()) * 0.25
    assert torch.allclose(a[1, 0, :25].double(), torch.softmax(lg, -1), rtol=2e-7)


# ----------------------------------------------------------------------------------------------------------------
# O2 fusion  (Eq. 5; reading A6)
# ----------------------------------------------------------------------------------------------------------------
def test_fuse_closed_forms():
    g = torch.Generator().manual_seed(0)
    a = torch.rand(2, 3, 17, generator=g)
    h = torch.rand(2, 3, 17, generator=g)
    assert torch.equal(ref.fuse_scores(a, h, 0.0), a)                         # alpha = 0: delta = 1 policy (:104)
    assert torch.equal(ref.fuse_scores(a, h, 1.0), (a.double() + h.double()).float())
    assert torch.equal(ref.fuse_scores(a, h, 0.5), (0.5 * h.double() + a.double()).float())
    # L calls with alpha = 1 == plain sum of L terms (Eq. 5 sums over layers)
    terms = [torch.rand(1, 1, 9, generator=g) for _ in range(5)]
    acc = torch.zeros(1, 1, 9)
    for t in terms:
        acc = ref.fuse_scores(t, acc, 1.0)
    assert torch.allclose(acc.double(), sum(t.double() for t in terms), rtol=1e-6)
    # entries past seq_len are untouched
    sl = torch.tensor([5, 17], dtype=torch.int32)
    out = ref.fuse_scores(a, h, 1.0, seq_lens=sl)
    assert torch.equal(out[0, :, 5:], h[0, :, 5:])
