"""Pins of the oracle's verification attention (App. G :568; reading A13) -- SURVEY.md §8c O4 -- and of
the paged view.  CPU only."""
import math

import pytest
import torch

from oracle import ref
from tests.test_oracle_pins import bf16, rand_case


def brute_attn(q, k, v, kn, vn, idx, cnt):
    """Independent pure-Python loops: visible set = selected cache rows + new rows u <= t."""
    B, T, Hq, d = q.shape
    Hkv = k.shape[2]
    r = Hq // Hkv
    out = torch.zeros(B, T, Hq, d, dtype=torch.float64)
    lse = torch.zeros(B, Hq, T, dtype=torch.float64)
    qd, kd, vd, knd, vnd = (x.double() for x in (q, k, v, kn, vn))
    for b in range(B):
        for h in range(Hq):
            g = h // r
            l = 0 if idx.shape[1] == 1 else g
            rows = idx[b, l, :cnt[b, l]].tolist()
            for t in range(T):
                keys = [kd[b, n, g] for n in rows] + [knd[b, u, g] for u in range(t + 1)]
                vals = [vd[b, n, g] for n in rows] + [vnd[b, u, g] for u in range(t + 1)]
                lg = [float((qd[b, t, h] * kk).sum()) / math.sqrt(d) for kk in keys]
                mx = max(lg)
                ex = [math.exp(x - mx) for x in lg]
                z = sum(ex)
                acc = torch.zeros(d, dtype=torch.float64)
                for e, vv in zip(ex, vals):
                    acc += (e / z) * vv
                out[b, t, h] = acc
                lse[b, h, t] = mx + math.log(z)
    return out, lse


def full_idx(B, G, N):
    idx = torch.arange(N, dtype=torch.int32).view(1, 1, N).expand(B, G, N).contiguous()
    return idx, torch.full((B, G), N, dtype=torch.int32)


@pytest.mark.parametrize("G", [1, 2])
def test_attn_brute_force_sparse(G):
    q, k, v, kn, vn = rand_case(B=2, N=23, Hq=4, Hkv=2, d=8, T=3, seed=13)
    g = torch.Generator().manual_seed(1)
    kk = 9
    idx = torch.stack([torch.stack([torch.randperm(23, generator=g)[:kk].sort().values for _ in range(G)])
                       for _ in range(2)]).to(torch.int32)
    cnt = torch.tensor([[kk] * G, [kk - 2] * G], dtype=torch.int32)
    idx[1, :, kk - 2:] = -1
    out, lse = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k, v), q, kn, vn, idx, cnt, 23)
    want, want_lse = brute_attn(q, k, v, kn, vn, idx, cnt)
    assert torch.allclose(out, want, rtol=1e-12, atol=1e-13)
    assert torch.allclose(lse, want_lse, rtol=1e-12, atol=1e-13)


def test_attn_budget_equals_context_is_dense_and_matches_sdpa():
    """k = N reproduces dense attention exactly (north_star invariant); the dense case equals torch SDPA in fp64
    with the explicit causal-among-new-tokens mask (library routine, test-only)."""
    B, N, Hq, Hkv, d, T = 2, 77, 6, 2, 32, 4
    q, k, v, kn, vn = rand_case(B, N, Hq, Hkv, d, T, seed=7)
    kv = ref.KV.contiguous_nhd(k, v)
    dense, lse_d = ref.sparse_verify_attn(kv, q, kn, vn, None, None, N)
    idx, cnt = full_idx(B, Hkv, N)
    sparse, lse_s = ref.sparse_verify_attn(kv, q, kn, vn, idx, cnt, N)
    assert torch.equal(dense, sparse) and torch.equal(lse_d, lse_s)
    r = Hq // Hkv
    kall = torch.cat([k, kn], 1).double().repeat_interleave(r, dim=2).permute(0, 2, 1, 3)    # [B,Hq,N+T,d]
    vall = torch.cat([v, vn], 1).double().repeat_interleave(r, dim=2).permute(0, 2, 1, 3)
    mask = torch.ones(T, N + T, dtype=torch.bool)
    mask[:, N:] = torch.tril(torch.ones(T, T, dtype=torch.bool))
    want = torch.nn.functional.scaled_dot_product_attention(q.double().permute(0, 2, 1, 3), kall, vall, attn_mask=mask)
    assert torch.allclose(dense, want.permute(0, 2, 1, 3), rtol=1e-10, atol=1e-12)
    # LSE against torch.logsumexp
    lg = torch.einsum("bthc,bhnc->bhtn", q.double(), kall) / math.sqrt(d)
    lg = lg.masked_fill(~mask.view(1, 1, T, N + T), float("-inf"))
    assert torch.allclose(lse_d, torch.logsumexp(lg, -1), rtol=1e-12)


def test_attn_constant_v_and_zero_k_closed_forms():
    B, N, Hq, Hkv, d, T = 1, 40, 2, 1, 16, 3
    q, k, v, kn, vn = rand_case(B, N, Hq, Hkv, d, T, seed=2)
    idx = torch.tensor([[[1, 5, 6, 30, -1]]], dtype=torch.int32)
    cnt = torch.tensor([[4]], dtype=torch.int32)
    c = bf16(torch.randn(d))
    vc, vnc = c.expand(B, N, Hkv, d).contiguous(), c.expand(B, T, Hkv, d).contiguous()
    out, _ = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k, vc), q, kn, vnc, idx, cnt, N)
    assert torch.allclose(out, c.double().expand_as(out), rtol=1e-13, atol=1e-15)        # probabilities sum to 1
    # K == 0 (cache and new): uniform weights => plain mean of the cnt + t + 1 visible V rows
    out, lse = ref.sparse_verify_attn(ref.KV.contiguous_nhd(torch.zeros_like(k), v), q, torch.zeros_like(kn), vn,
                                      idx, cnt, N)
    for t in range(T):
        rows = torch.cat([v[0, [1, 5, 6, 30], 0].double(), vn[0, :t + 1, 0].double()])
        assert torch.allclose(out[0, t, 0], rows.mean(0), rtol=1e-13, atol=1e-15)
        assert abs(lse[0, 0, t].item() - math.log(4 + t + 1)) < 1e-13


def test_attn_causality_among_new_tokens_and_index_order():
    B, N, Hq, Hkv, d, T = 1, 30, 2, 1, 16, 4
    q, k, v, kn, vn = rand_case(B, N, Hq, Hkv, d, T, seed=4)
    idx = torch.tensor([[[2, 3, 11, 20, 29]]], dtype=torch.int32)
    cnt = torch.tensor([[5]], dtype=torch.int32)
    kv = ref.KV.contiguous_nhd(k, v)
    base, _ = ref.sparse_verify_attn(kv, q, kn, vn, idx, cnt, N)
    kn2, vn2 = kn.clone(), vn.clone()
    kn2[:, 2:] += 1.0
    vn2[:, 2:] -= 2.0
    pert, _ = ref.sparse_verify_attn(kv, q, kn2, vn2, idx, cnt, N)
    assert torch.equal(base[:, :2], pert[:, :2]) and not torch.equal(base[:, 2:], pert[:, 2:])
    # self is visible: with a huge self-aligned key the output of row t tends to v_new[t]
    kn3 = kn.clone()
    kn3[0, 1, 0] = q[0, 1, 0] * 64
    out, _ = ref.sparse_verify_attn(kv, q, kn3, vn, idx, cnt, N)
    assert torch.allclose(out[0, 1, 0], vn[0, 1, 0].double(), atol=1e-6)
    # order of the index list does not matter
    shuf = torch.tensor([[[29, 2, 20, 11, 3]]], dtype=torch.int32)
    out2, _ = ref.sparse_verify_attn(kv, q, kn, vn, shuf, cnt, N)
    assert torch.allclose(base, out2, rtol=1e-12, atol=1e-14)


def test_gqa_head_to_group_mapping():
    """g = h div r (reading A2): head h must read KV head h // r, not h % Hkv."""
    B, N, Hq, Hkv, d, T = 1, 10, 4, 2, 8, 1
    q, k, v, kn, vn = rand_case(B, N, Hq, Hkv, d, T, seed=6)
    v2 = v.clone()
    v2[:, :, 1] += 3.0                                       # touch KV head 1 only -> heads 2,3 change, 0,1 do not
    a, _ = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k, v), q, kn, vn, None, None, N)
    b, _ = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k, v2), q, kn, vn, None, None, N)
    assert torch.equal(a[:, :, :2], b[:, :, :2]) and not torch.allclose(a[:, :, 2:], b[:, :, 2:])


def test_paged_equals_contiguous():
    B, N, Hq, Hkv, d, T, ps = 2, 70, 4, 2, 16, 2, 16
    q, k, v, kn, vn = rand_case(B, N, Hq, Hkv, d, T, seed=12)
    sl = torch.tensor([70, 45], dtype=torch.int32)
    max_pages = (N + ps - 1) // ps
    perm = torch.randperm(B * max_pages, generator=torch.Generator().manual_seed(3)).to(torch.int32)
    pt = perm.view(B, max_pages).contiguous()
    kp = torch.zeros(B * max_pages, ps, Hkv, d, dtype=torch.bfloat16)
    vp = torch.zeros_like(kp)
    for b in range(B):
        for n in range(N):
            kp[pt[b, n // ps], n % ps] = k[b, n]
            vp[pt[b, n // ps], n % ps] = v[b, n]
    kvc = ref.KV.contiguous_nhd(k, v, seq_lens=sl)
    kvp = ref.KV(kp, vp, ps * Hkv * d, Hkv * d, d, pt, ps, sl)
    a = ref.score_heads(kvc, q[:, 0], 0b1001, 2, Hkv, N)
    b_ = ref.score_heads(kvp, q[:, 0], 0b1001, 2, Hkv, N)
    assert torch.equal(a, b_)
    idx, cnt = ref.topk_select(torch.rand(B, N), a, 24, 2, 4, 1, 2, seq_lens=sl)
    oc, _ = ref.sparse_verify_attn(kvc, q, kn, vn, idx, cnt, N)
    op, _ = ref.sparse_verify_attn(kvp, q, kn, vn, idx, cnt, N)
    assert torch.equal(oc, op)
    dc, _ = ref.sparse_verify_attn(kvc, q, kn, vn, None, None, N)
    dp, _ = ref.sparse_verify_attn(kvp, q, kn, vn, None, None, N)
    assert torch.equal(dc, dp)
