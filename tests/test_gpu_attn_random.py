"""Randomised GPU parity of stage a4 / a5 (dustin_sparse_verify_attn) against the oracle: seeded random shapes, list
lengths, layouts (contiguous, ragged, paged with a shuffled page table), one list per sequence or per KV head, dense and
gathered -- the corners of the tcgen05 kernel's planning (whole units, cut units, cuts near new-row tiles, empty
lists, every row-count instantiation) are reached by construction of the ranges, not by hand-picked cases."""
import random

import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import api
from tests import harness as H

pytestmark = pytest.mark.gpu


def _case(seed: int):
    rnd = random.Random(1000 + seed)
    g = torch.Generator().manual_seed(5000 + seed)
    Hkv = rnd.choice([1, 2, 4, 8])
    r = rnd.choice([1, 2, 4, 8])
    T = rnd.randint(1, min(16, 96 // r))
    B = rnd.randint(1, 6)
    N = rnd.choice([64, 200, 777, 1500, 3000])
    d = 128
    mode = rnd.choice(["sparse", "sparse", "dense", "paged", "paged_dense"])
    ragged = mode != "sparse" or rnd.random() < 0.5
    bf = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16)
    q, k_new, v_new = bf(B, T, Hkv * r, d), bf(B, T, Hkv, d), bf(B, T, Hkv, d)
    lens = torch.tensor([rnd.randint(1, N) if ragged else N for _ in range(B)], dtype=torch.int32)
    if mode.startswith("paged"):
        page = rnd.choice([8, 16, 32])
        max_pages = (N + page - 1) // page
        n_pages = B * max_pages + 3
        perm = torch.randperm(n_pages, generator=g)[:B * max_pages].to(torch.int32).view(B, max_pages).contiguous()
        k, v = bf(n_pages, page, Hkv, d), bf(n_pages, page, Hkv, d)
        kv_gpu = lambda: api.KV.paged_nhd(k.cuda(), v.cuda(), perm.cuda(), lens.cuda())
        kv_cpu = ref.KV(k, v, page * Hkv * d, Hkv * d, d, perm, page, lens)
    else:
        k, v = bf(B, N, Hkv, d), bf(B, N, Hkv, d)
        sl = lens if ragged else None
        kv_gpu = lambda: api.KV.contiguous_nhd(k.cuda(), v.cuda(), None if sl is None else sl.cuda())
        kv_cpu = ref.KV.contiguous_nhd(k, v, sl)
    idx = cnt = None
    if not mode.endswith("dense"):
        G = rnd.choice([1, Hkv])
        k_max = rnd.randint(1, N)
        idx = torch.full((B, G, k_max), -1, dtype=torch.int32)
        cnt = torch.zeros((B, G), dtype=torch.int32)
        for b in range(B):
            for l in range(G):
                n = rnd.choice([0, rnd.randint(0, min(k_max, int(lens[b]))), min(k_max, int(lens[b]))])
                idx[b, l, :n] = torch.sort(torch.randperm(int(lens[b]), generator=g)[:n]).values.to(torch.int32)
                cnt[b, l] = n
    return dict(B=B, N=N, Hq=Hkv * r, Hkv=Hkv, d=d, T=T, q=q, k_new=k_new, v_new=v_new, kv_gpu=kv_gpu, kv_cpu=kv_cpu,
                idx=idx, cnt=cnt, mode=mode)


@pytest.fixture(params=["tcgen05", "mma_sync"])
def attn_impl(request):
    api.tune_attn_impl(1 if request.param == "mma_sync" else 0)
    yield request.param
    api.tune_attn_impl(0)


@pytest.mark.parametrize("seed", range(28))
def test_random_shapes_match_oracle(seed, attn_impl):
    c = _case(seed)
    sh = api.Shape(c["B"], c["Hq"], c["Hkv"], c["d"], c["T"], c["N"], 0.0)
    k_max = c["idx"].shape[2] if c["idx"] is not None else 0
    ws = api.alloc_workspace(sh, 1, k_max)
    out = torch.full(c["q"].shape, float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((c["B"], c["Hq"], c["T"]), float("nan"), device="cuda")
    api.sparse_verify_attn(sh, c["kv_gpu"](), c["q"].cuda(), c["k_new"].cuda(), c["v_new"].cuda(),
                           None if c["idx"] is None else c["idx"].cuda(), None if c["cnt"] is None else c["cnt"].cuda(),
                           out, ws, lse)
    torch.cuda.synchronize()
    o_ref, lse_ref = ref.sparse_verify_attn(c["kv_cpu"], c["q"], c["k_new"], c["v_new"], c["idx"], c["cnt"], c["N"])
    H.check_attn(out, o_ref, f"seed {seed} ({c['mode']})")
    assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=1e-5), (seed, c["mode"])
    assert int(ws.view(torch.uint8)[:4096].to(torch.int32).sum()) == 0   # the persistent header is left zero
