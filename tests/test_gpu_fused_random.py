"""Randomised GPU parity of the ONE-SHOT call (dustin_verify_layer_fused) on seeded random shapes: head subsets (packed,
spread, arbitrary), one list per sequence or per KV head, contiguous / ragged / paged caches, budgets from a few rows to
the whole context, draft quotas from none to all.  Per case: the one-shot call equals the four staged calls bit for bit
(lists, carried history, output), its lists are the ORACLE's selection on the scores it produced (Eq. 6, bit-exact), its
scores are the oracle's within the a1 tolerance and its attention output the oracle's on those lists (harness.py)."""
import dataclasses
import random

import pytest
import torch

from paper_2606_24957_b200 import api, synth
from tests import harness as H

pytestmark = pytest.mark.gpu


def _config(seed: int) -> synth.Config:
    rnd = random.Random(7000 + seed)
    base = rnd.choice(["qwen", "llama", "paged"])
    if base == "paged":
        cfg = synth.config_paged()
        Hq, Hkv = cfg.n_q_heads, cfg.n_kv_heads
    else:
        cfg = synth.config_qwen72b() if base == "qwen" else synth.config_llama8b()
        Hq, Hkv = cfg.n_q_heads, cfg.n_kv_heads
    r = Hq // Hkv
    kind = rnd.choice(["spread", "packed", "any"])
    if kind == "spread":
        heads = synth.spread_heads(Hq, rnd.choice([2, 4, 8]))
    elif kind == "packed":
        heads = synth.packed_heads(rnd.randint(1, min(8, r)))
    else:
        pool = list(range(Hq))
        rnd.shuffle(pool)
        heads, per_group = [], {}
        for h in pool:
            if len(heads) == rnd.randint(1, 12):
                break
            if per_group.get(h // r, 0) < 8:
                heads.append(h)
                per_group[h // r] = per_group.get(h // r, 0) + 1
        heads = tuple(sorted(heads)) or (0,)
    n_lists = rnd.choice([1, Hkv])
    batch = rnd.choice([1, 2, 3, 8, 12]) if n_lists == Hkv else rnd.choice([1, 4, 16, 70])
    ctx = rnd.choice([512, 1024, 1536, 2500, 4096, 6144]) if base != "paged" else rnd.choice([1024, 3072, 4096])
    if rnd.random() < 0.7:
        ctx = ctx // 4 * 4
    n_sink, n_recent = rnd.choice([(0, 0), (4, 16), (8, 40), (16, 64)])
    budget = rnd.choice([n_sink + n_recent, n_sink + n_recent + 1, 200, 300, ctx // 8, ctx // 2, ctx])
    budget = max(budget, n_sink + n_recent, 1)
    m_num, m_den = rnd.choice([(0, 1), (1, 2), (1, 3), (2, 3), (1, 1)])
    kw = dict(batch=batch, ctx=ctx, heads=heads, n_lists=n_lists, n_sink=n_sink, n_recent=n_recent, m_num=m_num,
              m_den=m_den, gamma=rnd.choice([1, 2, 4]), seed=20260624 + seed)
    if base == "paged":
        # k_b = N_b / 16 must cover the protected set (the oracle refuses a budget below S + W outright)
        kw.update(ragged_min=max(ctx // 5, 16 * (n_sink + n_recent + 1)))
        if kw["ragged_min"] >= ctx:
            kw.update(n_sink=4, n_recent=16, ragged_min=max(ctx // 5, 16 * 21))
    else:
        kw.update(budget=budget)
        if rnd.random() < 0.4:
            kw.update(ragged_min=max(ctx // 4, 8))
    return dataclasses.replace(cfg, **kw)


@pytest.mark.parametrize("seed", range(40))
def test_random_layers(seed):
    cfg = _config(seed)
    dev = synth.make_layer(cfg, 0, "cuda")
    staged = H.run_gpu_staged(dev)
    fused = H.run_gpu_fused(dev)
    again = H.run_gpu_fused(dev, want_scores=False)
    for r in (fused, again):
        assert torch.equal(r.cnt, staged.cnt), seed
        assert torch.equal(r.idx, staged.idx), seed
        assert torch.equal(r.hist.view(torch.int32), staged.hist.view(torch.int32)), seed
        assert torch.equal(r.out.view(torch.int16), staged.out.view(torch.int16)), seed
    assert torch.equal(fused.scores_now, staged.scores_now)
    cpu = dev.to("cpu")
    idx_same, cnt_same = H.oracle_select(cpu, again.hist.cpu())
    assert torch.equal(again.cnt.cpu(), cnt_same) and torch.equal(again.idx.cpu(), idx_same), seed
    H.check_index_lists_valid(cpu, again.idx, again.cnt)
    a_ref, h_ref = H.oracle_scores(cpu)
    H.check_scores(fused.scores_now, a_ref, "scores_now")
    H.check_scores(again.hist, h_ref, "hist")
    o_ref, _ = H.oracle_attn(cpu, again.idx.cpu(), again.cnt.cpu())
    H.check_attn(again.out, o_ref)
