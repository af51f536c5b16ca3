"""The selection path of the ONE-SHOT call (dustin_verify_layer_fused): the draft tier of Eq. 6 runs in a kernel of its
own beside stage a1 (256-thread CTAs when many rows are in flight, 1024-thread CTAs otherwise), the target tier picks the
membership bitmask up, materialises its own score row (a1's normalisation + Eq. 5) and emits the list.  Checked here:
  * bit-for-bit equality with the four staged calls -- lists, the carried history `hist`, attention output -- on shapes
    that take the in-kernel row path (batch * n_lists >= 64, ctx % 4 == 0), with ragged lengths and an invalid-budget row;
  * bit-exact agreement of the lists with the ORACLE's selection (Eq. 6) on adversarial score rows:
    heavy ties in both tiers, zeros, negatives, with every switch of dustin_debug.h that changes which kernels run.
Acceptance rules: tests/harness.py."""
import dataclasses

import pytest
import torch

from paper_2606_24957_b200 import api, synth
from tests import harness as H

pytestmark = pytest.mark.gpu


@pytest.fixture(params=["hoist", "no_hoist", "cluster2", "cluster4", "cluster8", "no_cluster"])
def hoist(request):
    """Which kernels serve the selection of the one-shot call: the draft tier hoisted beside a1 (default) or not; the
    target tier by one CTA per row or by a thread-block cluster of 2 / 4 / 8 CTAs per row (select_cluster.cu; by default
    only few-row shapes take it: forced here on every shape)."""
    api.tune_set(api.KNOB_DRAFT_HOIST, 0 if request.param == "no_hoist" else 1)
    api.tune_set(api.KNOB_SELECT_SPLIT, {"cluster2": 2, "cluster4": 4, "cluster8": 8, "no_cluster": 1}.get(request.param, 0))
    yield request.param
    api.tune_set(api.KNOB_DRAFT_HOIST, 1)
    api.tune_set(api.KNOB_SELECT_SPLIT, 0)


def many_rows_cases():
    llama = synth.config_llama8b()
    qwen = synth.config_qwen72b()
    return {
        # 64 rows, 16-byte rows: select kernels materialise their own rows; the light draft-tier kernel runs
        "llama_64rows": synth.shrink(llama, batch=8, ctx=2048, budget=300, n_sink=8, n_recent=40),
        # 160 rows: more rows than SMs, at most twice as many -- the 512-thread target-tier kernel (two CTAs per SM)
        "llama_160rows": synth.shrink(llama, batch=20, ctx=2048, budget=300, n_sink=8, n_recent=40),
        # ragged lengths + per-sequence budgets (one of them made invalid below), paged cache
        "paged_96rows": synth.shrink(synth.config_paged(), batch=12, ctx=3072, ragged_min=700, n_sink=4, n_recent=16),
        # few rows (1024-thread draft-tier kernel, separate normalisation launches), G = 1
        "qwen_packed_4rows": synth.shrink(qwen, batch=4, ctx=4096, budget=512, n_sink=16, n_recent=64,
                                          heads=synth.packed_heads(8), n_lists=1),
        # unaligned rows: the scalar kernels
        "qwen_72rows_odd": synth.shrink(qwen, batch=9, ctx=1531, budget=200, n_sink=8, n_recent=32),
    }


CASES = many_rows_cases()


@pytest.mark.parametrize("name", list(CASES))
def test_fused_equals_staged_bitwise_on_the_in_kernel_row_path(name, hoist):
    cfg = CASES[name]
    dev = synth.make_layer(cfg, 0, "cuda")
    if dev.budgets is not None:
        dev.budgets[1] = cfg.n_sink + cfg.n_recent - 1      # invalid budget: that row gets cnt = 0 and an all -1 list
    staged = H.run_gpu_staged(dev)
    fused = H.run_gpu_fused(dev)
    again = H.run_gpu_fused(dev, want_scores=False)        # the path bench.py times (no scores_now output)
    for r in (fused, again):
        assert torch.equal(r.cnt, staged.cnt)
        assert torch.equal(r.idx, staged.idx)
        assert torch.equal(r.hist.view(torch.int32), staged.hist.view(torch.int32))
        assert torch.equal(r.out.view(torch.int16), staged.out.view(torch.int16))
        assert torch.equal(r.lse.view(torch.int32), staged.lse.view(torch.int32))
    assert torch.equal(fused.scores_now, staged.scores_now)
    if dev.budgets is not None:
        assert (staged.cnt[1] == 0).all() and (staged.idx[1] == -1).all()
    # and the lists are the oracle's on the GPU's own scores (the oracle refuses an invalid budget outright, so it sees a
    # valid one for that sequence and its rows are left out of the comparison)
    cpu = dev.to("cpu")
    keep = torch.ones(cfg.batch, dtype=torch.bool)
    if cpu.budgets is not None:
        cpu.budgets[1] = cfg.n_sink + cfg.n_recent
        keep[1] = False
    idx_same, cnt_same = H.oracle_select(cpu, again.hist.cpu())
    assert torch.equal(again.cnt.cpu()[keep], cnt_same[keep]) and torch.equal(again.idx.cpu()[keep], idx_same[keep])


def _tie_heavy_inputs(cfg, seed, device="cuda"):
    """Zero K makes a1 exactly uniform (p = 1/N for every head and position), so the ties planted in `hist` survive the
    Eq. 5 accumulation; the draft scores carry ties, zeros and negatives of their own (reading A15: compare as
    max(s, 0))."""
    inp = synth.make_layer(cfg, 0, device)
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    B, G, N = cfg.batch, cfg.n_lists, cfg.ctx
    inp.k.zero_()
    levels = torch.randint(0, 6, (B, G, N), generator=g, device=device)
    inp.hist = (levels.float() * 0.125).contiguous()                   # six distinct values: massive ties
    d_shape = (B, N) if inp.s_draft.dim() == 2 else (B, G, N)
    dl = torch.randint(-2, 5, d_shape, generator=g, device=device).float() * 0.25   # ties, zeros, negatives
    rare = torch.rand(d_shape, generator=g, device=device) < 0.01
    inp.s_draft = torch.where(rare, torch.rand(d_shape, generator=g, device=device) + 2.0, dl).contiguous()
    return inp


@pytest.mark.parametrize("name,m", [("llama_64rows", (1, 2)), ("llama_64rows", (0, 1)), ("llama_64rows", (1, 1)),
                                    ("llama_160rows", (1, 2)), ("llama_160rows", (2, 3)),
                                    ("paged_96rows", (1, 3)), ("qwen_packed_4rows", (1, 2)), ("qwen_72rows_odd", (2, 3))])
def test_fused_selection_is_the_oracles_under_heavy_ties(name, m, hoist):
    cfg = dataclasses.replace(CASES[name], m_num=m[0], m_den=m[1])
    dev = _tie_heavy_inputs(cfg, 1234)
    got = H.run_gpu_fused(dev, want_scores=False)
    cpu = dev.to("cpu")
    # the carried history: uniform a1 (|subset heads feeding the list| / N_b per position) on top of the planted levels
    idx_ref, cnt_ref = H.oracle_select(cpu, got.hist.cpu())
    assert torch.equal(got.cnt.cpu(), cnt_ref)
    assert torch.equal(got.idx.cpu(), idx_ref)
    H.check_index_lists_valid(cpu, got.idx, got.cnt)
    a_ref, h_ref = H.oracle_scores(cpu)
    H.check_scores(got.hist, h_ref, "hist")
