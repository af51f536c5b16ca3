"""Back-to-back one-shot calls on ONE workspace, no host synchronisation in between (the shape of a decode loop and of
the CUDA-graph-replayed bench step).

The four kernels of dustin_verify_layer_fused are chained by programmatic dependent launch, and two of them start work
before their own dependency wait: the scoring kernel of a call with a hoisted draft tier reads q / K and writes the
logits scratch before any griddepcontrol.wait (score.cu, ScoreParams::defer_wait), and the tcgen05 attention kernel
releases its dependents at its very start (attn_tc.cu).  The attention kernel's stream-K scratch and the logits scratch
share the front of the workspace, so call n+1's scoring kernel must not start before call n's attention kernel is
complete.  That holds because the draft-tier selection kernel in between waits (for call n's attention) BEFORE it
triggers (call n+1's scoring) -- DESIGN.md section 5, "PDL chain invariant".  A reordering there would race silently; this test
makes it loud: a chain of unsynchronised calls, alternating two different layers on one workspace, must give bit for
bit what the same calls give when each is followed by a device synchronise -- with the attention kernel's early trigger
(default) and with its trigger at the end (DUSTIN_KNOB_ATTN_TRACE bit 64).
"""
import pytest
import torch

from paper_2606_24957_b200 import api, synth
from tests import harness as H

pytestmark = pytest.mark.gpu

N_CALLS = 24


def _chain(layers, ws, sync_each: bool):
    """Runs N_CALLS one-shot calls that alternate between the given layers, all on `ws`; returns per-call outputs."""
    res = []
    for i in range(N_CALLS):
        dev, state = layers[i % len(layers)]
        c = dev.cfg
        out = torch.full_like(dev.q, float("nan"))
        idx = torch.full((c.batch, c.n_lists, dev.k_max), -7, dtype=torch.int32, device="cuda")
        cnt = torch.full((c.batch, c.n_lists), -7, dtype=torch.int32, device="cuda")
        lse = torch.full((c.batch, c.n_q_heads, c.n_new), float("nan"), device="cuda")
        res.append((out, idx, cnt, lse))
    if sync_each:
        torch.cuda.synchronize()
    for i in range(N_CALLS):
        dev, state = layers[i % len(layers)]
        out, idx, cnt, lse = res[i]
        api.verify_layer_fused(H.shape_of(dev.cfg), H.gpu_kv(dev), dev.q, dev.k_new, dev.v_new, dev.cfg.head_mask,
                               dev.s_draft, state["hist"], 1.0, H.select_of(dev), out, idx, cnt, ws, None, lse)
        if sync_each:
            torch.cuda.synchronize()
    torch.cuda.synchronize()
    return res


@pytest.mark.parametrize("late_trigger", [False, True])
@pytest.mark.parametrize("name", ["few_units_cut_across_ctas", "many_units"])
def test_unsynchronised_chain_equals_synchronised_calls(name, late_trigger):
    qwen = synth.config_qwen72b()
    if name == "few_units_cut_across_ctas":      # 16 (sequence, KV head) units on 148 SMs: every unit is merged through the scratch
        cfg = synth.shrink(qwen, batch=2, ctx=4096, budget=1024, n_sink=16, n_recent=64, n_layers=2)
    else:                                        # 192 units: whole units per CTA, some cut
        cfg = synth.shrink(qwen, batch=24, ctx=2048, budget=512, n_sink=16, n_recent=64, n_layers=2)
    sh = H.shape_of(cfg)
    assert api.tune_get(api.KNOB_DRAFT_HOIST) == 1 and api.tune_get(api.KNOB_PDL) == 1
    api.tune_set(api.KNOB_ATTN_TRACE, 64 if late_trigger else 0)
    try:
        runs = []
        for sync_each in (True, False):
            layers = []
            for layer in (0, 1):
                dev = synth.make_layer(cfg, layer, "cuda")
                layers.append((dev, {"hist": dev.hist.clone()}))
            ws = api.alloc_workspace(sh, cfg.head_mask, layers[0][0].k_max)
            runs.append((_chain(layers, ws, sync_each), [st["hist"] for _, st in layers], ws))
    finally:
        api.tune_set(api.KNOB_ATTN_TRACE, 0)
    (ref_res, ref_hist, ref_ws), (got_res, got_hist, got_ws) = runs
    for i, (r, g) in enumerate(zip(ref_res, got_res)):
        for what, a, b in zip(("out", "idx", "cnt", "lse"), r, g):
            a = a.view(torch.int16) if a.dtype == torch.bfloat16 else a
            b = b.view(torch.int16) if b.dtype == torch.bfloat16 else b
            assert torch.equal(a, b), f"call {i}: {what} of the unsynchronised chain differs"
    for a, b in zip(ref_hist, got_hist):
        assert torch.equal(a, b), "carried history differs"
    # every call left the persistent header of the workspace zero again (dustin.h, "Workspace")
    for ws in (ref_ws, got_ws):
        assert not ws[:4096].any()
