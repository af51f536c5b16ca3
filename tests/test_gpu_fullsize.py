"""GPU parity at BASELINE.json's FULL sizes, through the fused one-shot call -- the launch configuration that
bench.py times (dustin_verify_layer_fused on one layer of the workload).  The oracle finishes one full-size layer
in well under a minute on the host cores, so the comparison is still element by element over the whole output
(scores, index lists, attention), with the acceptance rules of tests/harness.py.
Inputs are drawn on the GPU (seeded) and copied to the host for the oracle, so both sides see identical bits."""
import pytest
import torch

from paper_2606_24957_b200 import api, synth
from tests import harness as H

pytestmark = pytest.mark.gpu


def full_cases():
    return {
        # BASELINE.json configs[1]
        "llama8b_32k_b16": synth.config_llama8b(),
        # configs[2], both subset placements
        "qwen72b_32k_b16_spread": synth.config_qwen72b(),
        "qwen72b_32k_b16_packed": synth.config_qwen72b(spread=False),
        # configs[3]: ends of the context sweep, gamma 2 / 8, fixed and 6.25 % budgets (reading A18)
        "qwen72b_4k_b16_gamma2_k256": synth.config_qwen72b(ctx=4096, gamma=2, budget=256),
        "qwen72b_128k_b4_gamma8_k8192": synth.config_qwen72b(batch=4, ctx=131072, gamma=8, budget=8192),
        "qwen72b_64k_b8_gamma8_k2048": synth.config_qwen72b(batch=8, ctx=65536, gamma=8),
        # the benched gamma-4 points of the sweep whose few long units take the even-pieces attention plan, the middle
        # contexts, and the paper's own budget (k = 512, S = 4, W = 16)
        "qwen72b_64k_b8_gamma4_k2048": synth.config_qwen72b(batch=8, ctx=65536),
        "qwen72b_128k_b4_gamma4_k2048": synth.config_qwen72b(batch=4, ctx=131072),
        "qwen72b_8k_b16_gamma4_k2048": synth.config_qwen72b(ctx=8192),
        "qwen72b_16k_b16_gamma4_k1024": synth.config_qwen72b(ctx=16384, budget=1024),
        "qwen72b_32k_b16_gamma4_k512_paper": synth.shrink(synth.config_qwen72b(budget=512), n_sink=4, n_recent=16),
        # configs[4]
        "paged_ragged_b32": synth.config_paged(),
    }


CASES = full_cases()


@pytest.mark.parametrize("name", list(CASES))
def test_full_size_fused_layer_matches_oracle(name):
    cfg = CASES[name]
    torch.cuda.empty_cache()
    dev = synth.make_layer(cfg, 0, "cuda")
    dev.planted = None
    got = H.run_gpu_fused(dev)
    cpu = dev.to("cpu")
    a_ref, h_ref = H.oracle_scores(cpu)
    H.check_scores(got.scores_now, a_ref, "scores_now")
    H.check_scores(got.hist, h_ref, "hist")
    idx_same, cnt_same = H.oracle_select(cpu, got.hist.cpu())
    assert torch.equal(got.cnt.cpu(), cnt_same)
    assert torch.equal(got.idx.cpu(), idx_same)
    idx_ref, cnt_ref = H.oracle_select(cpu, h_ref)
    H.check_index_lists_valid(cpu, got.idx, got.cnt)
    H.check_near_tie_only(cpu, got.idx, got.cnt, idx_ref, cnt_ref, h_ref)
    o_ref, lse_ref = H.oracle_attn(cpu, got.idx.cpu(), got.cnt.cpu())
    H.check_attn(got.out, o_ref)
    assert torch.allclose(got.lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)
    # the same layer again: bit-identical (no order-dependent arithmetic anywhere, including the stream-K merge)
    again = H.run_gpu_fused(dev, want_scores=False)
    assert torch.equal(again.idx, got.idx)
    assert torch.equal(again.out.view(torch.int16), got.out.view(torch.int16))
    assert torch.equal(again.lse, got.lse)
    del dev, cpu, got, again


@pytest.mark.parametrize("name", ["qwen72b_32k_b16_spread", "paged_ragged_b32"])
def test_full_size_dense_baseline_sampled(name):
    """a5 at full size: the dense kernel over all N_b rows, checked on sampled sequences (the oracle's dense
    attention over the whole batch would take minutes)."""
    cfg = CASES[name]
    torch.cuda.empty_cache()
    dev = synth.make_layer(cfg, 0, "cuda", want_hist_draft=False)
    sh = H.shape_of(cfg)
    ws = api.alloc_workspace(sh, cfg.head_mask, 0)
    out = torch.full_like(dev.q, float("nan"))
    lse = torch.full((cfg.batch, cfg.n_q_heads, cfg.n_new), float("nan"), device="cuda")
    api.sparse_verify_attn(sh, H.gpu_kv(dev), dev.q, dev.k_new, dev.v_new, None, None, out, ws, lse)
    torch.cuda.synchronize()
    assert torch.isfinite(out.float()).all()
    from oracle import ref
    for b in (0, cfg.batch // 2, cfg.batch - 1):
        if dev.page_table is not None:
            n_b = int(dev.seq_lens[b])
            pages = dev.page_table[b, :(n_b + cfg.page_size - 1) // cfg.page_size].long()
            k_b = dev.k[pages].reshape(-1, cfg.n_kv_heads, cfg.head_dim)[:n_b].unsqueeze(0).cpu()
            v_b = dev.v[pages].reshape(-1, cfg.n_kv_heads, cfg.head_dim)[:n_b].unsqueeze(0).cpu()
        else:
            n_b = cfg.ctx
            k_b, v_b = dev.k[b:b + 1].cpu(), dev.v[b:b + 1].cpu()
        o_ref, lse_ref = ref.sparse_verify_attn(ref.KV.contiguous_nhd(k_b, v_b, None), dev.q[b:b + 1].cpu(),
                                                dev.k_new[b:b + 1].cpu(), dev.v_new[b:b + 1].cpu(), None, None, n_b)
        H.check_attn(out[b:b + 1], o_ref, f"dense attention, sequence {b}")
        assert torch.allclose(lse[b:b + 1].cpu().double(), lse_ref, atol=2e-3, rtol=0)
