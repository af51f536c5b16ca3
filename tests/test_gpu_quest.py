"""GPU parity of the Quest-16 estimator (dustin_quest_build_pages / dustin_quest_score_pages)
against the oracle's O8 / O9 on the same seeded layers: the page metadata bit for bit (min / max are selections), the
page scores within the a1 tolerance (tests/harness.py), the upper-bound logits within 1e-5 relative to their scale, the
bound property against exact logits, the incremental rebuild after an append, and page ranking through
dustin_topk_select."""
import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import api, synth
from tests import harness as H

pytestmark = pytest.mark.gpu

P = api.QUEST_PAGE


def cases():
    qwen, llama = synth.config_qwen72b(), synth.config_llama8b()
    return {
        # 8 scored groups, one head each; context not a multiple of 16 (short last page)
        "qwen_spread": synth.shrink(qwen, batch=2, ctx=4100, budget=600, n_sink=64, n_recent=256),
        "qwen_spread_one_list": synth.shrink(qwen, batch=2, ctx=4096, budget=600, n_sink=64, n_recent=256, n_lists=1),
        # 4 heads in ONE group; several scoring CTAs per sequence (> 128 pages)
        "llama_packed": synth.shrink(llama, batch=3, ctx=5000, budget=512, n_sink=8, n_recent=64,
                                     heads=synth.packed_heads(4), n_lists=1),
        # every head: 8 heads per group, list fed by 64 heads
        "qwen_all_heads": synth.shrink(qwen, batch=1, ctx=2600, budget=300, n_sink=8, n_recent=32,
                                       heads=tuple(range(64)), n_lists=1),
        # groups without a subset head (reading A2)
        "qwen_empty_groups": synth.shrink(qwen, batch=1, ctx=2049, budget=333, n_sink=4, n_recent=16,
                                          heads=(0, 1, 2, 17, 63), n_lists=8),
        "d64": synth.shrink(qwen, batch=2, ctx=1100, budget=200, n_sink=8, n_recent=32, gamma=2, head_dim=64),
        # paged cache, ragged lengths (pages without a token, a sequence ending inside a page)
        "paged_ragged": synth.shrink(synth.config_paged(), batch=3, ctx=4000, ragged_min=900, n_sink=4, n_recent=16),
    }


CASES = cases()


def _gpu_quest(dev, want_ub=True):
    c = dev.cfg
    sh = H.shape_of(c)
    meta = api.quest_alloc_meta(sh)
    meta.fill_(float("nan"))
    api.quest_build_pages(sh, H.gpu_kv(dev), meta)
    n_pages = meta.shape[1]
    ws = api.alloc_workspace(sh, c.head_mask, 1)
    scores = torch.full((c.batch, c.n_lists, n_pages), float("nan"), device="cuda")
    ub = torch.full((c.batch, len(c.heads), n_pages), float("nan"), device="cuda") if want_ub else None
    api.quest_score_pages(sh, meta, dev.q[:, 0], c.head_mask, c.n_lists, scores, ws, dev.seq_lens, ub)
    torch.cuda.synchronize()
    return meta, scores, ub


@pytest.mark.parametrize("name", list(CASES))
def test_quest_matches_oracle(name):
    cfg = CASES[name]
    cpu = synth.make_layer(cfg, 0, "cpu")
    dev = cpu.to("cuda")
    meta, scores, ub = _gpu_quest(dev)
    kmin, kmax = ref.quest_page_minmax(H.cpu_kv(cpu), cfg.n_kv_heads, cfg.ctx, P)
    # O8: selections, so bit for bit (as values: -0.0 == 0.0)
    assert torch.equal(meta[:, :, :, 0].cpu().double(), kmin), "kmin differs"
    assert torch.equal(meta[:, :, :, 1].cpu().double(), kmax), "kmax differs"
    # O9
    want, ub_ref = ref.quest_score_pages(kmin, kmax, cpu.q[:, 0], cfg.head_mask, cfg.n_lists, cfg.ctx, P, cpu.seq_lens,
                                         0.0, want_ub=True)
    H.check_scores(scores, want, "page_scores")
    ub_ref = ub_ref[:, sorted(cfg.heads)]
    err = (ub.cpu().double() - ub_ref).abs().max().item()
    assert err <= 1e-5 * max(1.0, ub_ref.abs().max().item()), f"upper-bound logits: max abs error {err:.3e}"
    # every list is a sum of per-head distributions over the live pages
    lens = cpu.seq_lens if cpu.seq_lens is not None else torch.full((cfg.batch,), cfg.ctx, dtype=torch.int32)
    for b in range(cfg.batch):
        live = (int(lens[b]) + P - 1) // P
        assert (scores[b, :, live:] == 0).all() and (ub[b, :, live:] == 0).all()


def test_upper_bound_dominates_exact_logits_on_the_gpu():
    cfg = CASES["qwen_spread"]
    dev = synth.make_layer(cfg, 0, "cuda")
    _, _, ub = _gpu_quest(dev)
    r = cfg.n_q_heads // cfg.n_kv_heads
    scale = cfg.head_dim ** -0.5
    for j, h in enumerate(sorted(cfg.heads)):
        logits = torch.einsum("bnc,bc->bn", dev.k[:, :, h // r].double(), dev.q[:, 0, h].double()) * scale
        n_pages = ub.shape[2]
        pad = n_pages * P - cfg.ctx
        page_max = torch.nn.functional.pad(logits, (0, pad), value=float("-inf")).view(cfg.batch, n_pages, P).amax(dim=2)
        slack = ub[:, j].double() - page_max
        assert (slack >= -1e-4).all(), f"head {h}: an exact logit exceeds its page's bound by {-slack.min().item():.3e}"


def test_incremental_rebuild_after_append_equals_full_rebuild():
    cfg = CASES["paged_ragged"]
    cpu = synth.make_layer(cfg, 0, "cpu")
    dev = cpu.to("cuda")
    sh = H.shape_of(cfg)
    kv = H.gpu_kv(dev)
    meta = api.quest_alloc_meta(sh)
    api.quest_build_pages(sh, kv, meta)
    old_lens = dev.seq_lens.clone()
    room = (cfg.ctx - old_lens).clamp(min=0)
    n_app = torch.minimum(torch.tensor([cfg.n_new, 2, 0], dtype=torch.int32, device="cuda")[:cfg.batch], room).to(torch.int32)
    api.append_kv(sh, kv, dev.seq_lens, dev.k_new, dev.v_new, n_app)          # lengths advance in place
    before = meta.clone()
    api.quest_build_pages(sh, kv, meta, first_token=old_lens)                 # only the pages the append touched
    full = api.quest_alloc_meta(sh)
    api.quest_build_pages(sh, kv, full)
    torch.cuda.synchronize()
    assert torch.equal(meta.view(torch.int16), full.view(torch.int16))
    assert int(n_app.sum()) > 0 and not torch.equal(before.view(torch.int16), meta.view(torch.int16))
    # and both equal the oracle on the appended cache
    k_cpu, lens_cpu = dev.k.cpu(), dev.seq_lens.cpu()
    ps, Hk, d = k_cpu.shape[1], k_cpu.shape[2], k_cpu.shape[3]
    kmin, kmax = ref.quest_page_minmax(ref.KV(k_cpu, None, ps * Hk * d, Hk * d, d, cpu.page_table, ps, lens_cpu),
                                       cfg.n_kv_heads, cfg.ctx, P)
    assert torch.equal(meta[:, :, :, 0].cpu().double(), kmin) and torch.equal(meta[:, :, :, 1].cpu().double(), kmax)


def test_page_scores_rank_pages_through_topk_select():
    """The page scores have the format of a1's scores (pages for tokens): dustin_topk_select on them, with m = 0, returns
    the oracle's top pages for those scores bit for bit."""
    cfg = CASES["qwen_spread"]
    dev = synth.make_layer(cfg, 0, "cuda")
    _, scores, _ = _gpu_quest(dev, want_ub=False)
    B, G, n_pages = scores.shape
    k_pages = 40
    idx = torch.full((B, G, k_pages), -7, dtype=torch.int32, device="cuda")
    cnt = torch.full((B, G), -7, dtype=torch.int32, device="cuda")
    sel = api.Select(k_pages, 1, 2, 0, 1, G)                                   # first page + last two pages always kept
    api.topk_select(sel, scores, scores, idx, cnt)
    torch.cuda.synchronize()
    idx_ref, cnt_ref = ref.topk_select(scores.cpu(), scores.cpu(), k_pages, 1, 2, 0, 1, k_pages)
    assert torch.equal(idx.cpu(), idx_ref) and torch.equal(cnt.cpu(), cnt_ref)


def test_quest_argument_errors():
    cfg = CASES["d64"]
    dev = synth.make_layer(cfg, 0, "cuda")
    sh = H.shape_of(cfg)
    meta = api.quest_alloc_meta(sh)
    scores = torch.empty((cfg.batch, cfg.n_lists, meta.shape[1]), device="cuda")
    tiny_ws = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    with pytest.raises(api.DustinError) as e:
        api.quest_score_pages(sh, meta, dev.q[:, 0], cfg.head_mask, cfg.n_lists, scores, tiny_ws)
    assert e.value.status == api.ERR_WORKSPACE
    ws = api.alloc_workspace(sh, cfg.head_mask, 1)
    with pytest.raises(api.DustinError) as e:
        api.quest_score_pages(sh, meta, dev.q[:, 0], 0, cfg.n_lists, scores, ws)
    assert e.value.status == api.ERR_INVALID_ARG
