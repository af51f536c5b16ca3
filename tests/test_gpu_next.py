"""GPU parity of the steps either side of the layer path: dustin_arr (Eq. 1-4), dustin_append_kv
(PAPER.md:153), dustin_draft_aggregate (Eq. 5, first line) and a multi-step decode loop that chains them with the
fused layer call.  Every expected value comes from oracle/."""
import math

import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import api, synth
from tests import harness as H

pytestmark = pytest.mark.gpu

ARR_ATOL = 2e-6            # fp64 accumulation on both sides, one fp32 rounding of the ratio
DRAFT_RTOL = 1e-5          # same arithmetic as a1 (DESIGN.md §7 rule 3), a sum of L * Gamma fp32 terms


def _rand_bf16(*shape, seed):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(*shape, generator=g).to(torch.bfloat16)


# ---- dustin_arr -------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("B,G,N,k", [(1, 1, 1024, 128), (3, 4, 5000, 700), (2, 8, 32768, 2048)])
def test_arr_matches_oracle(B, G, N, k):
    g = torch.Generator().manual_seed(N)
    a = torch.rand(B, G, N, generator=g) ** 8                       # a few heavy entries, like attention rows
    sd = torch.rand(B, G, N, generator=g)
    lens = torch.randint(k + 1, N + 1, (B,), generator=g, dtype=torch.int32)
    lens[0] = N
    idx, cnt = ref.topk_select(sd, a, k, 4, 16, 1, 2, k, lens)
    want = ref.arr(a, idx, cnt, lens)
    got = torch.full((B, G), float("nan"), device="cuda")
    api.arr(a.cuda(), idx.cuda(), cnt.cuda(), got, lens.cuda())
    assert torch.allclose(got.cpu().double(), want, atol=ARR_ATOL, rtol=0)
    # empty lists and rows without mass
    api.arr(torch.zeros(B, G, N, device="cuda"), idx.cuda(), cnt.cuda(), got, lens.cuda())
    assert torch.all(got == 0)
    api.arr(a.cuda(), idx.cuda(), torch.zeros_like(cnt).cuda(), got, lens.cuda())
    assert torch.all(got == 0)


def test_sd_oracle_bound_eq4_by_composition_of_select_and_arr():
    """Eq. 3-4: K = TopK_k of the window sum (dustin_fuse_scores, alpha = 1), ARR evaluated on it; and no policy list
    of the same size beats it."""
    B, G, N, k, w = 2, 2, 4096, 256, 4
    g = torch.Generator().manual_seed(7)
    steps = [(torch.rand(B, G, N, generator=g) ** 6).cuda() for _ in range(w)]
    acc = torch.zeros(B, G, N, device="cuda")
    for s in steps:
        api.fuse_scores(s, acc, 1.0)
    idx = torch.empty(B, G, k, dtype=torch.int32, device="cuda")
    cnt = torch.empty(B, G, dtype=torch.int32, device="cuda")
    api.topk_select(api.Select(k, 0, 0, 0, 1, G, None), acc, acc, idx, cnt)
    best = torch.empty(B, G, device="cuda")
    api.arr(acc, idx, cnt, best)
    want_idx, want_cnt = ref.topk_select(acc.cpu(), acc.cpu(), k, 0, 0, 0, 1)
    assert torch.equal(idx.cpu(), want_idx)
    assert torch.allclose(best.cpu().double(), ref.arr(acc.cpu(), want_idx, want_cnt), atol=ARR_ATOL)
    other = torch.empty(B, G, device="cuda")
    api.topk_select(api.Select(k, 0, 0, 0, 1, G, None), steps[0], steps[0], idx, cnt)   # look-back policy, delta = w
    api.arr(acc, idx, cnt, other)
    assert torch.all(other <= best + 1e-6)


# ---- dustin_append_kv -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("paged", [False, True])
def test_append_matches_oracle_bitwise(paged):
    B, cap, Hkv, Hq, d, T, G, page = 5, 96, 4, 8, 128, 5, 4, 16
    k, v = _rand_bf16(B, cap, Hkv, d, seed=1), _rand_bf16(B, cap, Hkv, d, seed=2)
    kn, vn = _rand_bf16(B, T, Hkv, d, seed=3), _rand_bf16(B, T, Hkv, d, seed=4)
    lens = torch.tensor([10, 93, 0, 96, 47], dtype=torch.int32)
    na = torch.tensor([5, 5, 1, 3, 0], dtype=torch.int32)
    hist = torch.rand(B, G, cap)
    shape = api.Shape(B, Hq, Hkv, d, T, cap, 0.0)
    if paged:
        n_pages = B * cap // page
        table = torch.randperm(n_pages, generator=torch.Generator().manual_seed(5)).to(torch.int32).view(B, cap // page)
        kp = torch.zeros(n_pages, page, Hkv, d, dtype=torch.bfloat16)
        vp = torch.zeros_like(kp)
        for b in range(B):
            for pg in range(cap // page):
                kp[table[b, pg]] = k[b, pg * page:(pg + 1) * page]
                vp[table[b, pg]] = v[b, pg * page:(pg + 1) * page]
        k, v = kp, vp
        cpu_kv = ref.KV(k, v, page * Hkv * d, Hkv * d, d, table.contiguous(), page)
        gk, gv = k.cuda(), v.cuda()
        gpu_kv = api.KV.paged_nhd(gk, gv, table.contiguous().cuda(), None)
    else:
        cpu_kv = ref.KV.contiguous_nhd(k, v)
        gk, gv = k.cuda(), v.cuda()
        gpu_kv = api.KV.contiguous_nhd(gk, gv, None)
    g_lens, g_hist = lens.cuda(), hist.cuda()
    api.append_kv(shape, gpu_kv, g_lens, kn.cuda(), vn.cuda(), na.cuda(), g_hist)
    torch.cuda.synchronize()
    want_lens = ref.append_kv(cpu_kv, lens, kn, vn, na, cap, hist)          # k, v, hist updated in place
    assert g_lens.cpu().tolist() == want_lens.tolist() == [15, 96, 1, 96, 47]
    assert torch.equal(gk.cpu().view(torch.int16), k.view(torch.int16))
    assert torch.equal(gv.cpu().view(torch.int16), v.view(torch.int16))
    assert torch.equal(g_hist.cpu(), hist)


# ---- dustin_draft_aggregate -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("one_pass", [True, False])
@pytest.mark.parametrize("B,N,Hq,Hkv,d,gamma,L,mask", [
    (2, 3000, 14, 2, 64, 4, 3, 0b00101000100010),      # Qwen2.5-0.5B-shaped draft: 14/2 heads, d = 64, 3 layers x 4 heads
    (1, 1024, 8, 8, 128, 2, 2, 0b10000001),
    (2, 2048, 8, 2, 128, 4, 2, 0b00000111),            # 3 heads of one KV group x 4 queries > 8 pairs: per-token passes
])
def test_draft_aggregate_matches_oracle(B, N, Hq, Hkv, d, gamma, L, mask, one_pass):
    ks = [_rand_bf16(B, N, Hkv, d, seed=10 + l) for l in range(L)]
    qs = [_rand_bf16(B, gamma, Hq, d, seed=20 + l) for l in range(L)]
    lens = torch.tensor([N] + [N - 333] * (B - 1), dtype=torch.int32)
    want = ref.draft_aggregate(ks, qs, mask, Hkv, N, N * Hkv * d, Hkv * d, d, seq_lens=lens)
    shape = api.Shape(B, Hq, Hkv, d, gamma, N, 0.0)
    # the larger workspace lets every layer be ONE pass over its K cache; the smaller one forces a pass per token
    ws = api.alloc_draft_workspace(shape, mask) if one_pass else api.alloc_workspace(shape, mask, 1)
    gks = [k.cuda() for k in ks]
    kvs = [api.KV.contiguous_nhd(k, None, lens.cuda()) for k in gks]
    got = torch.full((B, N), float("nan"), device="cuda")
    n0 = api.launch_count()
    api.draft_aggregate(shape, kvs, [q.cuda() for q in qs], mask, got, ws)
    torch.cuda.synchronize()
    launches = api.launch_count() - n0
    r = Hq // Hkv
    fits = max(bin((mask >> (g * r)) & ((1 << r) - 1)).count("1") for g in range(Hkv)) * gamma <= 8
    if not fits:
        assert launches == 3 * L * gamma
    elif one_pass:
        assert launches == 3 * L
    else:                                  # a generous general workspace may also hold the one-pass logits
        assert launches in (3 * L, 3 * L * gamma)
    H.check_scores(got.cpu().unsqueeze(1), want.unsqueeze(1), "s_draft", DRAFT_RTOL)
    n_terms = bin(mask).count("1") * L * gamma
    assert torch.allclose(got.sum(-1).cpu(), torch.full((B,), float(n_terms)), rtol=1e-4)   # Eq. 5 mass


# ---- multi-step decode loop: verify -> accept -> append, history carried ----------------------
def test_multi_step_decode_loop_matches_oracle():
    """Three speculative steps on one layer.  Each step: the fused layer call (a1..a4) on the GPU and the oracle on the
    CPU from the SAME state; a seeded acceptance length; dustin_append_kv on both sides.  State carried across steps:
    cache, lengths, accumulated scores (Eq. 5)."""
    cfg = synth.shrink(synth.config_llama8b(batch=3, ctx=2048, n_layers=1), budget=256, n_sink=8, n_recent=32)
    cap = cfg.ctx
    cpu = synth.make_layer(cfg, 0, "cpu")
    g = torch.Generator().manual_seed(99)
    lens = torch.tensor([cap - 40, cap - 400, cap - 2], dtype=torch.int32)       # the last one runs out of room
    cpu.seq_lens = lens.clone()
    for b in range(cfg.batch):                                                     # nothing accumulated beyond N_b yet
        cpu.hist[b, :, int(lens[b]):] = 0
    dev = cpu.to("cuda")
    sh = H.shape_of(cfg)
    ws = api.alloc_workspace(sh, cfg.head_mask, cpu.k_max)
    for step in range(3):
        # fresh verify block and draft scores of this step (seeded inputs, same on both sides)
        cpu.q = _rand_bf16(*cpu.q.shape, seed=100 + step)
        cpu.k_new = _rand_bf16(*cpu.k_new.shape, seed=200 + step)
        cpu.v_new = _rand_bf16(*cpu.v_new.shape, seed=300 + step)
        cpu.s_draft = torch.rand(cpu.s_draft.shape, generator=g)
        dev.q, dev.k_new, dev.v_new, dev.s_draft = cpu.q.cuda(), cpu.k_new.cuda(), cpu.v_new.cuda(), cpu.s_draft.cuda()
        got = H.run_gpu_fused(dev)
        a_ref, h_ref = H.oracle_scores(cpu)
        H.check_scores(got.hist.cpu(), h_ref, f"hist step {step}")
        idx_same, cnt_same = H.oracle_select(cpu, got.hist.cpu())
        assert torch.equal(got.idx.cpu(), idx_same) and torch.equal(got.cnt.cpu(), cnt_same)
        o_ref, _ = H.oracle_attn(cpu, got.idx.cpu(), got.cnt.cpu())
        H.check_attn(got.out, o_ref)
        # accept 1..T rows, append on both sides; the GPU history becomes the state of both (rule 2 of DESIGN.md §7)
        n_app = torch.randint(1, cfg.n_new + 1, (cfg.batch,), generator=g, dtype=torch.int32)
        dev.hist = got.hist
        api.append_kv(sh, H.gpu_kv(dev), dev.seq_lens, dev.k_new, dev.v_new, n_app.cuda(), dev.hist)
        torch.cuda.synchronize()
        cpu.hist = got.hist.cpu()
        cpu.seq_lens = ref.append_kv(H.cpu_kv(cpu), cpu.seq_lens, cpu.k_new, cpu.v_new, n_app, cap, cpu.hist)
        assert torch.equal(dev.seq_lens.cpu(), cpu.seq_lens)
        assert torch.equal(dev.k.cpu().view(torch.int16), cpu.k.view(torch.int16))
        assert torch.equal(dev.v.cpu().view(torch.int16), cpu.v.view(torch.int16))
        assert torch.equal(dev.hist.cpu(), cpu.hist)
    assert int(cpu.seq_lens[2]) == cap and int(cpu.seq_lens[0]) > cap - 40


# ---- dustin_probe_gather (measurement aid) ----------------------------------------------------------------------------
@pytest.mark.parametrize("paged", [False, True])
def test_probe_gather_runs_on_the_lists_of_a_fused_layer(paged):
    """The probe only reads (the K / V rows of the given lists): it must accept what the fused call produced, on
    contiguous and paged caches, and leave every tensor untouched."""
    cfg = synth.shrink(synth.config_paged(), batch=3, ctx=4096, ragged_min=1500) if paged else \
        synth.shrink(synth.config_llama8b(batch=2, ctx=4096, n_layers=1), budget=512)
    dev = synth.make_layer(cfg, 0, "cuda")
    got = H.run_gpu_fused(dev, want_scores=False)
    sh = H.shape_of(cfg)
    ws = api.alloc_workspace(sh, cfg.head_mask, dev.k_max)
    k0, idx0 = dev.k.clone(), got.idx.clone()
    api.probe_gather(sh, H.gpu_kv(dev), got.idx, got.cnt, ws)
    torch.cuda.synchronize()
    assert torch.equal(dev.k.view(torch.int16), k0.view(torch.int16)) and torch.equal(got.idx, idx0)
    assert int(ws[:4096].max()) == 0                     # the persistent header of the workspace stays zero


def test_graph_replayed_decode_steps_equal_eager_steps():
    """The decode step -- two target layers (paged caches, ragged lengths, per-sequence budgets) through the one-shot
    call, then the appends -- captured ONCE as a CUDA graph and replayed for three steps must leave bit for bit the state
    that the same calls leave when issued one by one: caches, lengths, accumulated scores, outputs, index lists.  Lengths,
    accept counts and every per-step input live in fixed device buffers, so one graph serves every step (bench.py --loop).
    The eager path is the one test_multi_step_decode_loop_matches_oracle holds against the oracle."""
    cfg = synth.shrink(synth.config_paged(), batch=3, ctx=2048, ragged_min=600, n_sink=4, n_recent=16, n_layers=2)
    T, n_steps = cfg.n_new, 3
    sh = H.shape_of(cfg)

    def run(use_graph: bool):
        layers = [synth.make_layer(cfg, l, "cuda") for l in (0, 1)]
        lens = layers[0].seq_lens.clamp(max=cfg.ctx - n_steps * T).contiguous()      # room for every append
        for x in layers:
            x.seq_lens = lens                                                        # one set of lengths for all layers
            for b in range(cfg.batch):
                x.hist[b, :, int(lens[b]):] = 0
        ws = api.alloc_workspace(sh, cfg.head_mask, layers[0].k_max)
        outs = [torch.zeros_like(x.q) for x in layers]
        idxs = [torch.full((cfg.batch, cfg.n_lists, x.k_max), -1, dtype=torch.int32, device="cuda") for x in layers]
        cnts = [torch.zeros((cfg.batch, cfg.n_lists), dtype=torch.int32, device="cuda") for x in layers]
        n_app = torch.zeros(cfg.batch, dtype=torch.int32, device="cuda")
        scratch = torch.zeros_like(lens)

        def step():
            for l, x in enumerate(layers):
                api.verify_layer_fused(sh, H.gpu_kv(x), x.q, x.k_new, x.v_new, cfg.head_mask, x.s_draft, x.hist, 1.0,
                                       H.select_of(x), outs[l], idxs[l], cnts[l], ws)
            scratch.copy_(lens)
            api.append_kv(sh, H.gpu_kv(layers[0]), scratch, layers[0].k_new, layers[0].v_new, n_app, layers[0].hist)
            api.append_kv(sh, H.gpu_kv(layers[1]), lens, layers[1].k_new, layers[1].v_new, n_app, layers[1].hist)

        replay = None
        if use_graph:
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                step()
            replay = g.replay
        trail = []
        gen = torch.Generator().manual_seed(4242)
        for s in range(n_steps):
            for l, x in enumerate(layers):                                           # this step's inputs, in place
                x.q.copy_(_rand_bf16(*x.q.shape, seed=1000 + 10 * s + l))
                x.k_new.copy_(_rand_bf16(*x.k_new.shape, seed=2000 + 10 * s + l))
                x.v_new.copy_(_rand_bf16(*x.v_new.shape, seed=3000 + 10 * s + l))
                x.s_draft.copy_(torch.rand(x.s_draft.shape, generator=gen))
            n_app.copy_(torch.randint(0, T + 1, (cfg.batch,), generator=gen, dtype=torch.int32))
            (replay or step)()
            torch.cuda.synchronize()
            trail.append([t.clone() for t in (*outs, *idxs, *cnts, lens)])
        state = [t for x in layers for t in (x.k, x.v, x.hist)] + [lens, ws[:4096]]
        return trail, state

    eager_trail, eager_state = run(False)        # also loads every kernel before the capture below
    graph_trail, graph_state = run(True)
    bits = lambda t: t.view(torch.int16) if t.dtype == torch.bfloat16 else t
    for s, (a, b) in enumerate(zip(eager_trail, graph_trail)):
        for i, (x, y) in enumerate(zip(a, b)):
            assert torch.equal(bits(x), bits(y)), f"step {s}: tensor {i} differs between eager and graph replay"
    for i, (x, y) in enumerate(zip(eager_state, graph_state)):
        assert torch.equal(bits(x), bits(y)), f"final state tensor {i} differs"
    assert int(eager_state[-2].sum()) > int(synth.make_layer(cfg, 0, "cpu").seq_lens.clamp(max=cfg.ctx - n_steps * T).sum())
    assert not graph_state[-1].any()             # the workspace header is zero again
