"""Shared plumbing of the GPU parity tests: runs the same seeded LayerInputs through the CUDA path (via the
ctypes binding of the C ABI) and through the CPU oracle, and states the acceptance rules of DESIGN.md §7
(SURVEY.md §8c "GPU-vs-oracle acceptance") in one place.  Test infrastructure only."""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import torch

from oracle import ref
from paper_2606_24957_b200 import api, synth

# Tolerances (north_star / DESIGN.md §7)
SCORE_RTOL = 1e-5          # fp32 scores vs fp64 oracle, on entries > SCORE_FLOOR
SCORE_FLOOR = 1e-30
NEAR_TIE_RTOL = 1e-5       # an index may differ only if its tier score is this close to the tier threshold
ATTN_MAX_ABS = 2e-2
ATTN_MEAN_ABS = 2e-3


def shape_of(cfg: synth.Config, sm_scale: float = 0.0) -> api.Shape:
    return api.Shape(cfg.batch, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.n_new, cfg.ctx, sm_scale)


def gpu_kv(inp: synth.LayerInputs) -> api.KV:
    if inp.page_table is not None:
        return api.KV.paged_nhd(inp.k, inp.v, inp.page_table, inp.seq_lens)
    return api.KV.contiguous_nhd(inp.k, inp.v, inp.seq_lens)


def cpu_kv(inp: synth.LayerInputs) -> ref.KV:
    if inp.page_table is not None:
        P, ps, H, d = inp.k.shape
        return ref.KV(inp.k, inp.v, ps * H * d, H * d, d, inp.page_table, ps, inp.seq_lens)
    return ref.KV.contiguous_nhd(inp.k, inp.v, inp.seq_lens)


def select_of(inp: synth.LayerInputs) -> api.Select:
    c = inp.cfg
    return api.Select(c.budget, c.n_sink, c.n_recent, c.m_num, c.m_den, c.n_lists, inp.budgets)


@dataclass
class Result:
    scores_now: torch.Tensor      # fp32 [B,G,N]
    hist: torch.Tensor            # fp32 [B,G,N] (after Eq. 5 accumulation)
    idx: torch.Tensor             # int32 [B,G,k_max]
    cnt: torch.Tensor             # int32 [B,G]
    out: torch.Tensor             # [B,T,Hq,d] (bf16 on the GPU, fp64 from the oracle)
    lse: torch.Tensor             # [B,Hq,T]


def run_gpu_staged(inp: synth.LayerInputs, alpha: float = 1.0, sm_scale: float = 0.0) -> Result:
    """a1 -> a2 -> a3 -> a4 through the four stage entry points.  `inp` lives on the GPU."""
    c = inp.cfg
    sh = shape_of(c, sm_scale)
    kv = gpu_kv(inp)
    ws = api.alloc_workspace(sh, c.head_mask, inp.k_max)
    B, G, N = c.batch, c.n_lists, c.ctx
    scores = torch.full((B, G, N), float("nan"), device="cuda")
    hist = inp.hist.clone()
    idx = torch.full((B, G, inp.k_max), -7, dtype=torch.int32, device="cuda")
    cnt = torch.full((B, G), -7, dtype=torch.int32, device="cuda")
    out = torch.full_like(inp.q, float("nan"))
    lse = torch.full((B, c.n_q_heads, c.n_new), float("nan"), device="cuda")
    api.score_heads(sh, kv, inp.q[:, 0], c.head_mask, G, scores, ws)
    api.fuse_scores(scores, hist, alpha, inp.seq_lens)
    api.topk_select(select_of(inp), inp.s_draft, hist, idx, cnt, inp.seq_lens)
    api.sparse_verify_attn(sh, kv, inp.q, inp.k_new, inp.v_new, idx, cnt, out, ws, lse)
    torch.cuda.synchronize()
    return Result(scores, hist, idx, cnt, out, lse)


def run_gpu_fused(inp: synth.LayerInputs, alpha: float = 1.0, sm_scale: float = 0.0,
                  want_scores: bool = True) -> Result:
    c = inp.cfg
    sh = shape_of(c, sm_scale)
    ws = api.alloc_workspace(sh, c.head_mask, inp.k_max)
    B, G, N = c.batch, c.n_lists, c.ctx
    scores = torch.full((B, G, N), float("nan"), device="cuda") if want_scores else None
    hist = inp.hist.clone()
    idx = torch.full((B, G, inp.k_max), -7, dtype=torch.int32, device="cuda")
    cnt = torch.full((B, G), -7, dtype=torch.int32, device="cuda")
    out = torch.full_like(inp.q, float("nan"))
    lse = torch.full((B, c.n_q_heads, c.n_new), float("nan"), device="cuda")
    api.verify_layer_fused(sh, gpu_kv(inp), inp.q, inp.k_new, inp.v_new, c.head_mask, inp.s_draft, hist, alpha,
                           select_of(inp), out, idx, cnt, ws, scores, lse)
    torch.cuda.synchronize()
    return Result(scores, hist, idx, cnt, out, lse)


def oracle_scores(inp: synth.LayerInputs, alpha: float = 1.0, sm_scale: float = 0.0):
    """(A_now, H_new) of the oracle.  `inp` lives on the CPU."""
    c = inp.cfg
    a = ref.score_heads(cpu_kv(inp), inp.q[:, 0], c.head_mask, c.n_lists, c.n_kv_heads, c.ctx, sm_scale)
    h = ref.fuse_scores(a, inp.hist, alpha, inp.seq_lens)
    return a, h


def oracle_select(inp: synth.LayerInputs, s_target: torch.Tensor):
    c = inp.cfg
    return ref.topk_select(inp.s_draft, s_target, c.budget, c.n_sink, c.n_recent, c.m_num, c.m_den, inp.k_max,
                           inp.seq_lens, inp.budgets)


def oracle_attn(inp: synth.LayerInputs, idx: Optional[torch.Tensor], cnt: Optional[torch.Tensor],
                sm_scale: float = 0.0):
    return ref.sparse_verify_attn(cpu_kv(inp), inp.q, inp.k_new, inp.v_new, idx, cnt, inp.cfg.ctx, sm_scale)


# ---- acceptance rules -------------------------------------------------------------------------------------------
def check_scores(got: torch.Tensor, want: torch.Tensor, what: str = "scores", rtol: float = SCORE_RTOL):
    got, want = got.detach().cpu().double(), want.double()
    assert torch.isfinite(got).all(), f"{what}: non-finite values"
    big = want > SCORE_FLOOR
    rel = ((got - want).abs() / want.clamp_min(1e-300))[big]
    worst = rel.max().item() if rel.numel() else 0.0
    assert worst <= rtol, f"{what}: max relative error {worst:.3e} > {rtol:.1e}"
    assert (got[~big].abs() <= 2e-30).all(), f"{what}: entries that should be ~0 are not"
    return worst


def check_attn(got: torch.Tensor, want: torch.Tensor, what: str = "attention output"):
    err = (got.detach().cpu().double() - want.double()).abs()
    assert torch.isfinite(got.float()).all(), f"{what}: non-finite values"
    mx, mean = err.max().item(), err.mean().item()
    assert mx <= ATTN_MAX_ABS, f"{what}: max-abs {mx:.3e} > {ATTN_MAX_ABS}"
    assert mean <= ATTN_MEAN_ABS, f"{what}: mean-abs {mean:.3e} > {ATTN_MEAN_ABS}"
    return mx, mean


def check_index_lists_valid(inp: synth.LayerInputs, idx: torch.Tensor, cnt: torch.Tensor):
    """What is unique about any correct answer: sizes, order, range, protected membership, -1 tail."""
    c = inp.cfg
    idx, cnt = idx.cpu(), cnt.cpu()
    B, G, K = idx.shape
    for b in range(B):
        N = int(inp.seq_lens[b]) if inp.seq_lens is not None else c.ctx
        k = int(inp.budgets[b]) if inp.budgets is not None else c.budget
        for g in range(G):
            n = int(cnt[b, g])
            assert n == min(k, N), (b, g, n, k, N)
            row = idx[b, g]
            assert (row[n:] == -1).all()
            sel = row[:n]
            if n:
                assert (sel[1:] > sel[:-1]).all() and sel[0] >= 0 and sel[-1] < N
            if k < N:
                s = set(sel.tolist())
                assert all(i in s for i in range(min(c.n_sink, N)))
                assert all(i in s for i in range(N - c.n_recent, N))


def check_near_tie_only(inp: synth.LayerInputs, got_idx, got_cnt, want_idx, want_cnt, s_target: torch.Tensor):
    """GPU lists may differ from the oracle's only at positions whose tier score lies within NEAR_TIE_RTOL
    (relative) of that tier's threshold in the ORACLE's fp32 scores (north_star).  Returns #swapped positions."""
    c = inp.cfg
    got_idx, got_cnt, want_idx, want_cnt = got_idx.cpu(), got_cnt.cpu(), want_idx.cpu(), want_cnt.cpu()
    assert torch.equal(got_cnt, want_cnt)
    B, G, K = want_idx.shape
    swaps = 0
    for b in range(B):
        N = int(inp.seq_lens[b]) if inp.seq_lens is not None else c.ctx
        k = int(inp.budgets[b]) if inp.budgets is not None else c.budget
        for g in range(G):
            if torch.equal(got_idx[b, g], want_idx[b, g]):
                continue
            n = int(want_cnt[b, g])
            a, w = set(got_idx[b, g, :n].tolist()), set(want_idx[b, g, :n].tolist())
            only_gpu, only_ref = sorted(a - w), sorted(w - a)
            assert len(only_gpu) == len(only_ref)
            swaps += len(only_gpu)
            sd = (inp.s_draft[b] if inp.s_draft.dim() == 2 else inp.s_draft[b, g]).double().clamp_min(0)
            st = s_target[b, g].double().clamp_min(0)
            # tier thresholds of the oracle's selection (recomputed from its definition: Eq. 6)
            S, W = min(c.n_sink, N), min(c.n_recent, N - min(c.n_sink, N))
            cc = k - S - W
            m = min(cc * c.m_num // c.m_den, cc)
            cand = torch.arange(S, N - W)
            wsel = torch.tensor(sorted(w), dtype=torch.long)
            wsel = wsel[(wsel >= S) & (wsel < N - W)]
            # tier 1 = the m best of the candidates by s_draft (stable): threshold t1
            order1 = cand[torch.sort(sd[cand], descending=True, stable=True).indices]
            tier1 = set(order1[:m].tolist())
            t1 = sd[order1[m - 1]].item() if m > 0 else float("inf")
            tier2 = [i for i in wsel.tolist() if i not in tier1]
            t2 = min(st[i].item() for i in tier2) if tier2 else float("inf")
            for i in only_gpu + only_ref:
                near1 = m > 0 and abs(sd[i].item() - t1) <= NEAR_TIE_RTOL * max(t1, 1e-300)
                near2 = abs(st[i].item() - t2) <= NEAR_TIE_RTOL * max(t2, 1e-300)
                assert near1 or near2, (f"row ({b},{g}) index {i}: s_draft {sd[i].item():.9e} (t1 {t1:.9e}), "
                                        f"s_target {st[i].item():.9e} (t2 {t2:.9e}) is not a near tie")
    return swaps
