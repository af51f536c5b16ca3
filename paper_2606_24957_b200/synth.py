"""Seeded synthetic inputs shaped like the paper's workloads.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's tests.  It holds no
part of the method (no scoring kernel, no selection, no attention): it draws tensors with torch's library
RNG / matmul / softmax on one device and hands the same bits to both sides.  It imports neither the CUDA
binding nor oracle/.

Stand-in statement: the paper measures on PG-19 / LongBench with Qwen2.5-72B and Llama-3.x weights
(PAPER.md:230, :256, :305-328); none of that exists here.  Only the shapes are used (head counts
PAPER.md:395, depths :457-466, context/batch grid :248, :305) with the value recipe of BASELINE.json's
configs: N(0,1) Q/K/V, a planted heavy-hitter set, draft scores correlated with the true logits, and a
slightly stale history.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import torch


@dataclass(frozen=True)
class Config:
    name: str
    batch: int
    ctx: int                      # N (max context; ragged configs draw N_b <= ctx)
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    gamma: int                    # draft depth; T = gamma + 1 verify positions
    budget: int                   # k (0 => per-sequence budgets = N_b * budget_frac)
    n_sink: int
    n_recent: int
    heads: tuple                  # the head subset (SRHs)
    n_lists: int                  # G: 1 (paper, global list) or n_kv_heads
    n_layers: int = 1
    planted_frac: float = 0.02    # fraction of positions that are heavy hitters (n_planted overrides)
    n_planted: int = 0
    drift: float = 0.10           # fraction of planted positions replaced per layer/step
    draft_noise: float = 0.5      # sigma of the N(0, sigma) noise on the draft logits (reading A19)
    tiny_recipe: bool = False     # config 1: draft = softmax(N(0,1) + 3*planted), hist = Dirichlet(0.1)
    paged: bool = False
    page_size: int = 16
    ragged_min: int = 0           # >0: N_b ~ U[ragged_min, ctx]
    budget_frac: float = 0.0      # >0: k_b = floor(N_b * budget_frac)
    m_num: int = 1                # draft quota m = floor((k-S-W) * m_num / m_den)   (reading A9)
    m_den: int = 2
    seed: int = 20260624

    @property
    def n_new(self) -> int:
        return self.gamma + 1

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def head_mask(self) -> int:
        m = 0
        for h in self.heads:
            m |= 1 << h
        return m


def spread_heads(n_q_heads: int, n_sel: int) -> tuple:
    """Subset at stride Hq/|H| (Qwen shape: one head per KV group; Llama shape: KV groups 0,2,4,6)."""
    return tuple(j * (n_q_heads // n_sel) for j in range(n_sel))


def packed_heads(n_sel: int) -> tuple:
    """Subset packed into the first KV group(s)."""
    return tuple(range(n_sel))


def config_tiny() -> Config:
    """BASELINE.json configs[0]."""
    return Config("tiny", batch=1, ctx=1024, n_q_heads=4, n_kv_heads=1, head_dim=64, gamma=4, budget=128,
                  n_sink=4, n_recent=32, heads=(0, 2), n_lists=1, n_layers=1, n_planted=8, tiny_recipe=True,
                  seed=20260624 + 1000)


def config_llama8b(batch: int = 16, ctx: int = 32768, n_layers: int = 32, spread: bool = True) -> Config:
    """BASELINE.json configs[1]: Llama-3-8B-shaped layer."""
    heads = spread_heads(32, 4) if spread else packed_heads(4)
    return Config("llama3-8b", batch=batch, ctx=ctx, n_q_heads=32, n_kv_heads=8, head_dim=128, gamma=4,
                  budget=2048, n_sink=64, n_recent=256, heads=heads, n_lists=8 if spread else 1,
                  n_layers=n_layers, seed=20260624 + 2000)


def config_qwen72b(batch: int = 16, ctx: int = 32768, n_layers: int = 80, spread: bool = True,
                   gamma: int = 4, budget: int = 2048) -> Config:
    """BASELINE.json configs[2] (and the shape of configs[3]): Qwen2.5-72B-shaped layer."""
    heads = spread_heads(64, 8) if spread else packed_heads(8)
    if budget == 2048:
        s, w = 64, 256
    else:                                    # reading A18: protected set scales with the budget
        s, w = budget // 32, budget // 8
    return Config("qwen2.5-72b", batch=batch, ctx=ctx, n_q_heads=64, n_kv_heads=8, head_dim=128, gamma=gamma,
                  budget=budget, n_sink=s, n_recent=w, heads=heads, n_lists=8 if spread else 1,
                  n_layers=n_layers, seed=20260624 + 3000)


def config_paged(batch: int = 32, ctx_min: int = 8192, ctx_max: int = 65536, n_layers: int = 1) -> Config:
    """BASELINE.json configs[4]: paged, ragged, Llama-3-8B-shaped heads, k_b = 6.25 % of N_b."""
    return Config("paged-ragged", batch=batch, ctx=ctx_max, n_q_heads=32, n_kv_heads=8, head_dim=128,
                  gamma=4, budget=0, n_sink=64, n_recent=256, heads=spread_heads(32, 4), n_lists=8,
                  n_layers=n_layers, paged=True, page_size=16, ragged_min=ctx_min, budget_frac=0.0625,
                  seed=20260624 + 5000)


@dataclass
class LayerInputs:
    cfg: Config
    q: torch.Tensor                 # bf16 [B, T, Hq, d]
    k_new: torch.Tensor             # bf16 [B, T, Hkv, d]
    v_new: torch.Tensor
    k: torch.Tensor                 # bf16 [B, N, Hkv, d]  or paged pool [n_pages, page, Hkv, d]
    v: torch.Tensor
    s_draft: torch.Tensor           # fp32 [B, N] (n_lists == 1) or [B, G, N]
    hist: torch.Tensor              # fp32 [B, G, N]
    seq_lens: Optional[torch.Tensor] = None    # int32 [B] (ragged) or None
    budgets: Optional[torch.Tensor] = None     # int32 [B] or None
    page_table: Optional[torch.Tensor] = None  # int32 [B, max_pages] or None
    planted: Optional[torch.Tensor] = None     # bool [B, Hkv, N]
    k_max: int = 0
    extras: dict = field(default_factory=dict)

    def to(self, device) -> "LayerInputs":
        kw = {}
        for name, val in self.__dict__.items():
            kw[name] = val.to(device) if isinstance(val, torch.Tensor) else val
        return LayerInputs(**kw)


def _gen(device, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _randn_bf16(shape, g, device):
    return torch.randn(shape, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)


def _planted_mask(cfg: Config, lens: torch.Tensor, g, device, layer: int) -> torch.Tensor:
    """bool [B, Hkv, N]: heavy-hitter positions inside the candidate range [S, N_b - W) of each row.
    Layer l+1 differs from layer l in a `drift` fraction of the planted set: position j is planted at layer l
    iff  u_j + drift*l (mod 1) < planted_frac' -- a sliding window over a fixed uniform field."""
    B, H, N = cfg.batch, cfg.n_kv_heads, cfg.ctx
    u = torch.rand((B, H, N), generator=g, device=device)
    pos = torch.arange(N, device=device).view(1, 1, N)
    hi = (lens.view(B, 1, 1) - cfg.n_recent).clamp(min=0)
    in_range = (pos >= cfg.n_sink) & (pos < hi)
    if cfg.n_planted > 0:
        # exactly n_planted positions per row: the smallest u inside the range
        u_masked = torch.where(in_range, u, torch.full_like(u, 2.0))
        thr = torch.kthvalue(u_masked, cfg.n_planted, dim=-1, keepdim=True).values
        return (u_masked <= thr) & in_range
    frac = cfg.planted_frac
    shifted = (u + cfg.drift * frac * layer) % 1.0
    return (shifted < frac) & in_range


def make_layer(cfg: Config, layer: int = 0, device="cpu", want_hist_draft: bool = True) -> LayerInputs:
    """All inputs of one decoder layer's sparse verification, seeded by (cfg.seed, layer)."""
    device = torch.device(device)
    g = _gen(device, cfg.seed + layer)
    B, N, Hq, Hkv, d, T, r = cfg.batch, cfg.ctx, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.n_new, cfg.group

    if cfg.ragged_min > 0:
        lens = torch.randint(cfg.ragged_min, N + 1, (B,), generator=_gen("cpu", cfg.seed + 7), dtype=torch.int64)
        lens = lens.to(device)
        seq_lens = lens.to(torch.int32)
    else:
        lens = torch.full((B,), N, dtype=torch.int64, device=device)
        seq_lens = None
    budgets = None
    k_max = cfg.budget
    if cfg.budget_frac > 0:
        budgets = (lens.double() * cfg.budget_frac).floor().to(torch.int32)
        k_max = int(math.floor(N * cfg.budget_frac))

    # heavy-hitter direction per (b, KV group); queries lean on it, planted keys align with it (scale 4)
    u_dir = torch.randn((B, Hkv, d), generator=g, device=device)
    u_dir = u_dir / u_dir.norm(dim=-1, keepdim=True)
    planted = _planted_mask(cfg, lens, _gen(device, cfg.seed + 100003), device, layer)   # same field every layer
    planted_prev = _planted_mask(cfg, lens, _gen(device, cfg.seed + 100003), device, layer - 1)

    q32 = torch.randn((B, T, Hq, d), generator=g, device=device)
    q32 = q32 + math.sqrt(d) * u_dir.repeat_interleave(r, dim=1).view(B, 1, Hq, d)
    q = q32.to(torch.bfloat16)
    del q32
    k = torch.randn((B, N, Hkv, d), generator=g, device=device)
    k += 4.0 * planted.permute(0, 2, 1).unsqueeze(-1) * u_dir.view(B, 1, Hkv, d)
    k = k.to(torch.bfloat16)
    v = _randn_bf16((B, N, Hkv, d), g, device)
    k_new = _randn_bf16((B, T, Hkv, d), g, device)
    v_new = _randn_bf16((B, T, Hkv, d), g, device)

    G = cfg.n_lists
    s_draft = hist = None
    if want_hist_draft:
        pos = torch.arange(N, device=device).view(1, 1, N)
        valid = pos < lens.view(B, 1, 1)
        if cfg.tiny_recipe:
            # draft: softmax_n(N(0,1) + 3*[planted]); history: Dirichlet(0.1) over positions
            pl = planted.any(dim=1)                                          # [B, N]
            logit = torch.randn((B, N), generator=g, device=device) + 3.0 * pl
            logit = logit.masked_fill(~valid[:, 0], float("-inf"))
            s_draft = torch.softmax(logit, dim=-1)
            conc = torch.full((B, G, N), 0.1, device=device)
            gam = torch._standard_gamma(conc, generator=g)
            gam = gam * valid
            hist = (gam / gam.sum(-1, keepdim=True)).float()
        else:
            # true position-0 logits (input generation only): [B, Hq, N]
            logits = _logits_chunked(q[:, 0], k, r) / math.sqrt(d)
            grp = logits.view(B, Hkv, r, N).mean(dim=2)                      # [B, Hkv, N]
            noise = cfg.draft_noise * torch.randn((B, Hkv, N), generator=g, device=device)
            dl = (grp + noise).masked_fill(~valid, float("-inf"))
            sd = torch.softmax(dl, dim=-1)                                   # [B, Hkv, N]
            s_draft = sd if G == Hkv else sd.mean(dim=1)
            # stale history: the subset heads' attention of the previous drift step (boost moved at logit level)
            delta = 4.0 * (planted_prev.float() - planted.float())          # [B, Hkv, N]
            hsum = torch.zeros((B, Hkv, N), device=device)
            hall = torch.zeros((B, N), device=device)
            for h in cfg.heads:
                gidx = h // r
                lp = (logits[:, h] + delta[:, gidx]).masked_fill(~valid[:, 0], float("-inf"))
                p = torch.softmax(lp, dim=-1)
                hsum[:, gidx] += p
                hall += p
            if G == 1:
                hist = hall.view(B, 1, N)
            else:
                has = torch.zeros(Hkv, dtype=torch.bool, device=device)
                for h in cfg.heads:
                    has[h // r] = True
                hist = torch.where(has.view(1, Hkv, 1), hsum, hall.view(B, 1, N).expand(B, Hkv, N))
            del logits
        s_draft = s_draft.float().contiguous()
        hist = hist.float().contiguous()

    page_table = None
    if cfg.paged:
        k, v, page_table = _to_paged(cfg, k, v, lens, device)

    return LayerInputs(cfg=cfg, q=q.contiguous(), k_new=k_new, v_new=v_new, k=k, v=v, s_draft=s_draft, hist=hist,
                       seq_lens=seq_lens, budgets=budgets, page_table=page_table, planted=planted, k_max=k_max)


def _logits_chunked(q0: torch.Tensor, k: torch.Tensor, r: int) -> torch.Tensor:
    """q0 [B, Hq, d] bf16, k [B, N, Hkv, d] bf16 -> fp32 [B, Hq, N], one sequence at a time."""
    B, Hq, d = q0.shape
    N, Hkv = k.shape[1], k.shape[2]
    out = torch.empty((B, Hq, N), dtype=torch.float32, device=k.device)
    for b in range(B):
        qb = q0[b].float().view(Hkv, r, d)                    # [Hkv, r, d]
        kb = k[b].float().permute(1, 2, 0)                    # [Hkv, d, N]
        out[b] = torch.bmm(qb, kb).view(Hq, N)
    return out


def _to_paged(cfg: Config, k: torch.Tensor, v: torch.Tensor, lens: torch.Tensor, device):
    """Scatter the logical [B, N, Hkv, d] caches into a page pool [n_pages, page, Hkv, d] under a random
    permutation of pages; returns (k_pool, v_pool, page_table int32 [B, max_pages])."""
    B, N, Hkv, d = k.shape
    ps = cfg.page_size
    max_pages = (N + ps - 1) // ps
    n_pages_b = ((lens + ps - 1) // ps).cpu()
    total = int(n_pages_b.sum())
    perm = torch.randperm(total, generator=_gen("cpu", cfg.seed + 11))
    page_table = torch.zeros((B, max_pages), dtype=torch.int32)
    k_pool = torch.zeros((total, ps, Hkv, d), dtype=k.dtype, device=device)
    v_pool = torch.zeros((total, ps, Hkv, d), dtype=v.dtype, device=device)
    off = 0
    pad = max_pages * ps - N
    for b in range(B):
        nb = int(n_pages_b[b])
        ids = perm[off:off + nb]
        off += nb
        page_table[b, :nb] = ids.to(torch.int32)
        kb, vb = k[b], v[b]
        if pad:
            kb = torch.cat([kb, torch.zeros((pad, Hkv, d), dtype=k.dtype, device=device)])
            vb = torch.cat([vb, torch.zeros((pad, Hkv, d), dtype=v.dtype, device=device)])
        k_pool[ids.to(device)] = kb.view(max_pages, ps, Hkv, d)[:nb]
        v_pool[ids.to(device)] = vb.view(max_pages, ps, Hkv, d)[:nb]
    return k_pool, v_pool, page_table.to(device)


def shrink(cfg: Config, **kw) -> Config:
    """A smaller copy of a named config for element-by-element parity tests (same shape family)."""
    return replace(cfg, **kw)
