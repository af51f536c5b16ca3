"""ctypes front end of the CPU oracle (oracle/dustin_ref.cpp) -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It never imports the CUDA package.  Arguments are torch CPU tensors (bf16 tensors are passed as
their raw 16-bit patterns); results are fresh torch CPU tensors.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dustin_ref.cpp")
_LIB = os.path.join(_HERE, "libdustin_ref.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c++17", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.dustin_ref_threads.restype = ctypes.c_int
    return _lib


def threads() -> int:
    return int(lib().dustin_ref_threads())


@dataclass
class KV:
    """Host view of a bf16 KV cache.  Strides are in elements.  page_table=None: contiguous, sequence b starts
    at b*stride_seq; else row (b,n) lives in page page_table[b, n // page_size] at offset n % page_size and
    stride_seq is the page stride."""
    k: torch.Tensor
    v: Optional[torch.Tensor]
    stride_seq: int
    stride_token: int
    stride_head: int
    page_table: Optional[torch.Tensor] = None
    page_size: int = 0
    seq_lens: Optional[torch.Tensor] = None

    @staticmethod
    def contiguous_nhd(k: torch.Tensor, v: Optional[torch.Tensor], seq_lens=None) -> "KV":
        """k, v: [B, N, Hkv, d] bf16."""
        B, N, H, d = k.shape
        return KV(k, v, N * H * d, H * d, d, None, 0, seq_lens)


def _p(t: Optional[torch.Tensor], typ=ctypes.c_void_p):
    if t is None:
        return typ(None) if typ is ctypes.c_void_p else None
    assert t.device.type == "cpu" and t.is_contiguous()
    return ctypes.c_void_p(t.data_ptr())


def _i32(t):
    if t is None:
        return None
    assert t.dtype == torch.int32 and t.is_contiguous()
    return t


def _bits(t: torch.Tensor) -> torch.Tensor:
    assert t.dtype == torch.bfloat16 and t.device.type == "cpu" and t.is_contiguous()
    return t


def _f32(t: torch.Tensor) -> torch.Tensor:
    assert t.dtype == torch.float32 and t.device.type == "cpu" and t.is_contiguous()
    return t


def score_heads(kv: KV, q: torch.Tensor, head_mask: int, n_lists: int, n_kv_heads: int, max_ctx: int,
                sm_scale: float = 0.0) -> torch.Tensor:
    """q: [B, Hq, d] bf16 (the scored verify position).  Returns fp32 [B, n_lists, max_ctx]."""
    B, Hq, d = q.shape
    assert q.dtype == torch.bfloat16 and q.device.type == "cpu" and q.stride(2) == 1   # strided view allowed
    k = _bits(kv.k)
    pt, sl = _i32(kv.page_table), _i32(kv.seq_lens)
    out = torch.zeros(B, n_lists, max_ctx, dtype=torch.float32)
    rc = lib().dustin_ref_score_heads(
        ctypes.c_int(B), ctypes.c_int(Hq), ctypes.c_int(n_kv_heads), ctypes.c_int(d), ctypes.c_int(max_ctx),
        ctypes.c_float(sm_scale), _p(k), ctypes.c_int64(kv.stride_seq), ctypes.c_int64(kv.stride_token),
        ctypes.c_int64(kv.stride_head), _p(pt), ctypes.c_int(kv.page_size),
        ctypes.c_int(0 if pt is None else pt.shape[1]), _p(sl), ctypes.c_void_p(q.data_ptr()),
        ctypes.c_int64(q.stride(0)), ctypes.c_int64(q.stride(1)), ctypes.c_uint64(head_mask), ctypes.c_int(n_lists), _p(out))
    if rc != 0:
        raise ValueError(f"dustin_ref_score_heads: status {rc}")
    return out


def fuse_scores(scores_now: torch.Tensor, hist: torch.Tensor, alpha: float, seq_lens=None) -> torch.Tensor:
    """Returns the new history alpha*hist + scores_now (fp32 [B, G, N]); inputs are not modified."""
    B, G, N = scores_now.shape
    h = hist.contiguous().clone()
    rc = lib().dustin_ref_fuse_scores(ctypes.c_int(B), ctypes.c_int(G), ctypes.c_int(N), _p(_i32(seq_lens)),
                                      _p(_f32(scores_now)), _p(h), ctypes.c_float(alpha))
    if rc != 0:
        raise ValueError(f"dustin_ref_fuse_scores: status {rc}")
    return h


def topk_select(s_draft: torch.Tensor, s_target: torch.Tensor, budget: int, n_sink: int, n_recent: int,
                m_num: int, m_den: int, k_max: Optional[int] = None, seq_lens=None, budgets=None):
    """s_target: fp32 [B, G, N]; s_draft: fp32 [B, N] (broadcast over lists) or [B, G, N].
    Returns (idx int32 [B, G, k_max] ascending with -1 tail, cnt int32 [B, G])."""
    B, G, N = s_target.shape
    if k_max is None:
        k_max = int(budgets.max()) if budgets is not None else budget
    dls = 0 if s_draft.dim() == 2 else N
    idx = torch.full((B, G, k_max), -1, dtype=torch.int32)
    cnt = torch.zeros(B, G, dtype=torch.int32)
    rc = lib().dustin_ref_topk_select(
        ctypes.c_int(B), ctypes.c_int(N), _p(_i32(seq_lens)), ctypes.c_int(budget), _p(_i32(budgets)),
        ctypes.c_int(n_sink), ctypes.c_int(n_recent), ctypes.c_int(m_num), ctypes.c_int(m_den),
        ctypes.c_int(G), _p(_f32(s_draft)), ctypes.c_int64(dls), _p(_f32(s_target)),
        _p(idx), _p(cnt), ctypes.c_int(k_max))
    if rc != 0:
        raise ValueError(f"dustin_ref_topk_select: status {rc}")
    return idx, cnt


def sparse_verify_attn(kv: KV, q: torch.Tensor, k_new: torch.Tensor, v_new: torch.Tensor,
                       idx: Optional[torch.Tensor], cnt: Optional[torch.Tensor], max_ctx: int,
                       sm_scale: float = 0.0):
    """q: [B,T,Hq,d] bf16; k_new, v_new: [B,T,Hkv,d] bf16; idx int32 [B,G,k_max] or None (dense).
    Returns (out fp64 [B,T,Hq,d], lse fp64 [B,Hq,T])."""
    B, T, Hq, d = q.shape
    Hkv = k_new.shape[2]
    if idx is not None:
        G, k_max = idx.shape[1], idx.shape[2]
        idx, cnt = _i32(idx), _i32(cnt)
    else:
        G, k_max = 1, 0
    pt, sl = _i32(kv.page_table), _i32(kv.seq_lens)
    out = torch.zeros(B, T, Hq, d, dtype=torch.float64)
    lse = torch.zeros(B, Hq, T, dtype=torch.float64)
    rc = lib().dustin_ref_sparse_verify_attn(
        ctypes.c_int(B), ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(T),
        ctypes.c_int(max_ctx), ctypes.c_float(sm_scale), _p(_bits(kv.k)), _p(_bits(kv.v)),
        ctypes.c_int64(kv.stride_seq), ctypes.c_int64(kv.stride_token), ctypes.c_int64(kv.stride_head),
        _p(pt), ctypes.c_int(kv.page_size), ctypes.c_int(0 if pt is None else pt.shape[1]), _p(sl),
        _p(_bits(q)), _p(_bits(k_new)), _p(_bits(v_new)), _p(idx), _p(cnt), ctypes.c_int(G),
        ctypes.c_int(k_max), _p(out), _p(lse))
    if rc != 0:
        raise ValueError(f"dustin_ref_sparse_verify_attn: status {rc}")
    return out, lse


def arr(a: torch.Tensor, idx: torch.Tensor, cnt: torch.Tensor, seq_lens=None) -> torch.Tensor:
    """Eq. 1.  a: fp32 [B, G, N] non-negative weights; idx int32 [B, G, k_max] distinct entries;
    cnt int32 [B, G].  Returns fp64 [B, G]."""
    B, G, N = a.shape
    out = torch.zeros(B, G, dtype=torch.float64)
    rc = lib().dustin_ref_arr(ctypes.c_int(B), ctypes.c_int(G), ctypes.c_int(N), _p(_i32(seq_lens)), _p(_f32(a)),
                              _p(_i32(idx)), _p(_i32(cnt)), ctypes.c_int(idx.shape[2]), _p(out))
    if rc != 0:
        raise ValueError(f"dustin_ref_arr: status {rc}")
    return out


def append_kv(kv: KV, seq_lens: torch.Tensor, k_new: torch.Tensor, v_new: torch.Tensor, n_append: torch.Tensor,
              max_ctx: int, hist: Optional[torch.Tensor] = None):
    """PAPER.md:153.  Writes the first n_append[b] rows of k_new / v_new ([B,T,Hkv,d] bf16) behind sequence b IN PLACE
    in kv.k / kv.v, zeroes the new positions of hist ([B,G,max_ctx] fp32, in place) and returns the new int32 lengths."""
    B, T, Hkv, d = k_new.shape
    lens = seq_lens.to(torch.int32).contiguous().clone()
    assert kv.k.is_contiguous() and kv.v.is_contiguous() and (hist is None or hist.is_contiguous())
    pt = _i32(kv.page_table)
    rc = lib().dustin_ref_append_kv(
        ctypes.c_int(B), ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(T), ctypes.c_int(max_ctx),
        ctypes.c_void_p(kv.k.data_ptr()), ctypes.c_void_p(kv.v.data_ptr()), ctypes.c_int64(kv.stride_seq),
        ctypes.c_int64(kv.stride_token), ctypes.c_int64(kv.stride_head), _p(pt), ctypes.c_int(kv.page_size),
        ctypes.c_int(0 if pt is None else pt.shape[1]), _p(lens), _p(_bits(k_new)), _p(_bits(v_new)),
        _p(_i32(n_append)), _p(hist), ctypes.c_int(0 if hist is None else hist.shape[1]))
    if rc != 0:
        raise ValueError(f"dustin_ref_append_kv: status {rc}")
    return lens


def draft_aggregate(layer_k: list, layer_q: list, head_mask: int, n_kv_heads: int, max_ctx: int, stride_seq: int,
                    stride_token: int, stride_head: int, page_table=None, page_size: int = 0, seq_lens=None,
                    sm_scale: float = 0.0) -> torch.Tensor:
    """Eq. 5, first line.  layer_k[l]: bf16 K cache of draft layer l (all layers share the
    strides / page table); layer_q[l]: bf16 [B, Gamma, Hq, d].  Returns S_Draft fp32 [B, max_ctx]."""
    B, n_gamma, Hq, d = layer_q[0].shape
    L = len(layer_k)
    ks = [_bits(k) for k in layer_k]
    qs = [_bits(q) for q in layer_q]
    karr = (ctypes.c_void_p * L)(*[k.data_ptr() for k in ks])
    qarr = (ctypes.c_void_p * L)(*[q.data_ptr() for q in qs])
    pt = _i32(page_table)
    out = torch.zeros(B, max_ctx, dtype=torch.float32)
    rc = lib().dustin_ref_draft_aggregate(
        ctypes.c_int(B), ctypes.c_int(Hq), ctypes.c_int(n_kv_heads), ctypes.c_int(d), ctypes.c_int(n_gamma),
        ctypes.c_int(max_ctx), ctypes.c_float(sm_scale), ctypes.c_int(L), karr, ctypes.c_int64(stride_seq),
        ctypes.c_int64(stride_token), ctypes.c_int64(stride_head), _p(pt), ctypes.c_int(page_size),
        ctypes.c_int(0 if pt is None else pt.shape[1]), _p(_i32(seq_lens)), qarr, ctypes.c_uint64(head_mask), _p(out))
    if rc != 0:
        raise ValueError(f"dustin_ref_draft_aggregate: status {rc}")
    return out


def quest_page_minmax(kv: KV, n_kv_heads: int, max_ctx: int, quest_page: int = 16):
    """O8: per-page, per-channel min / max of the keys.  Returns (kmin, kmax), fp64
    [B, ceil(max_ctx / quest_page), Hkv, d]; B and d are taken from the (contiguous or paged) cache tensor."""
    k = _bits(kv.k)
    d = k.shape[-1]
    pt, sl = _i32(kv.page_table), _i32(kv.seq_lens)
    B = pt.shape[0] if pt is not None else k.shape[0]
    n_pages = (max_ctx + quest_page - 1) // quest_page
    kmin = torch.zeros(B, n_pages, n_kv_heads, d, dtype=torch.float64)
    kmax = torch.zeros_like(kmin)
    rc = lib().dustin_ref_quest_page_minmax(
        ctypes.c_int(B), ctypes.c_int(n_kv_heads), ctypes.c_int(d), ctypes.c_int(max_ctx), _p(k),
        ctypes.c_int64(kv.stride_seq), ctypes.c_int64(kv.stride_token), ctypes.c_int64(kv.stride_head), _p(pt),
        ctypes.c_int(kv.page_size), ctypes.c_int(0 if pt is None else pt.shape[1]), _p(sl), ctypes.c_int(quest_page),
        _p(kmin), _p(kmax))
    if rc != 0:
        raise ValueError(f"dustin_ref_quest_page_minmax: status {rc}")
    return kmin, kmax


def quest_score_pages(kmin: torch.Tensor, kmax: torch.Tensor, q: torch.Tensor, head_mask: int, n_lists: int,
                      max_ctx: int, quest_page: int = 16, seq_lens=None, sm_scale: float = 0.0, want_ub: bool = False):
    """O9 (readings A20 / A21).  q: [B, Hq, d] bf16.  Returns fp32 [B, n_lists, n_pages] page
    scores (and, with want_ub, the fp64 [B, Hq, n_pages] upper-bound logits of the subset heads)."""
    B, Hq, d = q.shape
    assert q.dtype == torch.bfloat16 and q.device.type == "cpu" and q.stride(2) == 1
    n_pages, Hkv = kmin.shape[1], kmin.shape[2]
    assert kmin.dtype == torch.float64 and kmin.is_contiguous() and kmax.is_contiguous() and kmax.shape == kmin.shape
    assert n_pages == (max_ctx + quest_page - 1) // quest_page
    out = torch.zeros(B, n_lists, n_pages, dtype=torch.float32)
    ub = torch.zeros(B, Hq, n_pages, dtype=torch.float64) if want_ub else None
    rc = lib().dustin_ref_quest_score_pages(
        ctypes.c_int(B), ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(max_ctx),
        ctypes.c_float(sm_scale), _p(_i32(seq_lens)), ctypes.c_int(quest_page), _p(kmin), _p(kmax),
        ctypes.c_void_p(q.data_ptr()), ctypes.c_int64(q.stride(0)), ctypes.c_int64(q.stride(1)),
        ctypes.c_uint64(head_mask), ctypes.c_int(n_lists), _p(out), _p(ub))
    if rc != 0:
        raise ValueError(f"dustin_ref_quest_score_pages: status {rc}")
    return (out, ub) if want_ub else out
