"""Thin ctypes binding of libdustin.so (include/dustin.h) -- argument marshalling only.

Every function here has the name of the C entry point it calls (minus the `dustin_` prefix), takes torch CUDA
tensors for device buffers, enqueues on torch's current stream and returns without synchronising.  No step of
the path is computed in Python or by torch ops: torch only owns the device memory and the stream.
A missing or unloadable libdustin.so is a hard error; there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdustin.so")
_lib = None

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA, ERR_STATIC_SCRATCH = 0, -1, -2, -3, -4, -5
STATIC_SCRATCH_BYTES = 16 * 1024 * 1024     # DUSTIN_STATIC_SCRATCH_BYTES (dustin.h)


class DustinError(RuntimeError):
    def __init__(self, fn: str, status: int):
        self.status = status
        msg = lib().dustin_status_string(status).decode()
        if status == ERR_CUDA:
            msg += f" [cudaError {lib().dustin_last_cuda_error()}]"
        super().__init__(f"{fn}: {msg} ({status})")


class Shape(ctypes.Structure):
    _fields_ = [("batch", ctypes.c_int32), ("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("n_new", ctypes.c_int32), ("max_ctx", ctypes.c_int32),
                ("sm_scale", ctypes.c_float)]


class _Kv(ctypes.Structure):
    _fields_ = [("k", ctypes.c_void_p), ("v", ctypes.c_void_p), ("stride_seq", ctypes.c_int64),
                ("stride_token", ctypes.c_int64), ("stride_head", ctypes.c_int64), ("page_table", ctypes.c_void_p),
                ("page_size", ctypes.c_int32), ("max_pages", ctypes.c_int32), ("seq_lens", ctypes.c_void_p)]


class _Select(ctypes.Structure):
    _fields_ = [("budget", ctypes.c_int32), ("budgets", ctypes.c_void_p), ("n_sink", ctypes.c_int32),
                ("n_recent", ctypes.c_int32), ("m_num", ctypes.c_int32), ("m_den", ctypes.c_int32),
                ("n_lists", ctypes.c_int32)]


def lib():
    """Loads libdustin.so (built in-tree by paper_2606_24957_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_24957_b200.build` "
                              "(the CUDA path has no fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64, u64, f32, sz = (ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_uint64,
                                      ctypes.c_float, ctypes.c_size_t)
        sp, kp, selp = ctypes.POINTER(Shape), ctypes.POINTER(_Kv), ctypes.POINTER(_Select)
        L.dustin_version.restype = ctypes.c_int
        L.dustin_version.argtypes = []
        L.dustin_status_string.restype = ctypes.c_char_p
        L.dustin_status_string.argtypes = [ctypes.c_int]
        L.dustin_last_cuda_error.restype = ctypes.c_int
        L.dustin_last_cuda_error.argtypes = []
        L.dustin_tune_attn_split_tokens.restype = None
        L.dustin_tune_attn_split_tokens.argtypes = [i32]
        L.dustin_tune_attn_impl.restype = None
        L.dustin_tune_attn_impl.argtypes = [i32]
        L.dustin_tune_set.restype = None
        L.dustin_tune_set.argtypes = [i32, i32]
        L.dustin_tune_get.restype = i32
        L.dustin_tune_get.argtypes = [i32]
        L.dustin_debug_trace_buffer.restype = None
        L.dustin_debug_trace_buffer.argtypes = [vp, sz]
        L.dustin_debug_occupy.restype = ctypes.c_int
        L.dustin_debug_occupy.argtypes = [i32, i32, i32, i32, vp]
        L.dustin_launch_count.restype = ctypes.c_uint64
        L.dustin_launch_count.argtypes = []
        L.dustin_profile_enable.restype = None
        L.dustin_profile_enable.argtypes = [i32]
        L.dustin_profile_collect.restype = ctypes.c_int
        L.dustin_profile_collect.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)]
        L.dustin_kernel_name.restype = ctypes.c_char_p
        L.dustin_kernel_name.argtypes = [i32]
        L.dustin_workspace_bytes.restype = sz
        L.dustin_workspace_bytes.argtypes = [sp, u64, i32]
        L.dustin_score_heads.restype = ctypes.c_int
        L.dustin_score_heads.argtypes = [sp, kp, vp, i64, i64, u64, i32, vp, vp, sz, vp]
        L.dustin_score_heads_static.restype = ctypes.c_int
        L.dustin_score_heads_static.argtypes = [sp, kp, vp, i64, i64, u64, i32, vp, vp]
        L.dustin_fuse_scores.restype = ctypes.c_int
        L.dustin_fuse_scores.argtypes = [i32, i32, i32, vp, vp, vp, f32, vp]
        L.dustin_topk_select.restype = ctypes.c_int
        L.dustin_topk_select.argtypes = [i32, i32, vp, selp, vp, i64, vp, vp, vp, i32, vp]
        L.dustin_sparse_verify_attn.restype = ctypes.c_int
        L.dustin_sparse_verify_attn.argtypes = [sp, kp, vp, vp, vp, vp, vp, i32, i32, vp, vp, vp, sz, vp]
        L.dustin_verify_layer_fused.restype = ctypes.c_int
        L.dustin_verify_layer_fused.argtypes = [sp, kp, vp, vp, vp, u64, vp, i64, vp, f32, selp, i32, vp, vp, vp,
                                                vp, vp, vp, sz, vp]
        L.dustin_probe_gather.restype = ctypes.c_int
        L.dustin_probe_gather.argtypes = [sp, kp, vp, vp, i32, i32, vp, sz, vp]
        L.dustin_debug_block_scan.restype = ctypes.c_int
        L.dustin_debug_block_scan.argtypes = [i32, i32, vp, vp, vp, vp]
        L.dustin_arr.restype = ctypes.c_int
        L.dustin_arr.argtypes = [i32, i32, i32, vp, vp, vp, vp, i32, vp, vp]
        L.dustin_append_kv.restype = ctypes.c_int
        L.dustin_append_kv.argtypes = [sp, kp, vp, vp, vp, vp, vp, i32, vp]
        L.dustin_prefer_dense.restype = ctypes.c_int
        L.dustin_prefer_dense.argtypes = [sp, u64, i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        L.dustin_quest_meta_bytes.restype = sz
        L.dustin_quest_meta_bytes.argtypes = [sp]
        L.dustin_quest_build_pages.restype = ctypes.c_int
        L.dustin_quest_build_pages.argtypes = [sp, kp, vp, vp, vp]
        L.dustin_quest_score_pages.restype = ctypes.c_int
        L.dustin_quest_score_pages.argtypes = [sp, vp, vp, vp, i64, i64, u64, i32, vp, vp, vp, sz, vp]
        L.dustin_draft_workspace_bytes.restype = sz
        L.dustin_draft_workspace_bytes.argtypes = [sp, u64]
        L.dustin_draft_aggregate.restype = ctypes.c_int
        L.dustin_draft_aggregate.argtypes = [sp, kp, ctypes.POINTER(vp), i32, u64, vp, vp, sz, vp]
        _lib = L
    return _lib


N_KERNELS = 13

# include/dustin.h (the product surface) ...
EXPORTS = ("dustin_version", "dustin_status_string", "dustin_last_cuda_error",
           "dustin_workspace_bytes", "dustin_score_heads", "dustin_fuse_scores", "dustin_topk_select",
           "dustin_sparse_verify_attn", "dustin_verify_layer_fused", "dustin_arr", "dustin_append_kv",
           "dustin_draft_workspace_bytes", "dustin_draft_aggregate", "dustin_score_heads_static",
           "dustin_quest_meta_bytes", "dustin_quest_build_pages", "dustin_quest_score_pages", "dustin_prefer_dense")
# ... and include/dustin_debug.h (measurement / tuning / testing aids)
DEBUG_EXPORTS = ("dustin_tune_attn_split_tokens", "dustin_tune_attn_impl", "dustin_tune_set", "dustin_tune_get",
                 "dustin_debug_trace_buffer", "dustin_launch_count", "dustin_profile_enable", "dustin_profile_collect",
                 "dustin_kernel_name", "dustin_probe_gather", "dustin_debug_occupy", "dustin_debug_block_scan")

# enum dustin_knob (dustin_debug.h)
(KNOB_PDL, KNOB_FUSED_ROWS, KNOB_ATTN_TRACE, KNOB_SELECT_SPLIT, KNOB_DRAFT_HOIST, KNOB_SCORE_CHUNK, KNOB_SELECT_TRACE,
 KNOB_L2_HYGIENE) = range(8)


@dataclass
class KV:
    """Device view of a bf16 GQA KV cache (dustin_kv_t).  Strides in elements."""
    k: torch.Tensor
    v: Optional[torch.Tensor]
    stride_seq: int
    stride_token: int
    stride_head: int
    page_table: Optional[torch.Tensor] = None     # int32 [B, max_pages]
    page_size: int = 0
    seq_lens: Optional[torch.Tensor] = None       # int32 [B]

    @staticmethod
    def contiguous_nhd(k, v, seq_lens=None) -> "KV":
        """k, v: [B, N, Hkv, d] bf16."""
        B, N, H, d = k.shape
        return KV(k, v, N * H * d, H * d, d, None, 0, seq_lens)

    @staticmethod
    def contiguous_hnd(k, v, seq_lens=None) -> "KV":
        """k, v: [B, Hkv, N, d] bf16."""
        B, H, N, d = k.shape
        return KV(k, v, H * N * d, d, N * d, None, 0, seq_lens)

    @staticmethod
    def paged_nhd(k_pool, v_pool, page_table, seq_lens=None) -> "KV":
        """k_pool, v_pool: [n_pages, page_size, Hkv, d] bf16; page_table int32 [B, max_pages]."""
        P, ps, H, d = k_pool.shape
        return KV(k_pool, v_pool, ps * H * d, H * d, d, page_table, ps, seq_lens)

    def c(self) -> _Kv:
        pt = self.page_table
        return _Kv(_ptr(self.k, torch.bfloat16), _ptr(self.v, torch.bfloat16), self.stride_seq, self.stride_token,
                   self.stride_head, _ptr(pt, torch.int32), self.page_size, 0 if pt is None else pt.shape[1],
                   _ptr(self.seq_lens, torch.int32))


@dataclass
class Select:
    """dustin_select_t: Eq. 6 parameters."""
    budget: int
    n_sink: int
    n_recent: int
    m_num: int = 1
    m_den: int = 2
    n_lists: int = 1
    budgets: Optional[torch.Tensor] = None        # int32 [B] device

    def c(self) -> _Select:
        return _Select(self.budget, _ptr(self.budgets, torch.int32), self.n_sink, self.n_recent, self.m_num,
                       self.m_den, self.n_lists)


def _ptr(t: Optional[torch.Tensor], dtype=None):
    if t is None:
        return None
    if not t.is_cuda:
        raise TypeError("device buffers must be CUDA tensors (there is no CPU path)")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected {dtype}, got {t.dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _dense(t: torch.Tensor, dtype):
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return _ptr(t, dtype)


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(fn: str, rc: int):
    if rc != OK:
        raise DustinError(fn, rc)


def version() -> int:
    return int(lib().dustin_version())


def tune_attn_split_tokens(split_tokens: int) -> None:
    lib().dustin_tune_attn_split_tokens(int(split_tokens))


def tune_attn_impl(impl: int) -> None:
    """0 = automatic, 1 = mma.sync cluster kernel, 2 = tcgen05 kernel where usable (dustin_tune_attn_impl)."""
    lib().dustin_tune_attn_impl(int(impl))


def tune_set(knob: int, value: int) -> None:
    """dustin_tune_set (dustin_debug.h): process-wide A/B switch."""
    lib().dustin_tune_set(int(knob), int(value))


def tune_get(knob: int) -> int:
    return int(lib().dustin_tune_get(int(knob)))


def debug_trace_buffer(buf: Optional[torch.Tensor]) -> None:
    """Attach (or, with None, detach) the device buffer that receives the DUSTIN_KNOB_SELECT_TRACE timestamps."""
    if buf is None:
        lib().dustin_debug_trace_buffer(None, 0)
    else:
        lib().dustin_debug_trace_buffer(_ptr(buf), buf.numel() * buf.element_size())


def debug_occupy(n_ctas: int, threads: int, smem_bytes: int, microseconds: int, stream=None) -> None:
    """dustin_debug_occupy: CTAs that hold SM resources for a while (occupancy experiments)."""
    st = ctypes.c_void_p((stream or torch.cuda.current_stream()).cuda_stream)
    _check("dustin_debug_occupy", lib().dustin_debug_occupy(n_ctas, threads, smem_bytes, microseconds, st))


def debug_block_scan(threads: int, values: torch.Tensor):
    """dustin_debug_block_scan: values int32 [n_blocks, threads] (bit patterns of uint32) -> (prefixes int32
    [2, n_blocks, threads], totals int32 [2, n_blocks]) of v and v + 1, by the `threads`-wide selection-kernel scan."""
    n_blocks = values.shape[0]
    if values.shape[1] != threads:
        raise ValueError("values must be [n_blocks, threads]")
    out = torch.empty((2, n_blocks, threads), dtype=torch.int32, device=values.device)
    total = torch.empty((2, n_blocks), dtype=torch.int32, device=values.device)
    _check("dustin_debug_block_scan", lib().dustin_debug_block_scan(threads, n_blocks, _dense(values, torch.int32),
                                                                    _ptr(out), _ptr(total), _stream()))
    return out, total


def launch_count() -> int:
    return int(lib().dustin_launch_count())


def profile_enable(on: bool) -> None:
    lib().dustin_profile_enable(1 if on else 0)


def profile_collect() -> dict:
    """{kernel name: (total ms, launches)} of everything launched since profile_enable(True); synchronises."""
    ms = (ctypes.c_double * N_KERNELS)()
    n = (ctypes.c_int64 * N_KERNELS)()
    _check("dustin_profile_collect", lib().dustin_profile_collect(ms, n))
    return {lib().dustin_kernel_name(i).decode(): (float(ms[i]), int(n[i])) for i in range(N_KERNELS)}


def workspace_bytes(shape: Shape, head_mask: int = 0, k_max: int = 0) -> int:
    n = int(lib().dustin_workspace_bytes(ctypes.byref(shape), ctypes.c_uint64(head_mask), int(k_max)))
    if n == 0:
        raise DustinError("dustin_workspace_bytes", ERR_INVALID_ARG)
    return n


def alloc_workspace(shape: Shape, head_mask: int = 0, k_max: int = 0, device="cuda") -> torch.Tensor:
    """A uint8 device buffer of dustin_workspace_bytes (torch allocations are 512-byte aligned), zeroed: the first
    DUSTIN_WS_HEADER_BYTES must be zero before the first call (dustin.h, "Workspace")."""
    return torch.zeros(workspace_bytes(shape, head_mask, k_max), dtype=torch.uint8, device=device)


def score_heads(shape: Shape, kv: KV, q: torch.Tensor, head_mask: int, n_lists: int, scores_now: torch.Tensor,
                ws: torch.Tensor) -> None:
    """q: bf16 [B, Hq, d] view (last dim contiguous; any batch/head strides)."""
    if q.dim() != 3 or q.stride(2) != 1:
        raise ValueError("q must be a [B, Hq, d] view with a contiguous last dimension")
    kvc, = (kv.c(),)
    rc = lib().dustin_score_heads(ctypes.byref(shape), ctypes.byref(kvc), _ptr(q, torch.bfloat16), q.stride(0),
                                  q.stride(1), ctypes.c_uint64(head_mask), n_lists,
                                  _dense(scores_now, torch.float32), _ptr(ws), ws.numel(), _stream())
    _check("dustin_score_heads", rc)


def score_heads_static(shape: Shape, kv: KV, q: torch.Tensor, head_mask: int, n_lists: int,
                       scores_now: torch.Tensor) -> None:
    """score_heads for a caller that cannot hand over a workspace (its process may not allocate device memory: the
    serving engine around it owns all of HBM, or its operator interface passes inputs and outputs only).  Same
    arguments minus `ws`, same result bit for bit; the scratch is the library's built-in array of STATIC_SCRATCH_BYTES
    per GPU, so shapes that need more raise DustinError(ERR_STATIC_SCRATCH).  All calls on a GPU share that array:
    keep them on one stream.  The first call on each device does a one-time set-up (dustin.h)."""
    if q.dim() != 3 or q.stride(2) != 1:
        raise ValueError("q must be a [B, Hq, d] view with a contiguous last dimension")
    kvc = kv.c()
    rc = lib().dustin_score_heads_static(ctypes.byref(shape), ctypes.byref(kvc), _ptr(q, torch.bfloat16), q.stride(0),
                                         q.stride(1), ctypes.c_uint64(head_mask), n_lists,
                                         _dense(scores_now, torch.float32), _stream())
    _check("dustin_score_heads_static", rc)


def fuse_scores(scores_now: torch.Tensor, hist_inout: torch.Tensor, alpha: float,
                seq_lens: Optional[torch.Tensor] = None) -> None:
    B, G, N = scores_now.shape
    if hist_inout.shape != scores_now.shape:
        raise ValueError("hist_inout and scores_now must have the same [B, G, N] shape")
    rc = lib().dustin_fuse_scores(B, G, N, _ptr(seq_lens, torch.int32), _dense(scores_now, torch.float32),
                                  _dense(hist_inout, torch.float32), float(alpha), _stream())
    _check("dustin_fuse_scores", rc)


def topk_select(select: Select, s_draft: torch.Tensor, s_target: torch.Tensor, idx_out: torch.Tensor,
                cnt_out: torch.Tensor, seq_lens: Optional[torch.Tensor] = None) -> None:
    """s_target fp32 [B, G, N]; s_draft fp32 [B, N] (broadcast over lists) or [B, G, N]; idx_out int32
    [B, G, k_max]; cnt_out int32 [B, G]."""
    B, G, N = s_target.shape
    if G != select.n_lists or idx_out.shape[:2] != (B, G) or cnt_out.shape != (B, G):
        raise ValueError("list dimensions do not match select.n_lists")
    dls = 0 if s_draft.dim() == 2 else N
    sel = select.c()
    rc = lib().dustin_topk_select(B, N, _ptr(seq_lens, torch.int32), ctypes.byref(sel),
                                  _dense(s_draft, torch.float32), dls, _dense(s_target, torch.float32),
                                  _dense(idx_out, torch.int32), _dense(cnt_out, torch.int32), idx_out.shape[2],
                                  _stream())
    _check("dustin_topk_select", rc)


def sparse_verify_attn(shape: Shape, kv: KV, q: torch.Tensor, k_new: torch.Tensor, v_new: torch.Tensor,
                       idx: Optional[torch.Tensor], cnt: Optional[torch.Tensor], out: torch.Tensor,
                       ws: Optional[torch.Tensor], lse_out: Optional[torch.Tensor] = None) -> None:
    """idx None => full-cache verification attention (the dense baseline)."""
    n_lists, k_max = (idx.shape[1], idx.shape[2]) if idx is not None else (1, 0)
    kvc = kv.c()
    rc = lib().dustin_sparse_verify_attn(
        ctypes.byref(shape), ctypes.byref(kvc), _dense(q, torch.bfloat16), _dense(k_new, torch.bfloat16),
        _dense(v_new, torch.bfloat16), None if idx is None else _dense(idx, torch.int32),
        None if cnt is None else _dense(cnt, torch.int32), n_lists, k_max, _dense(out, torch.bfloat16),
        None if lse_out is None else _dense(lse_out, torch.float32), _ptr(ws), 0 if ws is None else ws.numel(),
        _stream())
    _check("dustin_sparse_verify_attn", rc)


def verify_layer_fused(shape: Shape, kv: KV, q: torch.Tensor, k_new: torch.Tensor, v_new: torch.Tensor,
                       head_mask: int, s_draft: torch.Tensor, hist_inout: torch.Tensor, alpha: float,
                       select: Select, out: torch.Tensor, idx_out: torch.Tensor, cnt_out: torch.Tensor,
                       ws: torch.Tensor, scores_now_out: Optional[torch.Tensor] = None,
                       lse_out: Optional[torch.Tensor] = None) -> None:
    N = shape.max_ctx
    dls = 0 if s_draft.dim() == 2 else N
    kvc, sel = kv.c(), select.c()
    rc = lib().dustin_verify_layer_fused(
        ctypes.byref(shape), ctypes.byref(kvc), _dense(q, torch.bfloat16), _dense(k_new, torch.bfloat16),
        _dense(v_new, torch.bfloat16), ctypes.c_uint64(head_mask), _dense(s_draft, torch.float32), dls,
        _dense(hist_inout, torch.float32), float(alpha), ctypes.byref(sel), idx_out.shape[2],
        None if scores_now_out is None else _dense(scores_now_out, torch.float32), _dense(out, torch.bfloat16),
        None if lse_out is None else _dense(lse_out, torch.float32), _dense(idx_out, torch.int32),
        _dense(cnt_out, torch.int32), _ptr(ws), ws.numel(), _stream())
    _check("dustin_verify_layer_fused", rc)


def arr(a: torch.Tensor, idx: torch.Tensor, cnt: torch.Tensor, arr_out: torch.Tensor,
        seq_lens: Optional[torch.Tensor] = None) -> None:
    """Eq. 1: a fp32 [B,G,N], idx int32 [B,G,k_max], cnt int32 [B,G] -> arr_out fp32 [B,G]."""
    B, G, N = a.shape
    rc = lib().dustin_arr(B, G, N, None if seq_lens is None else _dense(seq_lens, torch.int32),
                          _dense(a, torch.float32), _dense(idx, torch.int32), _dense(cnt, torch.int32), idx.shape[2],
                          _dense(arr_out, torch.float32), _stream())
    _check("dustin_arr", rc)


def append_kv(shape: Shape, kv: KV, seq_lens_inout: torch.Tensor, k_new: torch.Tensor, v_new: torch.Tensor,
              n_append: torch.Tensor, hist_inout: Optional[torch.Tensor] = None) -> None:
    """the first n_append[b] rows of the verify block go behind sequence b; lengths advance in place."""
    kvc = kv.c()
    rc = lib().dustin_append_kv(
        ctypes.byref(shape), ctypes.byref(kvc), _dense(seq_lens_inout, torch.int32), _dense(k_new, torch.bfloat16),
        _dense(v_new, torch.bfloat16), _dense(n_append, torch.int32),
        None if hist_inout is None else _dense(hist_inout, torch.float32),
        0 if hist_inout is None else hist_inout.shape[1], _stream())
    _check("dustin_append_kv", rc)


def draft_aggregate(shape: Shape, kv_layers: list, q_layers: list, head_mask: int, s_draft: torch.Tensor,
                    ws: torch.Tensor) -> None:
    """Eq. 5, first line: kv_layers / q_layers are per-draft-layer KV views and bf16 [B,T,Hq,d]
    query tensors; s_draft fp32 [B, max_ctx] is written."""
    L = len(kv_layers)
    kvs = (_Kv * L)(*[kv.c() for kv in kv_layers])
    qs = (ctypes.c_void_p * L)(*[_dense(q, torch.bfloat16) for q in q_layers])
    rc = lib().dustin_draft_aggregate(ctypes.byref(shape), kvs, qs, L, ctypes.c_uint64(head_mask),
                                      _dense(s_draft, torch.float32), _ptr(ws), ws.numel(), _stream())
    _check("dustin_draft_aggregate", rc)


def probe_gather(shape: Shape, kv: KV, idx: torch.Tensor, cnt: torch.Tensor, ws: torch.Tensor) -> None:
    """Measurement aid: reads the K / V rows a4 would gather for these lists and nothing else."""
    kvc = kv.c()
    rc = lib().dustin_probe_gather(ctypes.byref(shape), ctypes.byref(kvc), _dense(idx, torch.int32),
                                   _dense(cnt, torch.int32), idx.shape[1], idx.shape[2], _ptr(ws), ws.numel(), _stream())
    _check("dustin_probe_gather", rc)


def alloc_draft_workspace(shape: Shape, head_mask: int, device="cuda") -> torch.Tensor:
    """Zero-initialised workspace for draft_aggregate's one-pass-per-layer path."""
    n = int(lib().dustin_draft_workspace_bytes(ctypes.byref(shape), ctypes.c_uint64(head_mask)))
    if n == 0:
        raise ValueError("dustin_draft_workspace_bytes: invalid shape or empty head mask")
    return torch.zeros(n, dtype=torch.uint8, device=device)


QUEST_PAGE = 16     # DUSTIN_QUEST_PAGE


def quest_alloc_meta(shape: Shape, device="cuda") -> torch.Tensor:
    """bf16 [B, ceil(max_ctx/16), Hkv, 2, d] page metadata buffer (dustin_quest_meta_bytes)."""
    n_pages = (shape.max_ctx + QUEST_PAGE - 1) // QUEST_PAGE
    meta = torch.empty((shape.batch, n_pages, shape.n_kv_heads, 2, shape.head_dim), dtype=torch.bfloat16, device=device)
    assert meta.numel() * 2 == int(lib().dustin_quest_meta_bytes(ctypes.byref(shape)))
    return meta


def quest_build_pages(shape: Shape, kv: KV, page_meta: torch.Tensor, first_token: Optional[torch.Tensor] = None) -> None:
    """per-page, per-channel key min / max; first_token (int32 [B]) limits the rebuild to later pages."""
    kvc = kv.c()
    rc = lib().dustin_quest_build_pages(ctypes.byref(shape), ctypes.byref(kvc),
                                        None if first_token is None else _dense(first_token, torch.int32),
                                        _dense(page_meta, torch.bfloat16), _stream())
    _check("dustin_quest_build_pages", rc)


def quest_score_pages(shape: Shape, page_meta: torch.Tensor, q: torch.Tensor, head_mask: int, n_lists: int,
                      page_scores: torch.Tensor, ws: torch.Tensor, seq_lens: Optional[torch.Tensor] = None,
                      ub_out: Optional[torch.Tensor] = None) -> None:
    """PAPER.md:51 / :297: page scores from the metadata alone.  q: bf16 [B, Hq, d] view; page_scores fp32
    [B, n_lists, n_pages]; ub_out fp32 [B, |subset|, n_pages] or None."""
    if q.dim() != 3 or q.stride(2) != 1:
        raise ValueError("q must be a [B, Hq, d] view with a contiguous last dimension")
    rc = lib().dustin_quest_score_pages(
        ctypes.byref(shape), None if seq_lens is None else _dense(seq_lens, torch.int32),
        _dense(page_meta, torch.bfloat16), _ptr(q, torch.bfloat16), q.stride(0), q.stride(1),
        ctypes.c_uint64(head_mask), n_lists, _dense(page_scores, torch.float32),
        None if ub_out is None else _dense(ub_out, torch.float32), _ptr(ws), ws.numel(), _stream())
    _check("dustin_quest_score_pages", rc)


def prefer_dense(shape: Shape, head_mask: int, k: int):
    """dustin_prefer_dense: (dense is predicted at least as fast, predicted fused us, predicted dense us) -- a hint from
    a byte model fitted on a B200 (dustin.h); host arithmetic only."""
    f, d = ctypes.c_double(), ctypes.c_double()
    rc = lib().dustin_prefer_dense(ctypes.byref(shape), ctypes.c_uint64(head_mask), int(k), ctypes.byref(f), ctypes.byref(d))
    if rc < 0:
        raise DustinError("dustin_prefer_dense", rc)
    return bool(rc), f.value, d.value
