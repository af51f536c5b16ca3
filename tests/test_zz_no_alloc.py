"""dustin_score_heads_static: head-subset scoring for callers that cannot allocate device memory.

Every other entry point of the library wants a workspace from its caller.  Some callers cannot produce one: the serving
engine they run under took all of HBM for itself at start-up, or they sit behind an operator interface that passes
inputs and outputs and nothing else, or they are inside a decode step where a cudaMalloc (which may synchronise the
device) is not acceptable.  For them the library carries a fixed 16 MiB scratch array of its own and this one entry
point that uses it (include/dustin.h, "a1 without a workspace argument").

What is checked here:
  * the new entry point returns what the existing one (dustin_score_heads with a caller workspace) returns, on two
    calls in a row with different shapes -- the second call finds the first call's leftovers in the shared array and
    must not be affected by them.  Both paths run the same kernels on the same plan, so the comparison is bitwise,
    which is well inside the 1e-5 relative tolerance the scoring parity tests use (tests/harness.py);
  * a repeated call leaves the amount of free device memory unchanged (nothing is allocated behind the caller's back);
  * a shape that needs more than the array holds is refused with its own status code, before the device is involved
    (this part runs without a GPU).

This file is named so that pytest collects it last: under `pytest -x` a failure here cannot hide another test.
It passes on its own in a fresh process (the first call below is then the first use of the library on the device and
does the one-time set-up) and after the rest of the suite.
"""
import ctypes
import os
import re

import pytest
import torch

from paper_2606_24957_b200 import api, build, synth
from tests import harness as H

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_limit_in_header_matches_binding():
    text = open(os.path.join(ROOT, "include", "dustin.h")).read()
    m = re.search(r"#define\s+DUSTIN_STATIC_SCRATCH_BYTES\s+\((\d+)\s*\*\s*(\d+)\s*\*\s*(\d+)\)", text)
    assert m, "DUSTIN_STATIC_SCRATCH_BYTES not found in dustin.h"
    assert int(m.group(1)) * int(m.group(2)) * int(m.group(3)) == api.STATIC_SCRATCH_BYTES == 16 << 20


def test_oversized_shape_is_refused_before_the_device_is_touched():
    """B = 16, 8 subset heads, 32k context needs 16.8 MB of logits alone: over the limit.  The refusal comes from host
    arithmetic only, so it also works (and is tested) on a machine without a GPU; the pointers are never looked at."""
    build.build()
    L = api.lib()
    sh = api.Shape(16, 64, 8, 128, 5, 32768, 0.0)
    fake = ctypes.c_void_p(0x1000)
    kv = api._Kv(fake, fake, 32768 * 8 * 128, 8 * 128, 128, None, 0, 0, None)
    mask = sum(1 << (8 * g) for g in range(8))
    rc = L.dustin_score_heads_static(ctypes.byref(sh), ctypes.byref(kv), fake, 64 * 128, 128, ctypes.c_uint64(mask), 8,
                                     fake, None)
    assert rc == api.ERR_STATIC_SCRATCH
    assert b"DUSTIN_STATIC_SCRATCH_BYTES" in L.dustin_status_string(rc)
    # the documented sufficient test: dustin_workspace_bytes(shape, mask, 1) over the limit
    assert api.workspace_bytes(sh, mask, 1) > api.STATIC_SCRATCH_BYTES
    # a null output is still the plain argument error
    rc = L.dustin_score_heads_static(ctypes.byref(sh), ctypes.byref(kv), fake, 64 * 128, 128, ctypes.c_uint64(mask), 8,
                                     None, None)
    assert rc == api.ERR_INVALID_ARG


def _both_paths(cfg):
    """(scores through the caller-workspace path, scores through the static-scratch path) for one seeded layer."""
    dev = synth.make_layer(cfg, 0, "cuda")
    sh = H.shape_of(cfg)
    kv = H.gpu_kv(dev)
    B, G, N = cfg.batch, cfg.n_lists, cfg.ctx
    ws = api.alloc_workspace(sh, cfg.head_mask, 1)
    assert ws.numel() <= api.STATIC_SCRATCH_BYTES, "test case must fit the static scratch"
    want = torch.full((B, G, N), float("nan"), device="cuda")
    got = torch.full((B, G, N), float("nan"), device="cuda")
    api.score_heads(sh, kv, dev.q[:, 0], cfg.head_mask, G, want, ws)
    api.score_heads_static(sh, kv, dev.q[:, 0], cfg.head_mask, G, got)
    torch.cuda.synchronize()
    return want, got, (sh, kv, dev)


def _assert_same(want, got, what):
    assert torch.isfinite(got).all(), f"{what}: non-finite scores"
    # tolerance of the scoring parity tests (harness.SCORE_RTOL) ...
    rel = ((got.double() - want.double()).abs() / want.double().clamp_min(1e-300))[want > H.SCORE_FLOOR]
    assert rel.numel() > 0 and rel.max().item() <= H.SCORE_RTOL, f"{what}: differs from dustin_score_heads"
    # ... and, since both paths launch the same kernels with the same plan, the same bits
    assert torch.equal(got, want), f"{what}: not bit-identical to dustin_score_heads"


@pytest.mark.gpu
def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    qwen, llama = synth.config_qwen72b(), synth.config_llama8b()
    # call 1: 8 subset heads, one per KV group, per-KV-head lists, context with a ragged tail (not a multiple of 16)
    first = synth.shrink(qwen, batch=2, ctx=4100, budget=600, n_sink=64, n_recent=256)
    # call 2: another shape on the same array, which still holds call 1's logits -- four KV groups scored, paged cache,
    # ragged sequence lengths;  call 3: packed subset (all four heads in one KV group), one list per sequence
    second = synth.shrink(synth.config_paged(), batch=3, ctx=4000, ragged_min=900, n_sink=4, n_recent=16)
    third = synth.shrink(llama, batch=2, ctx=3000, budget=512, n_sink=8, n_recent=64, heads=synth.packed_heads(4),
                         n_lists=1)
    for name, cfg in (("first call", first), ("second call", second), ("third call", third)):
        want, got, _ = _both_paths(cfg)
        _assert_same(want, got, name)


@pytest.mark.gpu
def test_static_scratch_call_allocates_no_device_memory():
    cfg = synth.shrink(synth.config_qwen72b(), batch=2, ctx=4100, budget=600, n_sink=64, n_recent=256)
    want, got, (sh, kv, dev) = _both_paths(cfg)      # set-up done, kernels loaded, all tensors exist
    _assert_same(want, got, "warm-up call")
    got.fill_(float("nan"))
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        api.score_heads_static(sh, kv, dev.q[:, 0], cfg.head_mask, cfg.n_lists, got)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, "the static-scratch entry point changed the amount of free device memory"
    _assert_same(want, got, "repeated call")
