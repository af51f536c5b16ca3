"""CPU-side checks of the boundary: libdustin.so builds/loads, exports every function include/dustin.h declares,
and rejects bad host-visible arguments with the documented status codes before touching the device
(no compute call is made here: every call below must fail validation)."""
import ctypes
import os
import re

import pytest

from paper_2606_24957_b200 import api, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return api.lib()


def declared_functions(header="dustin.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dustin_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert set(names) == set(api.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_debug_header_is_separate_and_exported(lib):
    """Measurement / tuning aids live in dustin_debug.h, none of them in the product header."""
    names = declared_functions("dustin_debug.h")
    assert set(names) == set(api.DEBUG_EXPORTS)
    assert not set(names) & set(declared_functions())
    for n in names:
        assert hasattr(lib, n), n
    assert api.tune_get(api.KNOB_PDL) == 1
    api.tune_set(api.KNOB_PDL, 0)
    assert api.tune_get(api.KNOB_PDL) == 0
    api.tune_set(api.KNOB_PDL, 1)
    assert api.tune_get(999) == 0


def test_library_reads_no_environment_variable(lib):
    """No object of csrc/ references getenv (the statically linked CUDA runtime does, for its own settings)."""
    import glob
    import subprocess
    objs = sorted(glob.glob(os.path.join(os.path.dirname(api.LIB_PATH), "build", "*.o")))
    assert objs
    out = subprocess.run(["nm", "--undefined-only", *objs], capture_output=True, text=True).stdout
    assert "getenv" not in out


def test_version_and_status_strings(lib):
    assert api.version() == 100
    for code in (0, -1, -2, -3, -4, -99):
        assert isinstance(lib.dustin_status_string(code), bytes)


def shape(**kw):
    d = dict(batch=2, n_q_heads=8, n_kv_heads=2, head_dim=128, n_new=5, max_ctx=4096, sm_scale=0.0)
    d.update(kw)
    return api.Shape(**d)


def test_workspace_bytes(lib):
    sh = shape()
    small = api.workspace_bytes(sh, 0b1, 512)
    big = api.workspace_bytes(sh, 0, 0)
    assert 0 < small < big
    assert lib.dustin_workspace_bytes(ctypes.byref(shape(head_dim=96)), 0, 0) == 0
    assert lib.dustin_workspace_bytes(ctypes.byref(shape(n_q_heads=7)), 0, 0) == 0
    assert lib.dustin_workspace_bytes(None, 0, 0) == 0


FAKE = ctypes.c_void_p(0x1000)      # never dereferenced: validation fails first


def kv(**kw):
    d = dict(k=FAKE, v=FAKE, stride_seq=4096 * 2 * 128, stride_token=2 * 128, stride_head=128, page_table=None,
             page_size=0, max_pages=0, seq_lens=None)
    d.update(kw)
    return api._Kv(**d)


def sel(**kw):
    d = dict(budget=512, budgets=None, n_sink=4, n_recent=16, m_num=1, m_den=2, n_lists=1)
    d.update(kw)
    return api._Select(**d)


@pytest.mark.parametrize("sh,mask,n_lists,want", [
    (shape(n_q_heads=7), 1, 1, api.ERR_INVALID_ARG),          # Hq % Hkv != 0
    (shape(head_dim=96), 1, 1, api.ERR_UNSUPPORTED),
    (shape(n_new=17), 1, 1, api.ERR_UNSUPPORTED),
    (shape(max_ctx=(1 << 20) + 1), 1, 1, api.ERR_UNSUPPORTED),
    (shape(), 0, 1, api.ERR_INVALID_ARG),                     # empty head subset
    (shape(), 1 << 8, 1, api.ERR_INVALID_ARG),                # head outside Hq
    (shape(), 1, 3, api.ERR_INVALID_ARG),                     # n_lists not in {1, Hkv}
    (shape(n_q_heads=64, n_kv_heads=2), (1 << 9) - 1, 1, api.ERR_UNSUPPORTED),   # 9 subset heads in one group
])
def test_score_heads_rejects(lib, sh, mask, n_lists, want):
    k = kv()
    rc = lib.dustin_score_heads(ctypes.byref(sh), ctypes.byref(k), FAKE, 8 * 128, 128, mask, n_lists, FAKE, FAKE,
                                1 << 40, None)
    assert rc == want


def test_score_heads_rejects_pointers_strides_and_workspace(lib):
    sh = shape()
    ok = kv()
    call = lambda k, q=FAKE, out=FAKE, ws=FAKE, wsb=1 << 40, qs=8 * 128: lib.dustin_score_heads(
        ctypes.byref(sh), ctypes.byref(k), q, qs, 128, 1, 1, out, ws, wsb, None)
    assert call(kv(k=None)) == api.ERR_INVALID_ARG
    assert call(kv(stride_token=0)) == api.ERR_INVALID_ARG
    assert call(kv(stride_token=2 * 128 + 4)) == api.ERR_INVALID_ARG          # rows not 16-byte aligned
    assert call(kv(page_table=FAKE, page_size=16, max_pages=10)) == api.ERR_INVALID_ARG   # 160 < max_ctx
    assert call(ok, q=None) == api.ERR_INVALID_ARG
    assert call(ok, out=None) == api.ERR_INVALID_ARG
    assert call(ok, qs=8 * 128 + 1) == api.ERR_INVALID_ARG
    assert call(ok, ws=None) == api.ERR_WORKSPACE
    assert call(ok, wsb=1024) == api.ERR_WORKSPACE


def test_fuse_and_select_reject(lib):
    assert lib.dustin_fuse_scores(0, 1, 16, None, FAKE, FAKE, 1.0, None) == api.ERR_INVALID_ARG
    assert lib.dustin_fuse_scores(1, 1, 16, None, None, FAKE, 1.0, None) == api.ERR_INVALID_ARG
    assert lib.dustin_fuse_scores(1, 1, 16, None, FAKE, FAKE, float("nan"), None) == api.ERR_INVALID_ARG
    call = lambda s, k_max=512, dls=0, sd=FAKE: lib.dustin_topk_select(
        2, 4096, None, ctypes.byref(s), sd, dls, FAKE, FAKE, FAKE, k_max, None)
    assert call(sel(n_sink=500, n_recent=100)) == api.ERR_INVALID_ARG        # S + W > k (reading A12)
    assert call(sel(budget=1024)) == api.ERR_INVALID_ARG                     # k > k_max
    assert call(sel(m_num=3, m_den=2)) == api.ERR_INVALID_ARG
    assert call(sel(m_den=0)) == api.ERR_INVALID_ARG
    assert call(sel(), dls=17) == api.ERR_INVALID_ARG
    assert call(sel(), sd=None) == api.ERR_INVALID_ARG
    assert lib.dustin_topk_select(2, 4096, None, None, FAKE, 0, FAKE, FAKE, FAKE, 512, None) == api.ERR_INVALID_ARG


def test_attn_and_fused_reject(lib):
    sh = shape()
    k = kv()
    attn = lambda idx=FAKE, cnt=FAKE, n_lists=1, k_max=512, out=FAKE, ws=FAKE, wsb=1 << 40, kvv=k, s=sh: \
        lib.dustin_sparse_verify_attn(ctypes.byref(s), ctypes.byref(kvv), FAKE, FAKE, FAKE, idx, cnt, n_lists, k_max,
                                      out, None, ws, wsb, None)
    # cnt == NULL states "every list holds k_max entries": refused where that cannot hold
    assert attn(cnt=None, kvv=kv(seq_lens=FAKE)) == api.ERR_INVALID_ARG
    assert attn(cnt=None, k_max=4097) == api.ERR_INVALID_ARG
    assert attn(n_lists=3) == api.ERR_INVALID_ARG
    assert attn(out=None) == api.ERR_INVALID_ARG
    assert attn(kvv=kv(v=None)) == api.ERR_INVALID_ARG
    assert attn(s=shape(n_q_heads=64, n_kv_heads=2, n_new=5)) == api.ERR_UNSUPPORTED   # T*r = 160 > 96 rows
    s = sel()
    fused = lambda mask=1, hist=FAKE, ws=FAKE, wsb=1 << 40, se=s: lib.dustin_verify_layer_fused(
        ctypes.byref(sh), ctypes.byref(k), FAKE, FAKE, FAKE, mask, FAKE, 0, hist, 1.0, ctypes.byref(se), 512, None,
        FAKE, None, FAKE, FAKE, ws, wsb, None)
    assert fused(mask=0) == api.ERR_INVALID_ARG
    assert fused(hist=None) == api.ERR_INVALID_ARG
    assert fused(wsb=4096) == api.ERR_WORKSPACE
    assert fused(se=sel(n_lists=3)) == api.ERR_INVALID_ARG


def test_binding_refuses_cpu_tensors():
    import torch
    with pytest.raises(TypeError):
        api.fuse_scores(torch.zeros(1, 1, 8), torch.zeros(1, 1, 8), 1.0)


def test_prefer_dense_hint_brackets_the_measured_crossover(lib):
    """dustin_prefer_dense is host arithmetic fitted to the B200 sweep (profiles/r03_sweep.json): at k = 2048, B = 16 the
    fused layer loses to dense at 4k and 8k and wins from 16k on (measured crossing: 10.5 k tokens); the predicted times
    stay within 10 % of the measured ones at the sweep points; a budget that keeps everything always prefers dense."""
    mask = sum(1 << (8 * g) for g in range(8))
    measured = {4096: (95.06, 56.79), 8192: (111.82, 96.56), 16384: (146.01, 182.78), 32768: (222.26, 337.4)}
    prev = None
    for ctx, (fused_us, dense_us) in measured.items():
        dense, f, d = api.prefer_dense(api.Shape(16, 64, 8, 128, 5, ctx, 0.0), mask, 2048)
        assert dense == (ctx <= 8192)
        assert abs(f - fused_us) <= 0.10 * fused_us and abs(d - dense_us) <= 0.10 * dense_us
        assert prev is None or (f > prev[0] and d > prev[1])
        prev = (f, d)
    assert api.prefer_dense(api.Shape(16, 64, 8, 128, 5, 32768, 0.0), mask, 32768)[0]
    assert not api.prefer_dense(api.Shape(16, 64, 8, 128, 5, 32768, 0.0), mask, 512)[0]
    assert lib.dustin_prefer_dense(None, mask, 2048, None, None) == api.ERR_INVALID_ARG
    assert lib.dustin_prefer_dense(ctypes.byref(shape()), 0, 2048, None, None) == api.ERR_INVALID_ARG
