"""GPU parity of stage a4/a5 alone (dustin_sparse_verify_attn) on inputs built to reach the corners of the two
attention kernels: the lazy reference exponent of the tcgen05 kernel (scores that jump far above everything seen
so far, several times within one piece), empty index lists, lists shorter than a tile, units that are cut across
many CTAs and CTAs that hold many units, and repeated indices."""
import pytest
import torch

from oracle import ref
from paper_2606_24957_b200 import api
from tests import harness as H

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True, params=["tcgen05", "mma_sync"])
def attn_impl(request):
    api.tune_attn_impl(1 if request.param == "mma_sync" else 0)
    yield request.param
    api.tune_attn_impl(0)


def _inputs(B, N, Hq, Hkv, d, T, seed):
    g = torch.Generator().manual_seed(seed)
    bf = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16)
    return dict(q=bf(B, T, Hq, d), k=bf(B, N, Hkv, d), v=bf(B, N, Hkv, d), k_new=bf(B, T, Hkv, d),
                v_new=bf(B, T, Hkv, d))


def _run_both(x, idx, cnt, N, sm_scale=0.0):
    B, T, Hq, d = x["q"].shape
    Hkv = x["k"].shape[2]
    sh = api.Shape(B, Hq, Hkv, d, T, N, sm_scale)
    k_max = idx.shape[2] if idx is not None else 0
    ws = api.alloc_workspace(sh, 1, k_max)
    dev = {n: t.cuda() for n, t in x.items()}
    out = torch.full_like(dev["q"], float("nan"))
    lse = torch.full((B, Hq, T), float("nan"), device="cuda")
    api.sparse_verify_attn(sh, api.KV.contiguous_nhd(dev["k"], dev["v"], None), dev["q"], dev["k_new"], dev["v_new"],
                           None if idx is None else idx.cuda(), None if cnt is None else cnt.cuda(), out, ws, lse)
    torch.cuda.synchronize()
    o_ref, lse_ref = ref.sparse_verify_attn(ref.KV.contiguous_nhd(x["k"], x["v"], None), x["q"], x["k_new"],
                                            x["v_new"], idx, cnt, N, sm_scale)
    return out, lse, o_ref, lse_ref


def _lists(B, G, N, counts, k_max, seed):
    g = torch.Generator().manual_seed(seed)
    idx = torch.full((B, G, k_max), -1, dtype=torch.int32)
    cnt = torch.zeros((B, G), dtype=torch.int32)
    for b in range(B):
        for l in range(G):
            n = counts[(b * G + l) % len(counts)]
            idx[b, l, :n] = torch.sort(torch.randperm(N, generator=g)[:n]).values.to(torch.int32)
            cnt[b, l] = n
    return idx, cnt


def test_scores_that_jump_far_above_the_reference_exponent():
    """Keys aligned with one head's query, of growing strength, planted in successive tiles with sm_scale = 1:
    each of them exceeds everything seen so far by far more than the slack of the lazy reference, so the
    accumulated output is rescaled several times inside one piece (factors from ~1e-1 down to 0)."""
    B, N, Hq, Hkv, d, T = 1, 1500, 8, 2, 128, 3
    x = _inputs(B, N, Hq, Hkv, d, T, 11)
    qv = x["q"][0, 0, 1].float()                          # head 1 (KV head 0), verify position 0
    for j, (pos, c) in enumerate([(200, 0.25), (420, 0.4), (700, 0.7), (1000, 1.0), (1300, 1.6)]):
        x["k"][0, pos, 0] = (c * qv).to(torch.bfloat16)
    idx = torch.arange(N, dtype=torch.int32).view(1, 1, N).contiguous()
    cnt = torch.tensor([[N]], dtype=torch.int32)
    for sc in (1.0, 0.3):
        out, lse, o_ref, lse_ref = _run_both(x, idx, cnt, N, sm_scale=sc)
        H.check_attn(out, o_ref)
        assert torch.allclose(lse.cpu().double(), lse_ref, atol=1e-2, rtol=1e-5)
        out, lse, o_ref, lse_ref = _run_both(x, None, None, N, sm_scale=sc)
        H.check_attn(out, o_ref, "dense")


def test_empty_and_short_lists_only_new_rows_visible():
    B, N, Hq, Hkv, d, T = 3, 700, 16, 4, 128, 5
    x = _inputs(B, N, Hq, Hkv, d, T, 12)
    idx, cnt = _lists(B, Hkv, N, [0, 1, 3, 127, 128, 129, 0, 300], 300, 5)
    out, lse, o_ref, lse_ref = _run_both(x, idx, cnt, N)
    H.check_attn(out, o_ref)
    assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)
    # a list with no cache rows: verify position 0 sees only its own new row, so its output is v_new[b, 0, g]
    got = out[0, 0, 0].float().cpu()
    assert torch.allclose(got, x["v_new"][0, 0, 0].float(), atol=1e-2)


def test_many_small_units_per_cta_and_units_cut_across_many_ctas():
    # 24 * 8 = 192 units of 40..90 tokens: every CTA holds several whole units plus cut ones
    B, N, Hq, Hkv, d, T = 24, 400, 32, 8, 128, 5
    x = _inputs(B, N, Hq, Hkv, d, T, 13)
    idx, cnt = _lists(B, Hkv, N, [35, 85, 60, 41, 77], 85, 6)
    out, lse, o_ref, lse_ref = _run_both(x, idx, cnt, N)
    H.check_attn(out, o_ref)
    assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)
    # one unit of 40k tokens: cut across every CTA of the grid (G = 1 list shared by the KV heads)
    B, N, Hq, Hkv, d, T = 1, 40000, 8, 1, 128, 9
    x = _inputs(B, N, Hq, Hkv, d, T, 14)
    out, lse, o_ref, lse_ref = _run_both(x, None, None, N)
    H.check_attn(out, o_ref)
    assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)


def test_global_list_and_repeated_indices():
    B, N, Hq, Hkv, d, T = 2, 3000, 32, 8, 128, 5
    x = _inputs(B, N, Hq, Hkv, d, T, 15)
    idx, cnt = _lists(B, 1, N, [777, 1024], 1024, 7)
    idx[0, 0, 5] = idx[0, 0, 4]                            # a repeated row simply counts twice (any order allowed)
    out, lse, o_ref, lse_ref = _run_both(x, idx, cnt, N)
    H.check_attn(out, o_ref)
    assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)


@pytest.mark.parametrize("T,r", [(1, 1), (3, 2), (16, 4), (12, 8), (2, 16), (13, 4), (9, 8), (10, 8), (11, 8)])
def test_query_row_counts(T, r):
    """T * r from 1 to 96 query rows per KV head: every NQ instantiation of the tcgen05 kernel (16, 32, 48 rows on one
    softmax warpgroup; 52 -> 64 = 2 x 32, 72 and 80 -> 80 = 2 x 40 with the 8-column TMEM loads, 88 and 96 -> 2 x 48)."""
    B, N, Hkv, d = 2, 900, 2, 128
    x = _inputs(B, N, Hkv * r, Hkv, d, T, 16 + T)
    idx, cnt = _lists(B, Hkv, N, [333, 500], 500, 8)
    out, lse, o_ref, lse_ref = _run_both(x, idx, cnt, N)
    H.check_attn(out, o_ref)
    assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)


@pytest.mark.parametrize("B,Hkv,k", [(2, 2, 300), (16, 8, 257), (1, 1, 2048)])
def test_cnt_null_means_full_lists(B, Hkv, k):
    """cnt == NULL (dustin.h: every list holds exactly k_max entries; the kernel plans without reading a length):
    bitwise the result of the same call with cnt = k_max everywhere, in whole-unit and in cut-unit decompositions, and
    against the oracle; refused when the lists could be shorter (ragged sequences, k_max > max_ctx)."""
    N, Hq, d, T = 4096, 4 * Hkv, 128, 5
    x = _inputs(B, N, Hq, Hkv, d, T, 77)
    idx, cnt = _lists(B, Hkv, N, [k], k, 78)
    out_c, lse_c, o_ref, lse_ref = _run_both(x, idx, cnt, N)
    sh = api.Shape(B, Hq, Hkv, d, T, N, 0.0)
    dev = {n: t.cuda() for n, t in x.items()}
    ws = api.alloc_workspace(sh, 1, k)
    out_n = torch.full_like(dev["q"], float("nan"))
    lse_n = torch.full((B, Hq, T), float("nan"), device="cuda")
    api.sparse_verify_attn(sh, api.KV.contiguous_nhd(dev["k"], dev["v"], None), dev["q"], dev["k_new"], dev["v_new"],
                           idx.cuda(), None, out_n, ws, lse_n)
    torch.cuda.synchronize()
    assert torch.equal(out_c, out_n) and torch.equal(lse_c, lse_n)
    H.check_attn(out_n, o_ref)
    assert torch.allclose(lse_n.cpu().double(), lse_ref, atol=1e-2, rtol=1e-5)
    lens = torch.full((B,), N, dtype=torch.int32, device="cuda")
    with pytest.raises(api.DustinError):
        api.sparse_verify_attn(sh, api.KV.contiguous_nhd(dev["k"], dev["v"], lens), dev["q"], dev["k_new"],
                               dev["v_new"], idx.cuda(), None, torch.empty_like(dev["q"]), ws)
    wide = torch.zeros((B, Hkv, N + 8), dtype=torch.int32, device="cuda")
    with pytest.raises(api.DustinError):
        api.sparse_verify_attn(sh, api.KV.contiguous_nhd(dev["k"], dev["v"], None), dev["q"], dev["k_new"],
                               dev["v_new"], wide, None, torch.empty_like(dev["q"]), ws)


def test_cuts_inside_the_new_row_tile_move_to_the_unit_start():
    """Short lists on a grid of as many CTAs as tiles: the equal cuts of the concatenated token space fall inside the
    new-row tiles (128 virtual positions at the head of every unit) and must move down to the unit's start -- no piece
    may begin in the padding of that tile.  Several list lengths so that one, two and three cuts
    land in one tile, with and without cache rows behind it."""
    B, N, Hkv, d, T, r = 3, 700, 2, 128, 5, 4
    x = _inputs(B, N, Hkv * r, Hkv, d, T, 91)
    for counts in ([40], [0, 40, 300], [7, 129, 0, 64, 511, 1], [200, 0, 0, 3]):
        idx, cnt = _lists(B, Hkv, N, counts, 512, 92)
        out, lse, o_ref, lse_ref = _run_both(x, idx, cnt, N)
        H.check_attn(out, o_ref)
        assert torch.allclose(lse.cpu().double(), lse_ref, atol=2e-3, rtol=0)
