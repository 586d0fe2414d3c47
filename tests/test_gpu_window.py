"""GPU parity of the sliding-window + attention-sink variant (comem_decode_attn_window_async, DESIGN.md
reading R17) against oracle.decode_attn_window on the same bits, plus the properties that fix bits."""
import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import MAX_ABS, MEAN_ABS, REL_L2, gpu_run

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t):
    return t.contiguous().view(torch.int16)


def run_window(b, window, sinks, ws=None):
    out = torch.full_like(b.q, float("nan"))
    lse = torch.full((b.batch, b.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
    ws = ws if ws is not None else comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    comem.comem_decode_attn_window_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                         out, ws, window, sinks, lse_out=lse)
    torch.cuda.synchronize()
    return out, lse


def check(oracle, b, window, sinks, what):
    out, lse = run_window(b, window, sinks)
    ref, ref_lse = oracle.decode_attn_window(b.q.cpu(), b.k_pages.cpu(), b.v_pages.cpu(), b.block_table.cpu(),
                                             b.seq_lens.cpu(), b.softmax_scale, window, sinks)
    g = out.double().cpu().numpy()
    d = np.abs(g - ref)
    assert np.isfinite(g).all(), what
    assert d.max() <= MAX_ABS and d.mean() <= MEAN_ABS, (what, d.max(), d.mean())
    assert np.linalg.norm(g - ref) / max(np.linalg.norm(ref), 1e-300) <= REL_L2, what
    assert d.max() <= 4 * 2.0 ** -9 * np.abs(ref).max() + 1e-6, what
    gl = lse.double().cpu().numpy()
    live = np.isfinite(ref_lse)
    assert np.array_equal(np.isneginf(gl), np.isneginf(ref_lse)), what
    if live.any():
        assert np.max(np.abs(gl[live] - ref_lse[live]) / np.maximum(1.0, np.abs(ref_lse[live]))) <= 2e-4, what
    return out, lse


@pytest.mark.parametrize("G,D,ps", [(1, 64, 16), (4, 128, 32), (8, 128, 16), (2, 64, 32)])
def test_window_small_grid(oracle, G, D, ps):
    lens = [1, 15, 16, 17, 31, 33, 127, 128, 129, 512, 1000, 0, 2049]
    b = W.make_batch(lens, 2 * G, 2, D, ps, seed=400 + G + D + ps, device=DEV, poison_unused=True)
    for window, sinks in ((1, 0), (16, 0), (17, 1), (100, 4), (128, 16), (129, 40), (5000, 3), (64, 1000)):
        check(oracle, b, window, sinks, f"G{G} D{D} ps{ps} w{window} s{sinks}")


def test_window_long_ragged_and_grids(oracle):
    lens = [20000, 37, 0, 50001, 8191, 16, 300]
    b = W.make_batch(lens, 64, 8, 128, 16, seed=421, device=DEV, poison_unused=True)
    for window, sinks in ((4096, 4), (1000, 64), (33, 0)):
        check(oracle, b, window, sinks, f"ragged w{window} s{sinks}")
    try:
        for g in (1, 5, 37, 296):
            comem.comem_set_grid_ctas(g)
            check(oracle, b, 4096, 4, f"grid {g}")
    finally:
        comem.comem_set_grid_ctas(0)


def test_window_closed_forms_and_identities():
    b = W.make_batch([777, 16, 4000], 16, 2, 128, 16, seed=431, device=DEV)
    # window 1, no sinks: out = V[L-1] bit for bit
    out, _ = run_window(b, 1, 0)
    for i, L in enumerate((777, 16, 4000)):
        pid = int(b.block_table[i, (L - 1) // 16])
        want = b.v_pages[pid, (L - 1) % 16].repeat_interleave(8, dim=0)
        assert torch.equal(bits(out[i]), bits(want))
    # no window == the full-attention entry point, bit for bit
    full, lse_full = gpu_run(b)
    torch.cuda.synchronize()
    for window, sinks in ((0, 0), (4000, 0), (10 ** 6, 7)):
        o, l = run_window(b, window, sinks)
        assert torch.equal(bits(o), bits(full)) and torch.equal(l, lse_full)


def test_window_masked_tokens_and_placement_do_not_matter():
    lens = [5000, 333, 64]
    window, sinks = 700, 20
    b = W.make_batch(lens, 32, 8, 128, 32, seed=441, device=DEV)
    o1, l1 = run_window(b, window, sinks)
    o2, l2 = run_window(W.permute_pages(b, seed=3), window, sinks)
    assert torch.equal(bits(o1), bits(o2)) and torch.equal(l1, l2)
    for poison in (float("nan"), float("inf"), -1e38):
        for i, L in enumerate(lens):
            t = torch.arange(L)
            dead = (t >= sinks) & (t < L - window)
            pid = b.block_table[i, (t[dead] // 32).to(DEV)].long()
            b.k_pages[pid, (t[dead] % 32).to(DEV)] = poison
            b.v_pages[pid, (t[dead] % 32).to(DEV)] = poison
        o3, l3 = run_window(b, window, sinks)
        assert torch.equal(bits(o1), bits(o3)) and torch.equal(l1, l3), poison
