"""comem_decode_attn_static_async — the decode step with its scratch in a fixed device array inside the library (for
callers that may not allocate): output against the existing path (comem_decode_attn_async with a caller workspace) on
two calls in a row, and the rejection of shapes beyond the array.  Collected last on purpose (file name)."""
import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import MAX_ABS, MEAN_ABS, REL_L2

pytestmark = pytest.mark.gpu
DEV = "cuda"


def existing(b, flags=0):
    out = torch.full_like(b.q, float("nan"))
    lse = torch.full((b.batch, b.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out, ws,
                                  lse_out=lse, flags=flags)
    torch.cuda.synchronize()
    return out, lse


def static(b, flags=0):
    out = torch.full_like(b.q, float("nan"))
    lse = torch.full((b.batch, b.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
    comem.comem_decode_attn_static_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out,
                                         lse_out=lse, flags=flags)
    return out, lse


def close(a, b, what):
    a, b = a.double().cpu().numpy(), b.double().cpu().numpy()
    d = np.abs(a - b)
    assert np.isfinite(a).all(), what
    assert d.max() <= MAX_ABS and d.mean() <= MEAN_ABS, (what, d.max(), d.mean())
    assert np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300) <= REL_L2, what


def test_static_scratch_two_calls_in_a_row_match_the_workspace_path():
    """Two different problems back to back on one stream, no synchronisation between them (the second call finds the
    first one's partials and counters in the shared array); then the first problem again."""
    b1 = W.make_batch([32768], 64, 8, 128, 16, seed=9101, device=DEV, poison_unused=True)          # every segment cut
    b2 = W.make_batch([5000, 0, 17, 20000, 333, 16, 1], 32, 8, 128, 32, seed=9102, device=DEV, poison_unused=True)
    want1, want1_lse = existing(b1)
    want2, want2_lse = existing(b2)
    got1, got1_lse = static(b1)
    got2, got2_lse = static(b2)
    got3, got3_lse = static(b1)
    torch.cuda.synchronize()
    for got, got_lse, want, want_lse, what in ((got1, got1_lse, want1, want1_lse, "first call"),
                                               (got2, got2_lse, want2, want2_lse, "second call"),
                                               (got3, got3_lse, want1, want1_lse, "third call")):
        close(got, want, what)
        # same kernels, same schedule, same reduction order: in fact the same bits
        assert torch.equal(got.view(torch.int16), want.view(torch.int16)), what
        assert torch.equal(got_lse.nan_to_num(neginf=-1e30), want_lse.nan_to_num(neginf=-1e30)), what
    # with the launch flags of the bench (early mode + small dependent combine)
    w7, w7_lse = existing(b1, flags=7)
    g7, g7_lse = static(b1, flags=7)
    torch.cuda.synchronize()
    close(g7, w7, "flags 7")
    assert torch.equal(g7.view(torch.int16), w7.view(torch.int16)) and torch.equal(g7_lse, w7_lse)


def test_static_scratch_rejects_shapes_beyond_the_array():
    assert comem.comem_static_scratch_bytes() == 12 << 20
    b = W.make_batch([40] * 600, 64, 8, 128, 16, seed=9103, device=DEV)
    assert comem.comem_decode_attn_workspace_bytes(600, 64, 8, 128, 16, b.block_table.shape[1]) > comem.comem_static_scratch_bytes()
    out = torch.empty_like(b.q)
    with pytest.raises(comem.ComemError) as e:
        comem.comem_decode_attn_static_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out)
    assert e.value.status == comem.COMEM_ERR_WORKSPACE
    # a batch that fits: 256 sequences at 16 q heads / 4 kv heads
    s = W.make_batch([int(x) for x in np.random.default_rng(5).integers(0, 900, 256)], 16, 4, 128, 16, seed=9104, device=DEV)
    want, _ = existing(s)
    got, _ = static(s)
    torch.cuda.synchronize()
    assert torch.equal(got.view(torch.int16), want.view(torch.int16))
