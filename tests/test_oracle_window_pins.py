"""Pins of oracle.decode_attn_window (sliding window + attention sinks, reading R17;
PAPER.md L19 / L316 name the technique, no formula).  What fixes it other than itself:
  W1  window >= L or window <= 0 -> bit-identical to the full oracle (itself pinned by O1..O15)
  W2  window = 1, no sinks -> out = V[L-1] exactly; window = 1 + sinks = 1 -> two-key logistic
  W3  equals FULL attention (the pinned oracle) over a cache compacted to the kept tokens
  W4  contents of masked tokens are irrelevant (NaN / Inf poison) -> bit-identical
  W5  brute-force dense masked softmax in numpy fp64
"""
import numpy as np
import pytest
import torch

from paper_2605_30842_b200 import workloads as W


def _kept(L, window, sinks):
    lo = 0 if (window <= 0 or window >= L) else L - window
    return [t for t in range(L) if t < sinks or t >= lo]


def _dense(batch, b):
    L, ps = int(batch.seq_lens[b]), batch.page_size
    n = W.pages_needed(L, ps)
    ids = batch.block_table[b, :n].long()
    k = batch.k_pages[ids].reshape(n * ps, batch.num_kv_heads, batch.head_dim)[:L].double().numpy()
    v = batch.v_pages[ids].reshape(n * ps, batch.num_kv_heads, batch.head_dim)[:L].double().numpy()
    return k, v


def test_w1_no_window_is_full_oracle(oracle):
    b = W.make_batch([1, 37, 0, 500], 8, 2, 64, 16, seed=301)
    full, lse = oracle.decode_attn(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale)
    for window, sinks in ((0, 0), (500, 0), (10 ** 6, 3), (-1, 0)):
        o, l = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                         window, sinks)
        assert np.array_equal(o, full) and np.array_equal(l, lse)
    # sinks that reach the window leave nothing masked either
    o, _ = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, 100, 400)
    assert np.array_equal(o, full)


def test_w2_window_one_closed_forms(oracle):
    b = W.make_batch([333], 4, 1, 64, 16, seed=302)
    o, lse = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, 1, 0)
    k, v = _dense(b, 0)
    assert np.array_equal(o[0], np.repeat(v[332][None, 0], 4, axis=0))         # weight exactly 1
    s_last = float(np.float32(b.softmax_scale)) * (b.q[0].double().numpy() @ k[332, 0])
    assert np.allclose(lse[0], s_last, rtol=0, atol=1e-12)
    # one sink + window 1: logistic mix of V[0] and V[L-1]
    o, _ = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, 1, 1)
    s0 = float(np.float32(b.softmax_scale)) * (b.q[0].double().numpy() @ k[0, 0])
    w0 = 1.0 / (1.0 + np.exp(s_last - s0))
    want = w0[:, None] * v[0, 0][None] + (1 - w0)[:, None] * v[332, 0][None]
    assert np.max(np.abs(o[0] - want)) <= 1e-13


@pytest.mark.parametrize("window,sinks", [(64, 0), (64, 4), (17, 16), (1, 5), (200, 33)])
def test_w3_equals_full_attention_on_compacted_cache(oracle, window, sinks):
    """Build a second cache holding ONLY the kept tokens, in order, and run the FULL oracle on it."""
    lens = [700, 65, 16]
    b = W.make_batch(lens, 8, 2, 64, 16, seed=303)
    o, lse = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                       window, sinks)
    ps = 16
    kept = [_kept(L, window, sinks) for L in lens]
    npg = [W.pages_needed(len(k), ps) for k in kept]
    kp = torch.zeros((sum(npg), ps, 2, 64), dtype=torch.bfloat16)
    vp = torch.zeros_like(kp)
    bt = torch.zeros((3, max(npg)), dtype=torch.int32)
    off = 0
    for i, L in enumerate(lens):
        bt[i, :npg[i]] = torch.arange(off, off + npg[i], dtype=torch.int32)
        for j, t in enumerate(kept[i]):
            src = int(b.block_table[i, t // ps])
            kp[off + j // ps, j % ps] = b.k_pages[src, t % ps]
            vp[off + j // ps, j % ps] = b.v_pages[src, t % ps]
        off += npg[i]
    sl = torch.tensor([len(k) for k in kept], dtype=torch.int32)
    ref, ref_lse = oracle.decode_attn(b.q, kp, vp, bt, sl, b.softmax_scale)
    assert np.max(np.abs(o - ref)) <= 1e-13 and np.max(np.abs(lse - ref_lse)) <= 1e-12


def test_w4_masked_tokens_do_not_matter(oracle):
    b = W.make_batch([400, 90], 8, 2, 64, 16, seed=304)
    window, sinks = 48, 5
    o1, l1 = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                       window, sinks)
    for poison in (float("nan"), float("inf"), -1e38):
        for i, L in enumerate((400, 90)):
            keep = set(_kept(L, window, sinks))
            for t in range(L):
                if t not in keep:
                    pid = int(b.block_table[i, t // 16])
                    b.k_pages[pid, t % 16] = poison
                    b.v_pages[pid, t % 16] = poison
        o2, l2 = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                           window, sinks)
        assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


@pytest.mark.parametrize("G,ps", [(1, 16), (4, 32), (8, 16)])
def test_w5_dense_masked_brute_force(oracle, G, ps):
    lens = [1, 15, 16, 17, 33, 260]
    b = W.make_batch(lens, 2 * G, 2, 64, ps, seed=305 + G)
    for window, sinks in ((8, 0), (16, 2), (31, 17), (100, 1)):
        o, lse = oracle.decode_attn_window(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                           window, sinks)
        scale = float(np.float32(b.softmax_scale))
        for i, L in enumerate(lens):
            k, v = _dense(b, i)
            idx = _kept(L, window, sinks)
            for h in range(2 * G):
                s = scale * (k[idx, h // G] @ b.q[i, h].double().numpy())
                p = np.exp(s - s.max())
                want = (p[:, None] * v[idx, h // G]).sum(0) / p.sum()
                assert np.max(np.abs(o[i, h] - want)) <= 1e-12
                assert abs(lse[i, h] - (s.max() + np.log(p.sum()))) <= 1e-12
