"""Pins of oracle.prefill_attn (causal prefill of the last q_len tokens of each sequence over the paged cache,
SURVEY.md §8(f).2, Alg. 1 lines 9-13; reading R20).  No kernel is built on it yet (next round).
  PF1  q_len = 1 for every sequence is the decode step: bit-identical to the pinned decode oracle (O1..O16)
  PF2  causality as a prefix property: row i of a chunk equals the DECODE oracle on the same cache truncated to
       pos_i + 1 tokens, with that row as its query -- bit-identical, every row, ragged chunk lengths
  PF3  uncached full prefill (q_len = L) against torch's fp64 scaled_dot_product_attention with is_causal=True
  PF4  chunking invariance (Alg. 1: cached incremental prefill == uncached full prefill on the same tokens):
       the rows of a prompt processed in chunks are bit-identical to the same rows of one full prefill
  PF5  brute-force dense masked softmax in numpy fp64; first token of a full prefill returns V[0] exactly
"""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2605_30842_b200 import workloads as W


def _ragged_q(lens_q, hq, d, seed):
    g = torch.Generator().manual_seed(seed)
    q = torch.randn((sum(lens_q), hq, d), generator=g).to(torch.bfloat16)
    qs = np.concatenate([[0], np.cumsum(lens_q)]).astype(np.int32)
    return q, qs


def test_pf1_single_query_is_decode(oracle):
    b = W.make_batch([1, 37, 500, 16], 8, 2, 64, 16, seed=701)
    qs = np.arange(5, dtype=np.int32)
    out, lse = oracle.prefill_attn(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, qs, b.softmax_scale)
    want, want_lse = oracle.decode_attn(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale)
    assert np.array_equal(out, want) and np.array_equal(lse, want_lse)


def test_pf2_each_row_is_decode_on_truncated_cache(oracle):
    lens, lens_q = [70, 33, 16, 200], [70, 5, 1, 64]
    b = W.make_batch(lens, 6, 3, 64, 16, seed=702)
    q, qs = _ragged_q(lens_q, 6, 64, seed=7)
    out, lse = oracle.prefill_attn(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, qs, b.softmax_scale)
    for s in range(4):
        for i in range(lens_q[s]):
            row = int(qs[s]) + i
            pos = lens[s] - lens_q[s] + i
            trunc = torch.tensor([pos + 1], dtype=torch.int32)
            want, want_lse = oracle.decode_attn(q[row:row + 1], b.k_pages, b.v_pages, b.block_table[s:s + 1], trunc,
                                                b.softmax_scale)
            assert np.array_equal(out[row], want[0]) and np.array_equal(lse[row], want_lse[0]), (s, i)


@pytest.mark.parametrize("G,ps", [(1, 16), (4, 32)])
def test_pf3_full_prefill_vs_torch_causal_sdpa(oracle, G, ps):
    L, hkv, d = 90, 2, 64
    b = W.make_batch([L], G * hkv, hkv, d, ps, seed=703 + G)
    q, qs = _ragged_q([L], G * hkv, d, seed=8)
    out, _ = oracle.prefill_attn(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, qs, b.softmax_scale)
    n = W.pages_needed(L, ps)
    ids = b.block_table[0, :n].long()
    k = b.k_pages[ids].reshape(n * ps, hkv, d)[:L].double().repeat_interleave(G, dim=1).permute(1, 0, 2)
    v = b.v_pages[ids].reshape(n * ps, hkv, d)[:L].double().repeat_interleave(G, dim=1).permute(1, 0, 2)
    ref = torch.nn.functional.scaled_dot_product_attention(q.double().permute(1, 0, 2)[None], k[None], v[None],
                                                           is_causal=True, scale=float(np.float32(b.softmax_scale)))
    assert np.max(np.abs(out - ref[0].permute(1, 0, 2).numpy())) <= 1e-12


def test_pf4_chunked_equals_full(oracle):
    L = 150
    b = W.make_batch([L], 4, 2, 64, 16, seed=704)
    q, qs = _ragged_q([L], 4, 64, seed=9)
    full, full_lse = oracle.prefill_attn(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, qs, b.softmax_scale)
    done = 0
    for chunk in (1, 15, 16, 17, 64, 37):               # the cache grows as Alg. 1's cached prefill appends
        sl = torch.tensor([done + chunk], dtype=torch.int32)
        o, l = oracle.prefill_attn(q[done:done + chunk], b.k_pages, b.v_pages, b.block_table, sl,
                                   np.array([0, chunk], np.int32), b.softmax_scale)
        assert np.array_equal(o, full[done:done + chunk]) and np.array_equal(l, full_lse[done:done + chunk])
        done += chunk
    assert done == L


def test_pf5_brute_force_and_first_token(oracle):
    lens, lens_q = [40, 9], [12, 9]
    b = W.make_batch(lens, 4, 2, 64, 16, seed=705)
    q, qs = _ragged_q(lens_q, 4, 64, seed=10)
    out, lse = oracle.prefill_attn(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, qs, b.softmax_scale)
    for s, (L, n) in enumerate(zip(lens, lens_q)):
        npg = W.pages_needed(L, 16)
        ids = b.block_table[s, :npg].long()
        k = b.k_pages[ids].reshape(npg * 16, 2, 64)[:L].double().numpy()
        v = b.v_pages[ids].reshape(npg * 16, 2, 64)[:L].double().numpy()
        for i in range(n):
            pos = L - n + i
            for h in range(4):
                sc = float(np.float32(b.softmax_scale)) * (k[:pos + 1, h // 2] @ q[int(qs[s]) + i, h].double().numpy())
                w = np.exp(sc - sc.max())
                want = (w[:, None] * v[:pos + 1, h // 2]).sum(0) / w.sum()
                assert np.max(np.abs(out[int(qs[s]) + i, h] - want)) <= 1e-13
    # sequence 1 is a full prefill (9 of 9): its first query sees one key and returns V[0] exactly
    ids = b.block_table[1, :1].long()
    v0 = b.v_pages[ids].reshape(16, 2, 64)[0].double().numpy()
    for h in range(4):
        assert np.array_equal(out[int(qs[1]), h], v0[h // 2])
    with pytest.raises(ValueError):
        oracle.prefill_attn(q, b.k_pages, b.v_pages, b.block_table, torch.tensor([5, 9], dtype=torch.int32), qs,
                            b.softmax_scale)                      # more new tokens than cached tokens
