"""Pins for oracle/decode_attn_oracle.c — CPU only.

Each pin checks the oracle against something other than itself: a closed form,
an invariant, a library routine (torch CPU fp64 SDPA) or an independent dense
numpy brute force.  PAPER.md prints no numeric attention output, so there is no
worked example to match ("Oracle pins").
"""
import math

import numpy as np
import pytest
import torch

from paper_2605_30842_b200 import workloads as W


def bf16(x) -> torch.Tensor:
    return torch.as_tensor(x, dtype=torch.float32).to(torch.bfloat16)


def to_f64(t: torch.Tensor) -> np.ndarray:
    return t.to(torch.float64).numpy()


def dense_kv(batch: W.DecodeBatch, b: int):
    """Gather sequence b's logical K, V as dense float64 [L, Hkv, D] (independent of the oracle)."""
    L = int(batch.seq_lens[b])
    ps = batch.page_size
    t = np.arange(L)
    pid = batch.block_table[b].numpy()[t // ps]
    k = to_f64(batch.k_pages)[pid, t % ps]
    v = to_f64(batch.v_pages)[pid, t % ps]
    return k, v


def brute_force(batch: W.DecodeBatch):
    """Independent dense numpy float64 softmax(QK^T)V with heads repeated (O13)."""
    B, Hq, D = batch.q.shape
    G = Hq // batch.num_kv_heads
    out = np.zeros((B, Hq, D))
    lse = np.full((B, Hq), -np.inf)
    q = to_f64(batch.q)
    scale = float(np.float32(batch.softmax_scale))
    for b in range(B):
        if int(batch.seq_lens[b]) == 0:
            continue
        k, v = dense_kv(batch, b)
        k = np.repeat(k, G, axis=1)            # [L, Hq, D]
        v = np.repeat(v, G, axis=1)
        s = scale * np.einsum("hd,lhd->hl", q[b], k)
        m = s.max(axis=1, keepdims=True)
        p = np.exp(s - m)
        z = p.sum(axis=1, keepdims=True)
        out[b] = np.einsum("hl,lhd->hd", p / z, v)
        lse[b] = (m + np.log(z))[:, 0]
    return out, lse


def single_seq(q, k, v, page_size=16, scale=None, num_kv_heads=1):
    """Lay a dense single sequence [L, Hkv, D] into an identity-mapped paged pool."""
    L, Hkv, D = k.shape
    npg = max(1, W.pages_needed(L, page_size))
    kp = torch.zeros((npg, page_size, Hkv, D), dtype=torch.bfloat16)
    vp = torch.zeros_like(kp)
    kp.view(-1, Hkv, D)[:L] = k
    vp.view(-1, Hkv, D)[:L] = v
    bt = torch.arange(npg, dtype=torch.int32).view(1, -1)
    sl = torch.tensor([L], dtype=torch.int32)
    if scale is None:
        scale = 1.0 / math.sqrt(D)
    return W.DecodeBatch(q=q.view(1, -1, D), k_pages=kp, v_pages=vp, block_table=bt, seq_lens=sl,
                         softmax_scale=W.f32(scale))


def run(oracle, batch, **kw):
    return oracle.decode_attn(batch.q, batch.k_pages, batch.v_pages, batch.block_table,
                              batch.seq_lens, batch.softmax_scale, **kw)


# ---- O1: single-token context returns V exactly ------------------------------------------
def test_o1_single_token_returns_v(oracle):
    b = W.make_batch([1, 1, 1], 8, 2, 64, 16, seed=11)
    out, lse = run(oracle, b)
    G = 4
    for i in range(3):
        _, v = dense_kv(b, i)
        for h in range(8):
            assert np.array_equal(out[i, h], v[0, h // G])


# ---- O2 / O15: identical keys -> mean of V, lse = s + log L -----------------------------------
@pytest.mark.parametrize("L", [2, 17, 300])
def test_o2_identical_keys_mean_of_v(oracle, L):
    g = torch.Generator().manual_seed(L)
    D = 64
    q = bf16(torch.randn(4, D, generator=g))
    k1 = bf16(torch.randn(1, 1, D, generator=g))
    k = k1.expand(L, 1, D).contiguous()
    v = bf16(torch.randn(L, 1, D, generator=g))
    b = single_seq(q, k, v)
    out, lse = run(oracle, b)
    mean_v = to_f64(v)[:, 0].mean(axis=0)
    s = float(np.float32(b.softmax_scale)) * (to_f64(q) @ to_f64(k1)[0, 0])
    for h in range(4):
        np.testing.assert_allclose(out[0, h], mean_v, rtol=1e-13, atol=1e-15)
        assert abs(lse[0, h] - (s[h] + math.log(L))) <= 1e-12 * max(1.0, abs(s[h]))


# ---- O3: zero scale or zero query -> mean of V --------------------------------------------
def test_o3_zero_scale_or_zero_query(oracle):
    b = W.make_batch([45], 4, 1, 64, 16, seed=3)
    _, v = dense_kv(b, 0)
    b0 = W.DecodeBatch(**{**b.__dict__, "softmax_scale": 0.0})
    out, _ = run(oracle, b0)
    np.testing.assert_allclose(out[0, 2], v[:, 0].mean(axis=0), rtol=1e-13, atol=1e-15)
    bq = W.DecodeBatch(**{**b.__dict__, "q": torch.zeros_like(b.q)})
    out, _ = run(oracle, bq)
    np.testing.assert_allclose(out[0, 1], v[:, 0].mean(axis=0), rtol=1e-13, atol=1e-15)


# ---- O4: two keys -> logistic closed form ---------------------------------------------------
def test_o4_two_keys_logistic(oracle):
    g = torch.Generator().manual_seed(4)
    D = 128
    q = bf16(torch.randn(2, D, generator=g))
    k = bf16(torch.randn(2, 1, D, generator=g))
    v = bf16(torch.randn(2, 1, D, generator=g))
    b = single_seq(q, k, v, page_size=32)
    out, _ = run(oracle, b)
    scale = float(np.float32(b.softmax_scale))
    for h in range(2):
        delta = scale * (to_f64(q)[h] @ (to_f64(k)[0, 0] - to_f64(k)[1, 0]))
        sig = 1.0 / (1.0 + math.exp(-delta))
        want = sig * to_f64(v)[0, 0] + (1.0 - sig) * to_f64(v)[1, 0]
        np.testing.assert_allclose(out[0, h], want, rtol=1e-13, atol=1e-15)


# ---- O5: constant V -> out = c ----------------------------------------------------------------
def test_o5_constant_v(oracle):
    b = W.make_batch([100, 33], 8, 2, 64, 16, seed=5)
    c = bf16(torch.randn(64, generator=torch.Generator().manual_seed(55)))
    b.v_pages[:] = c
    out, _ = run(oracle, b)
    np.testing.assert_allclose(out, np.broadcast_to(to_f64(c), out.shape), rtol=1e-14, atol=0)


# ---- O6: linearity in V (bf16-exact integer values) ------------------------------------
def test_o6_linear_in_v(oracle):
    b = W.make_batch([77], 4, 1, 64, 16, seed=6)
    g = torch.Generator().manual_seed(66)
    v1 = torch.randint(-8, 9, b.v_pages.shape, generator=g).float()
    v2 = torch.randint(-8, 9, b.v_pages.shape, generator=g).float()
    outs = []
    for v in (v1, v2, v1 + v2):
        bb = W.DecodeBatch(**{**b.__dict__, "v_pages": v.to(torch.bfloat16)})
        outs.append(run(oracle, bb)[0])
    np.testing.assert_allclose(outs[2], outs[0] + outs[1], rtol=1e-13, atol=1e-13)


# ---- O7: key-shift invariance (small-integer K so the shifted keys stay bf16-exact) ---------
def test_o7_key_shift_invariance(oracle):
    b = W.make_batch([50], 4, 1, 64, 16, seed=7)
    g = torch.Generator().manual_seed(77)
    k = torch.randint(-4, 5, b.k_pages.shape, generator=g).float()
    c = torch.randint(-3, 4, (64,), generator=g).float()
    b1 = W.DecodeBatch(**{**b.__dict__, "k_pages": k.to(torch.bfloat16)})
    b2 = W.DecodeBatch(**{**b.__dict__, "k_pages": (k + c).to(torch.bfloat16)})
    o1, l1 = run(oracle, b1)
    o2, l2 = run(oracle, b2)
    np.testing.assert_allclose(o1, o2, rtol=1e-12, atol=1e-13)
    # and lse shifts by exactly scale * q.c
    shift = float(np.float32(b.softmax_scale)) * (to_f64(b.q)[0] @ c.double().numpy())
    np.testing.assert_allclose(l2[0] - l1[0], shift, rtol=1e-10, atol=1e-10)


# ---- O8: one logit +80 above the rest -> its V, no overflow ----------------------------------
def test_o8_dominant_logit(oracle):
    D, L = 64, 40
    q = torch.zeros(1, D); q[0, 0] = 16.0
    k = torch.zeros(L, 1, D); k[:, 0, 0] = 30.0      # logits 16*30/8 = 60
    k[13, 0, 0] = 70.0                               # logit 140: +80 above, exp(140) finite in fp64? no: needs max-subtraction
    v = torch.randn(L, 1, D, generator=torch.Generator().manual_seed(8))
    b = single_seq(bf16(q), bf16(k), bf16(v))
    out, lse = run(oracle, b)
    assert np.all(np.isfinite(out)) and np.isfinite(lse[0, 0])
    want = to_f64(bf16(v))[13, 0]
    np.testing.assert_allclose(out[0, 0], want, rtol=0, atol=(L * math.exp(-80.0)) * 10)
    assert abs(lse[0, 0] - 140.0) < 1e-9
    # huge logits: scale * q.k = 800 would overflow exp() without the max subtraction
    k[:, 0, 0] = 100.0; k[13, 0, 0] = 400.0
    b = single_seq(bf16(q), bf16(k), bf16(v))
    out, lse = run(oracle, b)
    assert np.all(np.isfinite(out))
    np.testing.assert_array_equal(out[0, 0], want)


# ---- O9: physical page permutation leaves the result bit-identical ---------------------------
def test_o9_page_permutation_bit_identical(oracle):
    b = W.make_batch([130, 17, 64], 8, 2, 64, 16, seed=9, num_pages=40)
    o1, l1 = run(oracle, b)
    b2 = W.permute_pages(b, seed=99)
    assert not torch.equal(b.block_table, b2.block_table)
    o2, l2 = run(oracle, b2)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


# ---- O10: GQA convention kvh = h // G ------------------------------------------------------------
def test_o10_gqa_grouping(oracle):
    b = W.make_batch([60], 8, 2, 64, 16, seed=10)
    qrow = b.q[0, 0].clone()
    b.q[0, :] = qrow                     # identical q in all 8 heads
    out, _ = run(oracle, b)
    for h in (1, 2, 3):
        assert np.array_equal(out[0, h], out[0, 0])          # group 0 shares KV head 0
    for h in (5, 6, 7):
        assert np.array_equal(out[0, h], out[0, 4])          # group 1 shares KV head 1
    assert not np.array_equal(out[0, 0], out[0, 4])
    # head 4's result equals a 1-head problem run against KV head 1 alone
    k, v = dense_kv(b, 0)
    solo = single_seq(qrow.view(1, -1), bf16(k[:, 1:2]), bf16(v[:, 1:2]))
    o_solo, _ = run(oracle, solo)
    assert np.array_equal(o_solo[0, 0], out[0, 4])


# ---- O11: split invariance pins the partial + LSE-merge formulas -------------------------------
@pytest.mark.parametrize("cuts", [[0, 200], [0, 1, 200], [0, 16, 17, 100, 199, 200], [0, 0, 64, 64, 200]])
def test_o11_split_merge_invariance(oracle, cuts):
    b = W.make_batch([200], 4, 2, 64, 16, seed=111)
    full, lse_full = run(oracle, b)
    for h in range(4):
        accs, ms, ls = [], [], []
        for t0, t1 in zip(cuts[:-1], cuts[1:]):
            a, m, l = oracle.decode_attn_partial(b.q, b.k_pages, b.v_pages, b.block_table,
                                                 b.seq_lens, b.softmax_scale, 0, h, t0, t1)
            accs.append(a); ms.append(m); ls.append(l)
        out, lse = oracle.lse_merge(np.stack(accs), np.array(ms), np.array(ls))
        np.testing.assert_allclose(out, full[0, h], rtol=1e-13, atol=1e-15)
        assert abs(lse - lse_full[0, h]) < 1e-12
    # all-empty merge
    out, lse = oracle.lse_merge(np.zeros((2, 64)), np.array([-np.inf, -np.inf]), np.zeros(2))
    assert np.all(out == 0.0) and lse == -np.inf


# ---- O12: tail-poison independence ----------------------------------------------------------------
def test_o12_tail_poison_independence(oracle):
    lens = [37, 16, 5]
    clean = W.make_batch(lens, 8, 2, 64, 16, seed=12, num_pages=12, max_pages_per_seq=6)
    dirty = W.make_batch(lens, 8, 2, 64, 16, seed=12, num_pages=12, max_pages_per_seq=6,
                         poison_unused=True)
    assert torch.isnan(dirty.k_pages.float()).any()
    dirty.block_table[dirty.block_table < 0] = 2 ** 30        # out-of-range ids in ignored entries
    o1, l1 = run(oracle, clean)
    o2, l2 = run(oracle, dirty)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)
    for poison in (float("inf"), -float("inf"), 1e38):
        d2 = W.make_batch(lens, 8, 2, 64, 16, seed=12, num_pages=12, max_pages_per_seq=6,
                          poison_unused=True)
        d2.k_pages[torch.isnan(d2.k_pages.float())] = poison
        d2.v_pages[torch.isnan(d2.v_pages.float())] = poison
        o3, _ = run(oracle, d2)
        assert np.array_equal(o1, o3)


# ---- O13: brute force on tiny inputs ---------------------------------------------------------
@pytest.mark.parametrize("G", [1, 4, 8])
@pytest.mark.parametrize("D", [64, 128])
@pytest.mark.parametrize("ps", [16, 32])
def test_o13_dense_brute_force(oracle, G, D, ps):
    for B, lens in ((1, [512]), (3, [1, 17, 33]), (3, [15, 16, 31])):
        b = W.make_batch(lens, 2 * G, 2, D, ps, seed=1300 + G + D + ps + B)
        out, lse = run(oracle, b)
        want, want_lse = brute_force(b)
        np.testing.assert_allclose(out, want, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(lse, want_lse, rtol=1e-12, atol=1e-12)


def test_o13_pairs_subset_matches_full(oracle):
    b = W.make_batch([40, 90], 8, 2, 64, 16, seed=131)
    full, lse = run(oracle, b)
    pairs = [(1, 5), (0, 0), (1, 7)]
    sub, sub_lse = run(oracle, b, pairs=pairs)
    for i, (bb, h) in enumerate(pairs):
        assert np.array_equal(sub[i], full[bb, h]) and sub_lse[i] == lse[bb, h]
    one, _ = run(oracle, b, num_threads=1)
    assert np.array_equal(one, full)                      # thread count does not change bits


# ---- O14: torch CPU float64 scaled_dot_product_attention ----------------------------------
def test_o14_torch_sdpa_fp64(oracle):
    b = W.make_batch([257], 8, 2, 128, 16, seed=14)
    out, _ = run(oracle, b)
    k, v = dense_kv(b, 0)
    G = 4
    kt = torch.from_numpy(np.repeat(k, G, axis=1)).permute(1, 0, 2)    # [Hq, L, D]
    vt = torch.from_numpy(np.repeat(v, G, axis=1)).permute(1, 0, 2)
    qt = b.q[0].double().unsqueeze(1)                                  # [Hq, 1, D]
    ref = torch.nn.functional.scaled_dot_product_attention(
        qt, kt, vt, scale=float(np.float32(b.softmax_scale)))
    np.testing.assert_allclose(out[0], ref[:, 0].numpy(), rtol=1e-12, atol=1e-14)


# ---- R9: empty sequence -> zeros, lse = -inf -------------------------------------------------
def test_empty_sequence(oracle):
    b = W.make_batch([0, 20], 4, 1, 64, 16, seed=15, max_pages_per_seq=2)
    out, lse = run(oracle, b)
    assert np.all(out[0] == 0.0) and np.all(lse[0] == -np.inf)
    assert np.all(np.isfinite(out[1]))


# ---- O16: byte accounting (Qwen3-32B FP16, 16 GB per 64K tokens) ---------------
def test_o16_paper_kv_bytes():
    layers, hkv, d, bytes_per = 64, 8, 128, 2
    per_token = 2 * layers * hkv * d * bytes_per
    assert per_token == 262144
    assert per_token * 65536 == 16 * 2 ** 30                  # "16 GB to save a sequence of 64K tokens"
    b = W.make_batch([100, 28], 64, 8, 128, 16, seed=16)
    assert b.algorithmic_bytes() == 128 * 8 * 128 * 2 * 2 + 2 * 64 * 128 * 2


# ---- eq. 7 case study: closed form re-derived ----------------------------
def test_eq7_case_study_golden():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "eq7_case_study.txt")
    vals = dict(line.split("=") for line in open(path).read().split() if "=" in line)
    Wb, P, S, Y = (float(vals[k]) for k in ("W_GBps", "P_tok_s", "S_GB_per_tok", "Y_tokens"))
    ratio = 1.0 / (1.0 + Wb / (Y * S * P))
    assert round(ratio, 2) == float(vals["ratio_printed"])
    assert abs(float(vals["ratio_printed"]) * 32000 - float(vals["summary_tokens_printed"])) < 1e-6


# ---- KV append ----------------------------------------------------------------------
def test_kv_append_then_attend(oracle):
    b = W.make_batch([15, 16, 31], 4, 2, 64, 16, seed=17, spare_tokens=3)
    kb, vb = oracle.as_bits(b.k_pages).copy(), oracle.as_bits(b.v_pages).copy()
    sl = b.seq_lens.numpy().copy()
    dense_before = [dense_kv(b, i) for i in range(3)]
    news = []
    for step in range(3):
        _, nk, nv = W.decode_step_rows(b, step, 1700)
        oracle.kv_append(kb, vb, b.block_table, sl, nk, nv)
        news.append((nk, nv))
    assert list(sl) == [18, 19, 34]
    b2 = W.DecodeBatch(**{**b.__dict__,
                          "k_pages": torch.from_numpy(kb.view(np.int16)).view(torch.bfloat16),
                          "v_pages": torch.from_numpy(vb.view(np.int16)).view(torch.bfloat16),
                          "seq_lens": torch.from_numpy(sl)})
    for i in range(3):
        k, v = dense_kv(b2, i)
        k0, v0 = dense_before[i]
        assert np.array_equal(k[:len(k0)], k0) and np.array_equal(v[:len(v0)], v0)
        for step in range(3):
            assert np.array_equal(k[len(k0) + step], to_f64(news[step][0])[i])
            assert np.array_equal(v[len(v0) + step], to_f64(news[step][1])[i])
    out, _ = run(oracle, b2)
    want, _ = brute_force(b2)
    np.testing.assert_allclose(out, want, rtol=1e-12, atol=1e-14)
