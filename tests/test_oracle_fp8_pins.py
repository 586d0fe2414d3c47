"""Pins of oracle.decode_attn_fp8 / oracle.e4m3_decode (FP8 E4M3 KV cache with one fp32 scale per
physical page and kv head, reading R18; PAPER.md L25 names KV-cache quantisation, no format).
What fixes it other than itself:
  F1  the 256-entry decode table: the format's published values (OCP 8-bit floating point
      specification, E4M3: bias 7, max 448 = 0x7e, min normal 2^-6 = 0x08, min subnormal 2^-9 = 0x01,
      1.0 = 0x38, NaN = 0x7f / 0xff, no infinities), monotone in the magnitude bits, odd in the sign;
      and, independently, torch's own float8_e4m3fn -> float32 cast for every byte
  F2  on a cache whose values BOTH formats hold exactly (small dyadic numbers) with power-of-two
      scales, it is bit-identical to the bf16 oracle (itself pinned by O1..O16) on the dequantised
      cache -- also through the window arguments (vs the window oracle, W1..W5)
  F3  L = 1 -> out = v_scale * e4m3(V8[0]) exactly; lse = softmax_scale * q . (k_scale * e4m3(K8[0]))
  F4  scale linearity: v_scale * c (per page) with constant c -> out * c; k_scale * c == softmax_scale * c
      (c a power of two: exact)
  F5  tail slots, unowned pages and their scales are irrelevant (NaN poison) -> bit-identical
  F6  brute-force dense softmax in numpy fp64 on the dequantised arrays (dequantised with torch's
      cast, not the oracle's table), per-page scales that differ page to page
  F7  kv_layout "HND" ([P, Hkv, page_size, D]) on the transposed pools is bit-identical to "NHD" on the
      original ones (only the row address differs)
"""
import numpy as np
import pytest
import torch

from paper_2605_30842_b200 import workloads as W


def _torch_decode_all():
    return torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).float().double().numpy()


def test_f1_decode_table_published_values(oracle):
    dec = np.array([oracle.e4m3_decode(b) for b in range(256)])
    assert dec[0x00] == 0.0 and dec[0x80] == 0.0 and np.signbit(dec[0x80])
    assert dec[0x38] == 1.0 and dec[0xb8] == -1.0
    assert dec[0x7e] == 448.0 and dec[0xfe] == -448.0
    assert dec[0x08] == 2.0 ** -6 and dec[0x01] == 2.0 ** -9 and dec[0x07] == 7 * 2.0 ** -9
    assert dec[0x40] == 2.0 and dec[0x3c] == 1.5 and dec[0x39] == 1.125 and dec[0x30] == 0.5
    assert dec[0x78] == 256.0 and dec[0x77] == 240.0
    assert np.isnan(dec[0x7f]) and np.isnan(dec[0xff])
    assert np.isfinite(np.delete(dec, [0x7f, 0xff])).all()           # no infinities
    assert np.all(np.diff(dec[0:0x7f]) > 0)                            # monotone in the magnitude bits
    assert np.array_equal(dec[0x80:0xff], -dec[0x00:0x7f])             # sign bit only flips the sign


def test_f1_decode_table_matches_torch_cast(oracle):
    dec = np.array([oracle.e4m3_decode(b) for b in range(256)])
    ref = _torch_decode_all()
    assert np.array_equal(np.isnan(dec), np.isnan(ref))
    ok = ~np.isnan(ref)
    assert np.array_equal(dec[ok], ref[ok])


def _exact_batch(lens, hq, hkv, d, ps, seed):
    """A bf16 batch whose K/V values are k/8 for integer |k| <= 15 (exact in E4M3 and in bf16), and its
    FP8 twin with power-of-two page scales folded in: bf16 value = 2^e * e4m3 value exactly."""
    b = W.make_batch(lens, hq, hkv, d, ps, seed=seed)
    g = torch.Generator().manual_seed(seed)
    P = b.num_pages
    kq = torch.randint(-15, 16, (P, ps, hkv, d), generator=g).float() / 8
    vq = torch.randint(-15, 16, (P, ps, hkv, d), generator=g).float() / 8
    ke = torch.randint(-3, 4, (P, hkv), generator=g).float()
    ve = torch.randint(-3, 4, (P, hkv), generator=g).float()
    ks, vs = torch.exp2(ke), torch.exp2(ve)
    k8 = kq.to(torch.float8_e4m3fn)
    v8 = vq.to(torch.float8_e4m3fn)
    assert torch.equal(k8.float(), kq) and torch.equal(v8.float(), vq)   # representable: the cast is exact
    kb = (kq * ks.view(P, 1, hkv, 1)).to(torch.bfloat16)
    vb = (vq * vs.view(P, 1, hkv, 1)).to(torch.bfloat16)
    assert torch.equal(kb.float(), kq * ks.view(P, 1, hkv, 1))
    import dataclasses
    bf = dataclasses.replace(b, k_pages=kb, v_pages=vb)
    f8 = W.Fp8DecodeBatch(q=b.q, k_pages=k8.view(torch.uint8), v_pages=v8.view(torch.uint8), k_scale=ks, v_scale=vs,
                          block_table=b.block_table, seq_lens=b.seq_lens, softmax_scale=b.softmax_scale)
    return bf, f8


def _run8(oracle, f, window=0, sinks=0):
    return oracle.decode_attn_fp8(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                  f.softmax_scale, window, sinks)


def test_f2_equals_bf16_oracle_on_exactly_representable_cache(oracle):
    bf, f8 = _exact_batch([1, 77, 0, 300], 8, 2, 64, 16, seed=411)
    want, want_lse = oracle.decode_attn(bf.q, bf.k_pages, bf.v_pages, bf.block_table, bf.seq_lens, bf.softmax_scale)
    got, got_lse = _run8(oracle, f8)
    assert np.array_equal(got, want) and np.array_equal(got_lse, want_lse)
    for window, sinks in ((64, 0), (17, 5), (1, 0)):
        want, want_lse = oracle.decode_attn_window(bf.q, bf.k_pages, bf.v_pages, bf.block_table, bf.seq_lens,
                                                   bf.softmax_scale, window, sinks)
        got, got_lse = _run8(oracle, f8, window, sinks)
        assert np.array_equal(got, want) and np.array_equal(got_lse, want_lse)


def test_f2_page_size_32_and_gqa_map(oracle):
    bf, f8 = _exact_batch([95, 33], 6, 3, 64, 32, seed=412)
    want, _ = oracle.decode_attn(bf.q, bf.k_pages, bf.v_pages, bf.block_table, bf.seq_lens, bf.softmax_scale)
    got, _ = _run8(oracle, f8)
    assert np.array_equal(got, want)


def test_f3_single_token_closed_form(oracle):
    f = W.quantize_batch_fp8(W.make_batch([1], 4, 2, 64, 16, seed=413))
    out, lse = _run8(oracle, f)
    pid = int(f.block_table[0, 0])
    dec = _torch_decode_all()
    for h in range(4):
        kvh = h // 2
        v = float(f.v_scale[pid, kvh]) * dec[f.v_pages[pid, 0, kvh].numpy()]
        k = float(f.k_scale[pid, kvh]) * dec[f.k_pages[pid, 0, kvh].numpy()]
        assert np.array_equal(out[0, h], v)
        s = float(np.float32(f.softmax_scale)) * float(f.q[0, h].double().numpy() @ k)
        assert abs(lse[0, h] - s) <= 1e-12 * max(1.0, abs(s))


def test_f4_scale_linearity(oracle):
    import dataclasses
    f = W.quantize_batch_fp8(W.make_batch([200, 31], 8, 2, 64, 16, seed=414))
    out, lse = _run8(oracle, f)
    out4, lse4 = _run8(oracle, dataclasses.replace(f, v_scale=f.v_scale * 4))
    assert np.array_equal(out4, out * 4) and np.array_equal(lse4, lse)
    outk, lsek = _run8(oracle, dataclasses.replace(f, k_scale=f.k_scale * 2))
    outs, lses = _run8(oracle, dataclasses.replace(f, softmax_scale=f.softmax_scale * 2))
    assert np.array_equal(outk, outs) and np.array_equal(lsek, lses)
    assert not np.array_equal(outk, out)


def test_f5_poison_independence(oracle):
    lens = [100, 33, 0, 17]
    clean = W.quantize_batch_fp8(W.make_batch(lens, 8, 2, 64, 16, seed=415, num_pages=32))
    dirty = W.quantize_batch_fp8(W.make_batch(lens, 8, 2, 64, 16, seed=415, num_pages=32, poison_unused=True))
    assert (dirty.k_pages == 0x7f).any() and torch.isnan(dirty.k_scale).any()   # poison survived the quantiser
    a, la = _run8(oracle, clean)
    b, lb = _run8(oracle, dirty)
    assert np.isfinite(b[[0, 1, 3]]).all()
    # the live part of a last page has the same amax either way only if its live rows hold the block's
    # maximum; compare instead against a clean cache re-quantised from the poisoned one's live values
    import dataclasses
    fixed = dataclasses.replace(dirty,
                                k_pages=torch.where(dirty.k_pages == 0x7f, torch.zeros_like(dirty.k_pages), dirty.k_pages),
                                v_pages=torch.where(dirty.v_pages == 0x7f, torch.zeros_like(dirty.v_pages), dirty.v_pages),
                                k_scale=torch.nan_to_num(dirty.k_scale, nan=1.0), v_scale=torch.nan_to_num(dirty.v_scale, nan=1.0),
                                block_table=dirty.block_table.clamp_min(0))
    c, lc = _run8(oracle, fixed)
    assert np.array_equal(b, c) and np.array_equal(lb, lc)
    assert np.array_equal(b[2], np.zeros_like(b[2])) and np.isneginf(lb[2]).all()   # L = 0 (reading R9)
    assert np.allclose(a, b, atol=0.2)  # same underlying data, slightly different scales in last pages


@pytest.mark.parametrize("ps,window,sinks", [(16, 0, 0), (32, 0, 0), (16, 40, 3)])
def test_f6_brute_force_dense(oracle, ps, window, sinks):
    lens = [130, 47]
    f = W.quantize_batch_fp8(W.make_batch(lens, 8, 2, 64, ps, seed=416 + ps))
    out, lse = _run8(oracle, f, window, sinks)
    g = 4
    for b, L in enumerate(lens):
        n = W.pages_needed(L, ps)
        ids = f.block_table[b, :n].long()
        k = f.k_pages[ids].view(torch.float8_e4m3fn).float().double() * f.k_scale[ids].double().view(n, 1, 2, 1)
        v = f.v_pages[ids].view(torch.float8_e4m3fn).float().double() * f.v_scale[ids].double().view(n, 1, 2, 1)
        k = k.reshape(n * ps, 2, 64)[:L].numpy()
        v = v.reshape(n * ps, 2, 64)[:L].numpy()
        lo = 0 if (window <= 0 or window >= L) else L - window
        keep = np.array([t < sinks or t >= lo for t in range(L)])
        for h in range(8):
            s = float(np.float32(f.softmax_scale)) * (k[:, h // g, :] @ f.q[b, h].double().numpy())
            s = np.where(keep, s, -np.inf)
            w = np.exp(s - s.max())
            want = (w[:, None] * v[:, h // g, :]).sum(0) / w.sum()
            assert np.max(np.abs(out[b, h] - want)) <= 1e-13
            assert abs(lse[b, h] - (s.max() + np.log(w.sum()))) <= 1e-12


def test_f7_hnd_layout_is_a_relayout(oracle):
    f = W.quantize_batch_fp8(W.make_batch([130, 47, 0, 16], 8, 2, 64, 32, seed=417))
    h = W.to_hnd(f)
    assert h.k_pages.shape == (f.num_pages, 2, 32, 64) and h.num_kv_heads == 2 and h.page_size == 32
    for window, sinks in ((0, 0), (40, 3)):
        a, la = _run8(oracle, f, window, sinks)
        b, lb = oracle.decode_attn_fp8(h.q, h.k_pages, h.v_pages, h.k_scale, h.v_scale, h.block_table, h.seq_lens,
                                       h.softmax_scale, window, sinks, kv_layout="HND")
        assert np.array_equal(a, b) and np.array_equal(la, lb)
    # and it is not a no-op: reading the transposed pools as NHD gives something else
    c, _ = oracle.decode_attn_fp8(h.q, h.k_pages.view(f.k_pages.shape), h.v_pages.view(f.v_pages.shape), h.k_scale,
                                  h.v_scale, h.block_table, h.seq_lens, h.softmax_scale)
    assert not np.array_equal(a, c)


# ---- the E4M3 encoder and the quantising append (oracle.e4m3_encode, oracle.kv_append_fp8) -------------------
#   E1  decode(encode(v)) == v for every finite code, signs of zero kept
#   E2  torch's float8_e4m3fn cast (round-to-nearest-even) on random floats, on every midpoint between adjacent
#       codes (the ties) and on their fp32 neighbours
#   E3  saturation: everything above 448 (and inf) -> 0x7e / 0xfe; NaN -> a NaN code
#   E4  hand-computed ties: 1.0625 -> 1.0 (0x38), 1.1875 -> 1.25 (0x3a), 2^-10 -> 0, 3 * 2^-10 -> 2 * 2^-9 (0x02)
#   A1  append: the row lands at (page of position L, slot L % ps), nothing else in the pools changes, L += 1;
#       a full page moves on to the next table entry; HND == NHD transposed
def test_e1_encode_inverts_decode(oracle):
    for b in range(256):
        if b & 0x7f == 0x7f:
            continue
        assert oracle.e4m3_encode(oracle.e4m3_decode(b)) == b, hex(b)


def test_e2_encode_matches_torch_cast(oracle):
    dec = np.array([oracle.e4m3_decode(b) for b in range(0x7f)])            # positive codes, ascending
    mids = (dec[:-1] + dec[1:]) / 2                                         # exact in fp32: few significant bits
    pts = np.concatenate([mids, np.nextafter(mids.astype(np.float32), np.float32(1e9)),
                          np.nextafter(mids.astype(np.float32), np.float32(-1e9)), dec])
    rng = np.random.default_rng(7)
    pts = np.concatenate([pts, rng.uniform(0, 448, 20000), rng.uniform(0, 0.05, 20000), 2.0 ** rng.uniform(-12, 8.8, 20000)])
    pts = np.concatenate([pts, -pts]).astype(np.float32)
    pts = pts[np.abs(pts) <= 448]
    want = torch.from_numpy(pts).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = np.array([oracle.e4m3_encode(float(x)) for x in pts], dtype=np.uint8)
    assert np.array_equal(got, want)


def test_e3_saturation_and_nan(oracle):
    for x in (448.0001, 449.0, 464.0, 480.0, 1e9, float("inf")):
        assert oracle.e4m3_encode(x) == 0x7e and oracle.e4m3_encode(-x) == 0xfe
    assert oracle.e4m3_encode(float("nan")) & 0x7f == 0x7f


def test_e4_ties_to_even_by_hand(oracle):
    assert oracle.e4m3_encode(1.0625) == 0x38 and oracle.e4m3_encode(1.1875) == 0x3a
    assert oracle.e4m3_encode(2.0 ** -10) == 0x00 and oracle.e4m3_encode(3 * 2.0 ** -10) == 0x02
    assert oracle.e4m3_encode(-2.0 ** -10) == 0x80
    assert oracle.e4m3_encode(15 * 2.0 ** -10) == 0x08                       # 7.5 steps -> 8 steps = min normal


@pytest.mark.parametrize("layout", ["NHD", "HND"])
def test_a1_append_fp8_places_and_quantises(oracle, layout):
    ps, hkv, d = 16, 2, 64
    b = W.make_batch([15, 16, 0, 40], 4, hkv, d, ps, seed=431, spare_tokens=3)
    f = W.quantize_batch_fp8(b)
    f.k_scale.nan_to_num_(nan=0.01)
    f.v_scale.nan_to_num_(nan=0.02)
    f = f if layout == "NHD" else W.to_hnd(f)
    k8, v8 = f.k_pages.numpy().copy(), f.v_pages.numpy().copy()
    lens = f.seq_lens.numpy().astype(np.int32).copy()
    g = torch.Generator().manual_seed(3)
    nk = (torch.randn((4, hkv, d), generator=g) * 2).to(torch.bfloat16)
    nv = (torch.randn((4, hkv, d), generator=g) * 2).to(torch.bfloat16)
    nk[0, 0, 0], nk[0, 0, 1], nv[1, 1, 5] = 1e6, -1e6, 0.0                    # saturation both ways, a zero
    k0, v0, l0 = k8.copy(), v8.copy(), lens.copy()
    oracle.kv_append_fp8(k8, v8, f.k_scale, f.v_scale, f.block_table, lens, nk, nv, kv_layout=layout)
    assert np.array_equal(lens, l0 + 1)
    touched = np.zeros(k8.shape, bool)
    for s in range(4):
        L = int(l0[s])
        pid, slot = int(f.block_table[s, L // ps]), L % ps
        for h in range(hkv):
            idx = (pid, h, slot) if layout == "HND" else (pid, slot, h)
            touched[idx] = True
            for arr, new, sc in ((k8, nk, f.k_scale), (v8, nv, f.v_scale)):
                q = (new[s, h].float() / sc[pid, h]).clamp(-448, 448)          # fp32 quotient, saturated
                want = q.to(torch.float8_e4m3fn).view(torch.uint8).numpy()     # torch's RNE cast
                assert np.array_equal(arr[idx], want), (s, h)
    assert np.array_equal(k8[~touched], k0[~touched]) and np.array_equal(v8[~touched], v0[~touched])
    assert k8[(int(f.block_table[0, 0]), 0, 15) if layout == "HND" else (int(f.block_table[0, 0]), 15, 0)][0] == 0x7e
    assert int(f.block_table[1, 1]) != int(f.block_table[1, 0])               # sequence 1 (L = 16) opened its second page
