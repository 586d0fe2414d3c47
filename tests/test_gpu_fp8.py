"""GPU parity of the FP8 (E4M3 + per-page, per-kv-head scale) KV-cache variant
(comem_decode_attn_fp8_async, reading R18) against oracle.decode_attn_fp8 on the same bytes,
the properties that fix bits, and a sampled check at config 4's full size."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import MAX_ABS, MEAN_ABS, REL_L2

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t):
    return t.contiguous().view(torch.int16)


def run8(f, window=0, sinks=0, ws=None):
    out = torch.full_like(f.q, float("nan"))
    lse = torch.full((f.batch, f.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
    ws = ws if ws is not None else comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
    comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                      f.softmax_scale, out, ws, window, sinks, lse_out=lse, kv_layout=f.kv_layout)
    torch.cuda.synchronize()
    return out, lse


def gate(g, ref, gl, ref_lse, what):
    d = np.abs(g - ref)
    assert np.isfinite(g).all(), what
    assert d.max() <= MAX_ABS and d.mean() <= MEAN_ABS, (what, d.max(), d.mean())
    rel = np.linalg.norm(g - ref) / max(np.linalg.norm(ref), 1e-300)
    assert rel <= REL_L2, (what, rel)
    assert d.max() <= 4 * 2.0 ** -9 * np.abs(ref).max() + 1e-6, (what, d.max(), np.abs(ref).max())
    live = np.isfinite(ref_lse)
    assert np.array_equal(np.isneginf(gl), np.isneginf(ref_lse)), what
    if live.any():
        assert np.max(np.abs(gl[live] - ref_lse[live]) / np.maximum(1.0, np.abs(ref_lse[live]))) <= 2e-4, what
    return {"max_abs": float(d.max()), "mean_abs": float(d.mean()), "rel_l2": float(rel)}


def check(oracle, f, what, window=0, sinks=0):
    out, lse = run8(f, window, sinks)
    c = f.to("cpu")
    ref, ref_lse = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table,
                                          c.seq_lens, c.softmax_scale, window, sinks, kv_layout=c.kv_layout)
    gate(out.double().cpu().numpy(), ref, lse.double().cpu().numpy(), ref_lse, what)
    return out, lse


def fp8_batch(lens, hq, hkv, ps, seed, **kw):
    return W.quantize_batch_fp8(W.make_batch(lens, hq, hkv, 128, ps, seed=seed, device=DEV, poison_unused=True, **kw))


@pytest.mark.parametrize("G,ps", [(1, 16), (4, 32), (8, 16), (3, 32), (5, 16), (8, 32)])
def test_fp8_small_ragged(oracle, G, ps):
    lens = [1, 15, 16, 17, 31, 33, 127, 128, 129, 512, 1000, 0, 2049]
    f = fp8_batch(lens, 2 * G, 2, ps, seed=500 + G + ps)
    check(oracle, f, f"G{G} ps{ps}")


def test_fp8_long_ragged_grids_and_permutation(oracle):
    lens = [20000, 37, 0, 50001, 8191, 16, 300]
    f = fp8_batch(lens, 64, 8, 16, seed=521)
    base, base_lse = check(oracle, f, "ragged default grid")
    again, again_lse = run8(f)
    assert torch.equal(bits(base), bits(again)) and torch.equal(base_lse, again_lse)       # run to run
    g = W.permute_pages_fp8(f, seed=9)
    assert not torch.equal(g.block_table, f.block_table)
    po, pl = run8(g)
    assert torch.equal(bits(base), bits(po)) and torch.equal(base_lse, pl)                # page placement
    try:
        for grid in (1, 7, 148, 296):
            comem.comem_set_grid_ctas(grid)
            check(oracle, f, f"ragged grid {grid}")
    finally:
        comem.comem_set_grid_ctas(0)


@pytest.mark.parametrize("nats,v_mean", [(12.0, 0.3), (13.0, 0.3), (14.0, 0.15), (13.0, 0.05)])
def test_fp8_sink_token_small_v_scale(oracle, nats, v_mean):
    """One sink token 12-14 nats above a flat 32K tail, V with a nonzero mean, page scales amax/448 <= 2e-3: the
    tail's p * v_scale would fall into the fp16 subnormals (below 2^-14) and drop out of the numerator while the
    normaliser still counts it.  The kernel keeps only the scale's mantissa (times a power of two relative to the
    running largest exponent) on p and the power of two on the accumulator."""
    f = W.quantize_batch_fp8(W.sink_batch(32768, 32, 8, 128, 16, seed=530, device=DEV, sink_nats=nats, v_mean=v_mean,
                                          v_std=v_mean / 3))
    assert float(f.v_scale[f.block_table[0, :2048].long()].max()) <= 2e-3
    check(oracle, f, f"sink {nats} nats, v mean {v_mean}")
    check(oracle, W.to_hnd(f), f"sink {nats} nats, v mean {v_mean}, HND")


def test_fp8_mixed_page_scales(oracle):
    """Page scales spread over 2^-12 .. 2^6 within one sequence (the running reference exponent moves up and down)."""
    b = W.make_batch([3000, 777], 32, 8, 128, 16, seed=531, device=DEV, poison_unused=True)
    gen = torch.Generator(device=DEV)
    gen.manual_seed(5)
    expo = torch.randint(-12, 7, (b.v_pages.shape[0], 1, 8, 1), generator=gen, device=DEV).float()
    b.v_pages.copy_((b.v_pages.float() * torch.exp2(expo)).to(torch.bfloat16))
    f = W.quantize_batch_fp8(b)
    check(oracle, f, "mixed page scales")


def test_fp8_single_long_sequence_aligned_schedule(oracle):
    """one 32K sequence x 8 kv heads: the segment-aligned schedule (18-19 CTAs per head) and the fused merge"""
    f = fp8_batch([32768], 64, 8, 16, seed=522, k_scale=0.5)
    check(oracle, f, "c2-shaped fp8")


def test_fp8_window_and_sinks(oracle):
    f = fp8_batch([5000, 100, 0, 777, 16, 2048], 32, 8, 32, seed=523)
    for window, sinks in ((1, 0), (17, 1), (128, 16), (1000, 64), (4096, 4), (10 ** 6, 3)):
        check(oracle, f, f"fp8 w{window} s{sinks}", window, sinks)
    full, full_lse = run8(f)
    w_all, l_all = run8(f, 10 ** 6, 3)
    assert torch.equal(bits(full), bits(w_all)) and torch.equal(full_lse, l_all)


def test_fp8_all_byte_codes_exact(oracle):
    """L = 1, unit scales: out = bf16(e4m3(V byte)) exactly (3 mantissa bits fit bf16; the softmax weight
    is exactly 1) for every finite byte code -- checks the device conversion of all 254 of them, and the
    K conversion through lse = scale * q . k."""
    f = fp8_batch([1, 1], 8, 1, 16, seed=524)
    codes = torch.arange(256, dtype=torch.uint8, device=DEV)
    codes = torch.where((codes & 0x7f) == 0x7f, torch.zeros_like(codes), codes)      # NaN codes -> 0
    for b in range(2):
        pid = int(f.block_table[b, 0])
        f.v_pages[pid, 0, 0] = codes[128 * b:128 * (b + 1)]
        f.k_pages[pid, 0, 0] = codes[128 * b:128 * (b + 1)].flip(0)
        f.k_scale[pid, 0] = 1.0
        f.v_scale[pid, 0] = 1.0
    # q small enough that q . k stays well inside fp32 and the oracle comparison is tight
    f = dataclasses.replace(f, q=(f.q.float() / 64).to(torch.bfloat16))
    out, lse = run8(f)
    want = codes.view(torch.float8_e4m3fn).float()
    for b in range(2):
        for h in range(8):
            assert torch.equal(out[b, h].float(), want[128 * b:128 * (b + 1)]), (b, h)
    c = f.to("cpu")
    ref, ref_lse = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table,
                                          c.seq_lens, c.softmax_scale)
    assert np.array_equal(out.double().cpu().numpy(), ref)
    assert np.max(np.abs(lse.double().cpu().numpy() - ref_lse) / np.maximum(1.0, np.abs(ref_lse))) <= 1e-5


def test_fp8_scale_moves_between_page_and_bytes(oracle):
    """Doubling a page's v_scale doubles its contribution; per-page scales that differ wildly page to page."""
    f = fp8_batch([700, 90], 16, 4, 16, seed=525)
    g = torch.Generator().manual_seed(5)
    e = torch.randint(-4, 5, tuple(f.k_scale.shape), generator=g).float().to(DEV)
    f2 = dataclasses.replace(f, v_scale=torch.nan_to_num(f.v_scale, nan=1.0) * torch.exp2(e),
                             k_scale=torch.nan_to_num(f.k_scale, nan=1.0) * torch.exp2(-e.abs() / 2))
    check(oracle, f2, "wild page scales")


@pytest.mark.parametrize("G,ps", [(4, 32), (8, 16), (3, 16)])
def test_fp8_hnd_layout(oracle, G, ps):
    """[P, Hkv, page_size, D] pools: parity vs the oracle's HND reading, and bit-identical to the NHD call (the
    arithmetic and its order do not depend on where a tile sits in DRAM)."""
    lens = [1, 17, 33, 128, 1000, 0, 2049, 20000]
    f = fp8_batch(lens, 2 * G, 2, ps, seed=540 + G + ps)
    h = W.to_hnd(f)
    a, la = run8(f)
    b, lb = check(oracle, h, f"hnd G{G} ps{ps}")
    assert torch.equal(bits(a), bits(b)) and torch.equal(la, lb)
    for window, sinks in ((100, 4), (4096, 0)):
        a, la = run8(f, window, sinks)
        b, lb = check(oracle, h, f"hnd G{G} ps{ps} w{window}", window, sinks)
        assert torch.equal(bits(a), bits(b)) and torch.equal(la, lb)


@pytest.mark.parametrize("G,hkv,ps", [(4, 1, 16), (8, 2, 32), (1, 3, 16), (6, 2, 16)])
def test_fp8_head_dim_64(oracle, G, hkv, ps):
    """head_dim 64 (64-byte rows, unswizzled tiles, 64-stage ring): config 1's geometry among them; NHD and HND,
    window + sinks, grids, page permutation."""
    lens = [512, 1, 15, 16, 17, 33, 255, 1000, 0, 2049, 7000]
    f = W.quantize_batch_fp8(W.make_batch(lens, G * hkv, hkv, 64, ps, seed=580 + G + ps, device=DEV, poison_unused=True))
    base, base_lse = check(oracle, f, f"D64 G{G} hkv{hkv} ps{ps}")
    h = W.to_hnd(f)
    ho, hl = check(oracle, h, f"D64 hnd G{G} hkv{hkv} ps{ps}")
    assert torch.equal(bits(base), bits(ho)) and torch.equal(base_lse, hl)
    check(oracle, f, "D64 window", 300, 5)
    po, pl = run8(W.permute_pages_fp8(f, seed=3))
    assert torch.equal(bits(base), bits(po)) and torch.equal(base_lse, pl)
    try:
        for grid in (1, 5, 296):
            comem.comem_set_grid_ctas(grid)
            check(oracle, f, f"D64 grid {grid}")
    finally:
        comem.comem_set_grid_ctas(0)


def test_fp8_config1_tiny(oracle):
    """BASELINE.json configs[0] (batch 1, 4q/1kv, D 64, 512 tokens, 32 permuted pages) with its cache quantised."""
    f = W.quantize_batch_fp8(W.config1_tiny(DEV, poison_unused=True))
    check(oracle, f, "C1 fp8")


def test_fp8_all_byte_codes_exact_head_dim_64(oracle):
    f = W.quantize_batch_fp8(W.make_batch([1, 1, 1, 1], 8, 1, 64, 16, seed=526, device=DEV, poison_unused=True))
    codes = torch.arange(256, dtype=torch.uint8, device=DEV)
    codes = torch.where((codes & 0x7f) == 0x7f, torch.zeros_like(codes), codes)
    for b in range(4):
        pid = int(f.block_table[b, 0])
        f.v_pages[pid, 0, 0] = codes[64 * b:64 * (b + 1)]
        f.k_pages[pid, 0, 0] = codes[64 * b:64 * (b + 1)].flip(0)
        f.k_scale[pid, 0] = 1.0
        f.v_scale[pid, 0] = 1.0
    f = dataclasses.replace(f, q=(f.q.float() / 64).to(torch.bfloat16))
    out, lse = run8(f)
    want = codes.view(torch.float8_e4m3fn).float()
    for b in range(4):
        for h in range(8):
            assert torch.equal(out[b, h].float(), want[64 * b:64 * (b + 1)]), (b, h)
    c = f.to("cpu")
    ref, ref_lse = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table,
                                          c.seq_lens, c.softmax_scale)
    assert np.max(np.abs(lse.double().cpu().numpy() - ref_lse) / np.maximum(1.0, np.abs(ref_lse))) <= 1e-5


def test_fp8_rejects_unknown_layout_and_null_scales():
    b = W.make_batch([100], 8, 2, 128, 16, seed=1, device=DEV)
    k8 = torch.zeros(b.k_pages.shape, dtype=torch.uint8, device=DEV)
    sc = torch.ones((b.num_pages, 2), dtype=torch.float32, device=DEV)
    out = torch.empty_like(b.q)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    lib = comem.load_library()
    import ctypes
    p = lambda t: ctypes.c_void_p(t.data_ptr())
    args = lambda ks, layout: (p(b.q), p(k8), p(k8), ks, p(sc), p(b.block_table), p(b.seq_lens), 8, 2, 128, 16,
                               ctypes.c_float(0.1), p(out), 1, b.block_table.shape[1], b.num_pages, None, p(ws),
                               ws.numel(), None, 0, 0, layout, None)
    assert lib.comem_decode_attn_fp8_async(*args(None, 0)) == comem.COMEM_ERR_INVALID_ARG
    assert lib.comem_decode_attn_fp8_async(*args(p(sc), 5)) == comem.COMEM_ERR_INVALID_ARG
    assert lib.comem_decode_attn_fp8_async(*args(p(sc), 0)) == comem.COMEM_OK
    torch.cuda.synchronize()


def test_fp8_config4_full_size_sampled(oracle):
    """Config 4's shape (16 x 131072 tokens, 32q/8kv, page 32, peaked keys) with the cache quantised: oracle on
    two whole sequences (all 32 heads) from the same bytes; permutation bit-identity on the complete output."""
    bf = W.config4_memory_long(DEV, poison_unused=True)
    f = W.quantize_batch_fp8(bf)
    del bf
    torch.cuda.empty_cache()
    out, lse = run8(f)
    ps = f.page_size
    for b in (0, 11):
        n = W.pages_needed(int(f.seq_lens[b]), ps)
        ids = f.block_table[b, :n].long()
        sub = W.Fp8DecodeBatch(q=f.q[b:b + 1].cpu(), k_pages=f.k_pages[ids].cpu(), v_pages=f.v_pages[ids].cpu(),
                               k_scale=f.k_scale[ids].cpu(), v_scale=f.v_scale[ids].cpu(),
                               block_table=torch.arange(n, dtype=torch.int32).view(1, n),
                               seq_lens=f.seq_lens[b:b + 1].cpu(), softmax_scale=f.softmax_scale)
        ref, ref_lse = oracle.decode_attn_fp8(sub.q, sub.k_pages, sub.v_pages, sub.k_scale, sub.v_scale,
                                              sub.block_table, sub.seq_lens, sub.softmax_scale)
        err = gate(out[b:b + 1].double().cpu().numpy(), ref, lse[b:b + 1].double().cpu().numpy(), ref_lse, f"c4 fp8 seq {b}")
        print("c4 fp8 seq", b, err)
    g = W.permute_pages_fp8(f, seed=77)
    po, pl = run8(g)
    assert torch.equal(bits(out), bits(po)) and torch.equal(lse, pl)


@pytest.mark.parametrize("case", range(16))
def test_fp8_randomised_shapes(oracle, case):
    """Seeded random draws over what the FP8 entry point accepts: batch, kv heads, group 1..8, page size, pool
    layout, ragged lengths with zeros and tile / page-boundary values, window + sinks, and the persistent grid
    size (linear and segment-aligned schedules, whole and cut segments, one- and multi-round merges); each case
    also under a page permutation (bit-identical)."""
    rng = np.random.default_rng(9500 + case)
    G = int(rng.integers(1, 9))
    hkv = int(rng.integers(1, 9))
    ps = int(rng.choice([16, 32]))
    batch = int(rng.integers(1, 11))
    special = [0, 1, 15, 16, 17, ps - 1, ps, ps + 1, 255, 256, 257]
    lens = [int(rng.choice(special)) if rng.random() < 0.3 else int(rng.integers(1, 6000)) for _ in range(batch)]
    if case % 5 == 0:
        lens[0] = int(rng.integers(20000, 60000))
    grid = int(rng.choice([0, 0, 3, 17, 61, 148, 211, 600]))
    window, sinks = (0, 0) if rng.random() < 0.6 else (int(rng.integers(1, 3000)), int(rng.integers(0, 70)))
    pool = max(1, sum(W.pages_needed(l, ps) for l in lens)) + int(rng.integers(0, 9))
    f = fp8_batch(lens, G * hkv, hkv, ps, seed=9600 + case, num_pages=pool)
    if rng.random() < 0.5:
        f = W.to_hnd(f)
    what = f"case {case}: G{G} hkv{hkv} ps{ps} {f.kv_layout} lens{lens} grid{grid} w{window} s{sinks}"
    try:
        comem.comem_set_grid_ctas(grid)
        out, lse = check(oracle, f, what, window, sinks)
        out2, lse2 = run8(W.permute_pages_fp8(f, seed=case), window, sinks)
        assert torch.equal(bits(out), bits(out2)), what
        assert torch.equal(lse.nan_to_num(neginf=-1e30), lse2.nan_to_num(neginf=-1e30)), what
    finally:
        comem.comem_set_grid_ctas(0)


@pytest.mark.parametrize("layout,ps", [("NHD", 16), ("HND", 32)])
def test_fp8_append_then_attend_loop(oracle, layout, ps):
    """40 decode steps on the FP8 cache: comem_kv_append_fp8_async then attention.  The appended BYTES and
    seq_lens must equal the oracle's (byte work: bit-exact; both sides take the fp32 quotient and round it to
    E4M3 nearest-even, saturating), including rows that saturate, tiny quotients (subnormal codes), zeros and
    page crossings; the attention output after each of several steps matches the FP8 attention oracle on the
    oracle-appended cache."""
    hq, hkv = 16, 4
    lens = [ps - 3, 5000, 0, 2 * ps - 1, 777]
    b = W.make_batch(lens, hq, hkv, 128, ps, seed=561, device=DEV, spare_tokens=48)
    f = W.quantize_batch_fp8(b)
    # pages that will be opened by the appends hold nothing yet: give them the scales a serving engine would
    f.k_scale.copy_(torch.where(torch.isnan(f.k_scale) | (f.k_scale == 1.0), torch.full_like(f.k_scale, 0.011), f.k_scale))
    f.v_scale.copy_(torch.where(torch.isnan(f.v_scale) | (f.v_scale == 1.0), torch.full_like(f.v_scale, 0.009), f.v_scale))
    if layout == "HND":
        f = W.to_hnd(f)
    f = dataclasses.replace(f, seq_lens=f.seq_lens.clone())
    ok8, ov8 = f.k_pages.cpu().numpy().copy(), f.v_pages.cpu().numpy().copy()
    olens = f.seq_lens.cpu().numpy().astype(np.int32).copy()
    ks_c, vs_c, bt_c = f.k_scale.cpu(), f.v_scale.cpu(), f.block_table.cpu()
    ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=layout)
    for step in range(40):
        q, nk, nv = W.decode_step_rows(b, step, seed_base=7000)
        if step % 7 == 0:
            nk[0, 0, :4] = torch.tensor([1e4, -1e4, 0.0, 1e-5], dtype=torch.bfloat16, device=DEV)   # saturate, zero, subnormal code
            nv[1, 1, :2] = torch.tensor([-0.0, 3e-6], dtype=torch.bfloat16, device=DEV)
        comem.comem_kv_append_fp8_async(f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens, nk, nv,
                                        kv_layout=layout)
        oracle.kv_append_fp8(ok8, ov8, ks_c, vs_c, bt_c, olens, nk.cpu(), nv.cpu(), kv_layout=layout)
        fq = dataclasses.replace(f, q=q)
        if step in (0, 1, 2, 3, ps - 1, ps, 39):
            torch.cuda.synchronize()
            assert np.array_equal(f.seq_lens.cpu().numpy(), olens), step
            assert np.array_equal(f.k_pages.cpu().numpy(), ok8) and np.array_equal(f.v_pages.cpu().numpy(), ov8), step
            out, lse = run8(fq, ws=ws)
            ref, ref_lse = oracle.decode_attn_fp8(q.cpu(), ok8, ov8, ks_c, vs_c, bt_c, olens, f.softmax_scale, kv_layout=layout)
            gate(out.double().cpu().numpy(), ref, lse.double().cpu().numpy(), ref_lse, f"{layout} step {step}")
    assert (ok8 == 0x7e).any() and (ok8 == 0xfe).any()          # the saturating rows did saturate


def test_fp8_two_streams_overlap_equals_serial():
    """Config-5 style on the FP8 cache: an agent batch (64q/8kv, NHD) and a memory-model batch (32q/8kv, HND) each
    run 16 append + attend steps, once serially and once overlapped on two streams with their own workspaces:
    every step's output is bit-identical (no CTA ever waits for another; nothing depends on arrival order)."""
    def mk(hq, lens, seed, layout):
        b = W.make_batch(lens, hq, 8, 128, 16, seed=seed, device=DEV, spare_tokens=16)
        f = W.quantize_batch_fp8(b)
        for sc in (f.k_scale, f.v_scale):
            sc.copy_(torch.where(torch.isnan(sc) | (sc == 1.0), torch.full_like(sc, 0.01), sc))
        f = W.to_hnd(f) if layout == "HND" else f
        rows = [W.decode_step_rows(b, s, seed_base=seed * 10) for s in range(16)]
        return f, rows

    specs = [(64, [9000, 30000, 17, 12000, 4097, 20000], 571, "NHD"), (32, [40000, 65000, 33000], 572, "HND")]

    def run(overlap):
        outs = []
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        state = []
        for (hq, lens, seed, layout), st in zip(specs, streams):
            f, rows = mk(hq, lens, seed, layout)
            f = dataclasses.replace(f, seq_lens=f.seq_lens.clone(), k_pages=f.k_pages.clone(), v_pages=f.v_pages.clone())
            ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, stream=st, kv_layout=layout)
            state.append((f, rows, ws, st, [torch.full_like(f.q, float("nan")) for _ in range(16)]))  # unwritten rows fail
        torch.cuda.synchronize()
        for step in range(16):
            for f, rows, ws, st, o in state:
                q, nk, nv = rows[step]
                comem.comem_kv_append_fp8_async(f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                                nk, nv, stream=st, kv_layout=f.kv_layout)
                comem.comem_decode_attn_fp8_async(q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table,
                                                  f.seq_lens, f.softmax_scale, o[step], ws, stream=st,
                                                  kv_layout=f.kv_layout)
                if not overlap:
                    torch.cuda.synchronize()
        torch.cuda.synchronize()
        return [[bits(x).clone() for x in s[4]] for s in state]

    serial, both = run(False), run(True)
    for which, (a, b) in enumerate(zip(serial, both)):
        for step, (x, y) in enumerate(zip(a, b)):
            xf = x.view(torch.bfloat16).float()
            assert torch.isfinite(xf).all() and float(xf.abs().max()) < 16.0, (which, step, float(xf.abs().max()))
            assert torch.equal(x, y), (which, step)


@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pinned", [True, False])
def test_fp8_decode_step_host_equals_device_calls(oracle, layout, pinned):
    """comem_decode_step_host_fp8 (host rows in, quantising append, FP8 attention, host out back) against the same
    step made of comem_kv_append_fp8_async + comem_decode_attn_fp8_async on a twin cache: bytes, lengths and outputs
    bit-identical, on the pinned (zero-copy) and the pageable (copy-engine) path; last step checked against the oracle."""
    ps = 16
    b = W.make_batch([ps - 2, 3000, 0, 129], 16, 4, 128, ps, seed=571, device=DEV, spare_tokens=24)
    f = W.quantize_batch_fp8(b)
    f.k_scale.copy_(torch.where(torch.isnan(f.k_scale) | (f.k_scale == 1.0), torch.full_like(f.k_scale, 0.011), f.k_scale))
    f.v_scale.copy_(torch.where(torch.isnan(f.v_scale) | (f.v_scale == 1.0), torch.full_like(f.v_scale, 0.009), f.v_scale))
    if layout == "HND":
        f = W.to_hnd(f)
    twin = dataclasses.replace(f, k_pages=f.k_pages.clone(), v_pages=f.v_pages.clone(), seq_lens=f.seq_lens.clone())
    f = dataclasses.replace(f, seq_lens=f.seq_lens.clone())
    ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=layout)
    ws2 = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=layout)
    pin = (lambda t: t.cpu().pin_memory()) if pinned else (lambda t: t.cpu())
    out_h = pin(torch.zeros_like(f.q))
    lse_h = pin(torch.zeros((f.q.shape[0], f.q.shape[1]), dtype=torch.float32))
    for step in range(20):
        q, nk, nv = W.decode_step_rows(b, step, seed_base=7100)
        comem.comem_decode_step_host_fp8(pin(q), pin(nk), pin(nv), f.k_pages, f.v_pages, f.k_scale, f.v_scale,
                                         f.block_table, f.seq_lens, f.softmax_scale, out_h, ws, lse_host=lse_h,
                                         kv_layout=layout)
        comem.comem_kv_append_fp8_async(twin.k_pages, twin.v_pages, twin.k_scale, twin.v_scale, twin.block_table,
                                        twin.seq_lens, nk, nv, kv_layout=layout)
        out, lse = run8(dataclasses.replace(twin, q=q), ws=ws2)
        torch.cuda.synchronize()
        assert torch.equal(out_h.view(torch.int16), out.cpu().view(torch.int16)), step
        assert torch.equal(lse_h.view(torch.int32), lse.cpu().view(torch.int32)), step
        assert torch.equal(f.seq_lens, twin.seq_lens) and torch.equal(f.k_pages, twin.k_pages) and torch.equal(f.v_pages, twin.v_pages)
    ref, ref_lse = oracle.decode_attn_fp8(q.cpu(), f.k_pages.cpu(), f.v_pages.cpu(), f.k_scale.cpu(), f.v_scale.cpu(),
                                          f.block_table.cpu(), f.seq_lens.cpu(), f.softmax_scale, kv_layout=layout)
    gate(out_h.double().numpy(), ref, lse_h.double().numpy(), ref_lse, f"host step {layout}")
