"""GPU parity: the CUDA path (through the C-ABI) against the fp64 oracle, element by element, on
the same seeded inputs; plus the properties that must hold bit-exactly."""
import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import (all_pairs, assert_parity, check_batch, errors, gpu_run, oracle_rows)

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t: torch.Tensor) -> torch.Tensor:
    return t.contiguous().view(torch.int16)


# ---- small shapes: every G / D / page_size, lengths straddling tile, page and CTA boundaries ------
@pytest.mark.parametrize("G", [1, 2, 4, 8])
@pytest.mark.parametrize("D", [64, 128])
@pytest.mark.parametrize("ps", [16, 32])
def test_small_grid(oracle, G, D, ps):
    lens = [1, 15, 16, 17, 31, 32, 33, 127, 128, 129, 512, 1000, 0, 2049]
    b = W.make_batch(lens, 2 * G, 2, D, ps, seed=100 + G + D + ps, device=DEV, poison_unused=True)
    check_batch(oracle, b, what=f"G{G} D{D} ps{ps}")


@pytest.mark.parametrize("G", [3, 5, 6, 7])
def test_odd_group_sizes(oracle, G):
    """Any group size up to 8 is packed into the 8-wide MMA dimension (e.g. 40q/8kv models: G = 5)."""
    b = W.make_batch([9000, 33, 0, 2500, 17], G * 2, 2, 128, 16, seed=90 + G, device=DEV, poison_unused=True)
    check_batch(oracle, b, what=f"G{G}")
    b = W.make_batch([700, 64], G * 3, 3, 64, 32, seed=95 + G, device=DEV, poison_unused=True)
    check_batch(oracle, b, what=f"G{G} D64 ps32")


@pytest.mark.parametrize("hkv", [1, 3, 8])
def test_kv_head_counts(oracle, hkv):
    b = W.make_batch([700, 33, 4097], 4 * hkv, hkv, 128, 16, seed=7 + hkv, device=DEV, poison_unused=True)
    check_batch(oracle, b, what=f"hkv{hkv}")


def test_config1_tiny(oracle):
    b = W.config1_tiny(DEV, poison_unused=True)
    _, _, err = check_batch(oracle, b, what="C1")
    print("C1", err)


def test_ragged_many_ctas(oracle):
    # long enough that segments are cut by CTA-range boundaries (partials + combine) and short
    # enough that others are owned by one CTA (direct write), in one launch
    lens = [20000, 37, 0, 50001, 8191, 16, 300]
    b = W.make_batch(lens, 64, 8, 128, 16, seed=21, device=DEV, poison_unused=True)
    check_batch(oracle, b, what="ragged")
    b32 = W.make_batch(lens, 32, 8, 128, 32, seed=22, device=DEV, poison_unused=True)
    check_batch(oracle, b32, what="ragged ps32")


def test_single_cta_path_vs_split_path_same_row(oracle):
    """The same logical row computed with 1 CTA (no split) and with the full grid must both match
    the oracle; forcing the grid exercises comem_set_grid_ctas."""
    b = W.make_batch([6000], 8, 1, 128, 16, seed=31, device=DEV)
    try:
        comem.comem_set_grid_ctas(1)
        o1, _, _ = check_batch(oracle, b, what="grid1")
        comem.comem_set_grid_ctas(7)
        o7, _, _ = check_batch(oracle, b, what="grid7")
    finally:
        comem.comem_set_grid_ctas(0)
    ofull, _, _ = check_batch(oracle, b, what="gridfull")
    assert float((o1.float() - ofull.float()).abs().max()) < 2e-2


# ---- closed forms on the GPU --------------------------------------------------------------------------
def test_o1_single_token_bit_exact():
    b = W.make_batch([1, 1, 1, 1], 64, 8, 128, 16, seed=41, device=DEV, poison_unused=True)
    out, lse = gpu_run(b)
    for i in range(4):
        pid = int(b.block_table[i, 0])
        v = b.v_pages[pid, 0]                                   # [Hkv, D]
        want = v.repeat_interleave(8, dim=0)
        assert torch.equal(bits(out[i]), bits(want))


def test_o2_identical_keys_mean_of_v(oracle):
    b = W.make_batch([777], 8, 1, 128, 16, seed=42, device=DEV)
    b.k_pages[:] = b.k_pages[0, 0, 0].clone()
    out, _ = gpu_run(b)
    pid = b.block_table[0, :49].long()
    v = b.v_pages[pid].reshape(-1, 128)[:777].double().mean(dim=0)
    assert float((out[0].double() - v).abs().max()) <= 2.0 ** -8 * float(v.abs().max()) + 1e-6


def test_o5_constant_v():
    b = W.make_batch([5000, 90], 16, 2, 128, 16, seed=43, device=DEV)
    c = torch.randn(128, generator=torch.Generator().manual_seed(1)).to(torch.bfloat16).to(DEV)
    b.v_pages[:] = c
    out, _ = gpu_run(b)
    # out is an exact weighted mean of identical rows: only the final bf16 rounding may differ
    assert float((out.double() - c.double()).abs().max()) <= 2.0 ** -8 * float(c.double().abs().max())


def test_o8_large_logits_no_overflow(oracle):
    b = W.make_batch([300], 8, 1, 128, 16, seed=44, device=DEV)
    b.q[:] = 0
    b.q[0, :, 0] = 16.0
    b.k_pages[:] = 0
    b.k_pages[:, :, :, 0] = 30.0
    pid, slot = int(b.block_table[0, 13]), 5
    b.k_pages[pid, slot, 0, 0] = 640.0                       # logit 16*640/sqrt(128) ~ 905 vs 42
    out, lse = gpu_run(b)
    assert torch.isfinite(out.float()).all() and torch.isfinite(lse).all()
    assert torch.equal(bits(out[0, 3]), bits(b.v_pages[pid, slot, 0]))
    check_batch(oracle, b, what="large logits")


# ---- bit-identity properties ---------------------------------------------------------------------------
def test_o9_page_permutation_bit_identical():
    lens = [20000, 37, 50001, 8191]
    b = W.make_batch(lens, 64, 8, 128, 16, seed=51, device=DEV, num_pages=6000)
    o1, l1 = gpu_run(b)
    for s in (5, 6):
        b2 = W.permute_pages(b, seed=s)
        o2, l2 = gpu_run(b2)
        assert torch.equal(bits(o1), bits(o2)) and torch.equal(l1, l2)


def test_o12_tail_poison_bit_identical():
    lens = [37, 16, 5, 4000, 1]
    clean = W.make_batch(lens, 32, 8, 128, 32, seed=52, device=DEV, num_pages=300, max_pages_per_seq=200)
    o1, l1 = gpu_run(clean)
    for poison in (float("nan"), float("inf"), -float("inf"), 1e38):
        dirty = W.make_batch(lens, 32, 8, 128, 32, seed=52, device=DEV, num_pages=300,
                             max_pages_per_seq=200, poison_unused=True)
        nanmask_k = torch.isnan(dirty.k_pages.float())
        dirty.k_pages[nanmask_k] = poison
        dirty.v_pages[torch.isnan(dirty.v_pages.float())] = poison
        dirty.block_table[dirty.block_table < 0] = 2 ** 30
        o2, l2 = gpu_run(dirty)
        assert torch.equal(bits(o1), bits(o2)) and torch.equal(l1, l2), poison


def test_run_to_run_and_cross_stream_determinism():
    b = W.make_batch([30000, 9000, 123], 64, 8, 128, 16, seed=53, device=DEV)
    o0, l0 = gpu_run(b)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    for i in range(10):
        o, l = gpu_run(b, stream=side if i % 2 else None)
        torch.cuda.synchronize()
        assert torch.equal(bits(o), bits(o0)) and torch.equal(l, l0)


# ---- API surface -------------------------------------------------------------------------------------------
def test_sync_entry_point_and_no_lse(oracle):
    b = W.make_batch([1234, 77], 16, 2, 64, 16, seed=61, device=DEV)
    out = comem.comem_decode_attn(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale)
    ref, _ = oracle_rows(oracle, b, all_pairs(b))
    assert_parity(errors(out, ref, all_pairs(b)), "sync")


def test_kv_append_matches_oracle(oracle):
    b = W.make_batch([15, 16, 31, 1000], 16, 2, 128, 16, seed=62, device=DEV, spare_tokens=40)
    kb = oracle.as_bits(b.k_pages.cpu()).copy()
    vb = oracle.as_bits(b.v_pages.cpu()).copy()
    sl = b.seq_lens.cpu().numpy().copy()
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    out = torch.empty_like(b.q)
    for step in range(35):
        q, nk, nv = W.decode_step_rows(b, step, 6200)
        comem.comem_kv_append_async(b.k_pages, b.v_pages, b.block_table, b.seq_lens, nk, nv)
        comem.comem_decode_attn_async(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                      b.softmax_scale, out, ws)
        oracle.kv_append(kb, vb, b.block_table.cpu(), sl, nk.cpu(), nv.cpu())
        if step in (0, 1, 16, 17, 34):
            torch.cuda.synchronize()
            assert np.array_equal(b.seq_lens.cpu().numpy(), sl)
            assert np.array_equal(oracle.as_bits(b.k_pages.cpu()), kb)       # append is byte-exact
            assert np.array_equal(oracle.as_bits(b.v_pages.cpu()), vb)
            ref, _ = oracle.decode_attn(q.cpu(), kb, vb, b.block_table.cpu(), sl, b.softmax_scale)
            assert_parity(errors(out, ref.reshape(-1, 128), all_pairs(b)), f"step {step}")


def test_decode_step_host(oracle):
    b = W.make_batch([4000, 333], 64, 8, 128, 16, seed=63, device=DEV, spare_tokens=4)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    q, nk, nv = (t.cpu().pin_memory() for t in W.decode_step_rows(b, 0, 6300))
    out_h = torch.empty_like(q).pin_memory()
    lse_h = torch.empty((2, 64), dtype=torch.float32).pin_memory()
    comem.comem_decode_step_host(q, nk, nv, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                 b.softmax_scale, out_h, ws, lse_host=lse_h)
    assert b.seq_lens.cpu().tolist() == [4001, 334]
    b2 = W.DecodeBatch(q=q.to(DEV), k_pages=b.k_pages, v_pages=b.v_pages, block_table=b.block_table,
                       seq_lens=b.seq_lens, softmax_scale=b.softmax_scale)
    ref, ref_lse = oracle_rows(oracle, b2, all_pairs(b2))
    assert_parity(errors(out_h.to(DEV), ref, all_pairs(b2)), "step_host")
    assert np.max(np.abs(lse_h.numpy().reshape(-1) - ref_lse)) < 1e-3


def test_decode_step_host_prebound_call_object():
    """comem.DecodeStepHost (arguments marshalled once) drives the same C entry point: over a few steps, with the host
    rows swapped through rebind(), it leaves the cache, the lengths and the outputs exactly as the plain call does."""
    a = W.make_batch([900, 47], 16, 2, 128, 16, seed=64, device=DEV, spare_tokens=8)
    b = W.make_batch([900, 47], 16, 2, 128, 16, seed=64, device=DEV, spare_tokens=8)
    wa, wb = comem.alloc_workspace(a.q, a.k_pages, a.block_table), comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    rows = [tuple(t.cpu().pin_memory() for t in W.decode_step_rows(a, i, 6400)) for i in range(5)]
    oa, ob = torch.empty_like(rows[0][0]).pin_memory(), torch.empty_like(rows[0][0]).pin_memory()
    step = comem.DecodeStepHost(*rows[0], b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, ob, wb)
    for i, (q, nk, nv) in enumerate(rows):
        comem.comem_decode_step_host(q, nk, nv, a.k_pages, a.v_pages, a.block_table, a.seq_lens, a.softmax_scale, oa, wa)
        step.rebind(q_host=q, new_k_host=nk, new_v_host=nv)()
        assert torch.equal(oa.view(torch.int16), ob.view(torch.int16)), i
    assert torch.equal(a.seq_lens, b.seq_lens) and torch.equal(a.k_pages.view(torch.int16), b.k_pages.view(torch.int16))


def test_decode_step_host_pageable_fallback(oracle):
    """Pageable (un-pinned) host buffers take the cudaMemcpyAsync path; same answer as the zero-copy path."""
    outs = []
    for pinned in (True, False):
        b = W.make_batch([4000, 333, 16], 32, 8, 128, 32, seed=65, device=DEV, spare_tokens=4)
        ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
        q, nk, nv = (t.cpu() for t in W.decode_step_rows(b, 0, 6500))
        out_h = torch.empty_like(q)
        lse_h = torch.empty((3, 32), dtype=torch.float32)
        if pinned:
            q, nk, nv, out_h, lse_h = (t.pin_memory() for t in (q, nk, nv, out_h, lse_h))
        for step in range(2):   # second call: no append (k, v = None)
            comem.comem_decode_step_host(q, nk if step == 0 else None, nv if step == 0 else None, b.k_pages,
                                         b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out_h, ws,
                                         lse_host=lse_h)
        assert b.seq_lens.cpu().tolist() == [4001, 334, 17]
        outs.append((out_h.clone(), lse_h.clone()))
        b2 = W.DecodeBatch(q=q.to(DEV), k_pages=b.k_pages, v_pages=b.v_pages, block_table=b.block_table,
                           seq_lens=b.seq_lens, softmax_scale=b.softmax_scale)
        ref, _ = oracle_rows(oracle, b2, all_pairs(b2))
        assert_parity(errors(out_h.to(DEV), ref, all_pairs(b2)), f"step_host pinned={pinned}")
    assert torch.equal(bits(outs[0][0]), bits(outs[1][0])) and torch.equal(outs[0][1], outs[1][1])


def test_unsupported_and_invalid_raise():
    b = W.make_batch([100], 16, 1, 128, 16, seed=64, device=DEV)                # group 16
    with pytest.raises(comem.ComemError) as e:
        gpu_run(b)
    assert e.value.status == comem.COMEM_ERR_UNSUPPORTED
    b = W.make_batch([100], 8, 1, 128, 16, seed=64, device=DEV)
    with pytest.raises(comem.ComemError) as e:
        gpu_run(b, workspace=torch.empty(1024, dtype=torch.uint8, device=DEV))
    assert e.value.status == comem.COMEM_ERR_WORKSPACE


# ---- fused combine (S7 inside K1) vs the stand-alone K2 ---------------------------------------------------
def test_fused_vs_two_phase_and_workspace_reuse(oracle):
    """One workspace, initialised once for the largest shape, serves fused calls of several shapes
    back to back (the arrival counters re-arm themselves); the two-call form SPLIT then COMBINE
    (un-fused K1 + K2) agrees with the fused launch within rounding and with the oracle."""
    big = W.make_batch([20000, 37, 0, 50001, 8191, 16, 300], 64, 8, 128, 16, seed=71, device=DEV)
    small = W.make_batch([9000, 1], 8, 2, 64, 32, seed=72, device=DEV)
    ws = comem.alloc_workspace(big.q, big.k_pages, big.block_table)
    for rep in range(3):
        for b in (big, small):
            fused, lse_f = gpu_run(b, workspace=ws)
            two = torch.full_like(b.q, float("nan"))
            lse_t = torch.full_like(lse_f, float("nan"))
            for ph in (comem.COMEM_PHASE_SPLIT, comem.COMEM_PHASE_COMBINE):
                comem.comem_decode_attn_phases_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                                     b.softmax_scale, two, ws, lse_out=lse_t, phases=ph)
            torch.cuda.synchronize()
            ref, _ = oracle_rows(oracle, b, all_pairs(b))
            assert_parity(errors(fused, ref, all_pairs(b)), f"fused rep{rep}")
            assert_parity(errors(two, ref, all_pairs(b)), f"two-phase rep{rep}")
            assert float((fused.float() - two.float()).abs().max()) <= 2.0 ** -7 * float(fused.float().abs().max())
            live = torch.isfinite(lse_f)
            assert torch.equal(live, torch.isfinite(lse_t))
            assert float((lse_f[live] - lse_t[live]).abs().max()) < 1e-4


def test_every_grid_size_same_answer(oracle):
    """Sweep the persistent grid (1 CTA ... more CTAs than tiles): every cut pattern of the
    segments goes through the fused merge and must match the oracle."""
    b = W.make_batch([3000, 555, 16], 16, 2, 128, 16, seed=73, device=DEV, poison_unused=True)
    try:
        for g in (1, 2, 3, 5, 8, 13, 37, 64, 148, 296, 1024):
            comem.comem_set_grid_ctas(g)
            check_batch(oracle, b, what=f"grid {g}")
    finally:
        comem.comem_set_grid_ctas(0)


def test_validate_inputs_debug_aid():
    """comem_validate_inputs flags exactly the two things the hot path trusts; the workspace it borrows
    stays usable (its counters are re-zeroed)."""
    b = W.make_batch([100, 37, 0, 5000], 8, 2, 64, 16, seed=81, device=DEV, poison_unused=True)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    ok = lambda bt, sl: comem.comem_validate_inputs(bt, sl, 16, b.num_pages, ws)  # noqa: E731
    assert ok(b.block_table, b.seq_lens) == comem.COMEM_OK            # -1 in IGNORED entries is fine
    bad = b.block_table.clone()
    bad[3, 7] = b.num_pages                                           # a used entry outside the pool
    assert ok(bad, b.seq_lens) == comem.COMEM_ERR_INVALID_ARG
    bad[3, 7] = -5
    assert ok(bad, b.seq_lens) == comem.COMEM_ERR_INVALID_ARG
    long = b.seq_lens.clone()
    long[1] = b.block_table.shape[1] * 16 + 1                         # longer than the table row reaches
    assert ok(b.block_table, long) == comem.COMEM_ERR_INVALID_ARG
    out, _ = gpu_run(b, workspace=ws)                                 # the borrowed workspace still works
    out2, _ = gpu_run(b)
    assert torch.equal(bits(out), bits(out2))


@pytest.mark.parametrize("case", range(24))
def test_randomised_shapes(oracle, case):
    """Seeded random draws over everything the ABI accepts: batch, kv heads, group, head_dim, page size,
    ragged lengths with zeros and tile/page-boundary values mixed in, and the persistent grid size
    (so that linear and segment-aligned schedules, whole and cut segments, one- and multi-round
    merges all occur)."""
    rng = np.random.default_rng(9000 + case)
    G = int(rng.choice([1, 2, 4, 8]))
    hkv = int(rng.integers(1, 9))
    D = int(rng.choice([64, 128]))
    ps = int(rng.choice([16, 32]))
    batch = int(rng.integers(1, 13))
    special = [0, 1, 15, 16, 17, ps - 1, ps, ps + 1, 255, 256, 257]
    lens = [int(rng.choice(special)) if rng.random() < 0.3 else int(rng.integers(1, 6000)) for _ in range(batch)]
    if case % 6 == 0:
        lens[0] = int(rng.integers(20000, 60000))          # one long sequence: many splits per segment
    grid = int(rng.choice([0, 0, 3, 17, 61, 148, 211, 600]))
    pool = max(1, sum(W.pages_needed(l, ps) for l in lens)) + int(rng.integers(0, 9))   # an all-empty batch still has a pool
    b = W.make_batch(lens, G * hkv, hkv, D, ps, seed=9100 + case, device=DEV, poison_unused=True, num_pages=pool)
    try:
        comem.comem_set_grid_ctas(grid)
        out, lse, _ = check_batch(oracle, b, what=f"case {case}: G{G} hkv{hkv} D{D} ps{ps} lens{lens} grid{grid}")
        out2, lse2 = gpu_run(W.permute_pages(b, seed=case))
        assert torch.equal(bits(out), bits(out2)) and torch.equal(lse.nan_to_num(neginf=-1e30), lse2.nan_to_num(neginf=-1e30))
    finally:
        comem.comem_set_grid_ctas(0)


# ---- the paper's batch sizes (Fig. 2: batch 1 / 16 / 64; L257 section 4.4: 32 -> 256; L463-470 Table 7:
# concurrency up to 128) and the ABI's limit: the strided prefix sum of the scheduler's prologue (batch > 32), the
# shared-memory prefix table at COMEM_MAX_BATCH, the linear schedule with thousands of segments, K2 at large batch ----
def _ragged(rng, batch, hi, zero_frac=0.1):
    special = [0, 1, 15, 16, 17, 31, 32, 33]
    return [0 if rng.random() < zero_frac else (int(rng.choice(special)) if rng.random() < 0.2 else int(rng.integers(1, hi)))
            for _ in range(batch)]


@pytest.mark.parametrize("batch,hi", [(33, 3000), (64, 2500), (128, 1200), (256, 700), (4096, 90)])
@pytest.mark.parametrize("G,ps", [(8, 16), (4, 32)])
def test_large_batches(oracle, batch, hi, G, ps):
    rng = np.random.default_rng(7000 + batch + G)
    lens = _ragged(rng, batch, hi)
    lens[batch // 2] = 4 * hi                      # one long sequence among the short ones: cut by several CTAs
    b = W.make_batch(lens, G * 8, 8, 128, ps, seed=7100 + batch + G, device=DEV, poison_unused=True)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    base = None
    for grid in (None, 1, 37, 148, 1024):
        out = torch.full_like(b.q, float("nan"))
        lse = torch.full((b.batch, b.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
        comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out, ws,
                                      lse_out=lse, grid_ctas=grid)
        torch.cuda.synchronize()
        if base is None:
            pairs = all_pairs(b) if batch <= 256 else [(x, h) for x in range(0, batch, 7) for h in range(0, G * 8, 5)] + \
                [(batch // 2, h) for h in range(G * 8)]
            ref, ref_lse = oracle_rows(oracle, b, pairs)
            base = (out, lse)
        assert_parity(errors(out, ref, pairs), f"batch {batch} grid {grid}")
        glse = np.array([float(lse[x, h]) for x, h in pairs])
        assert np.array_equal(np.isneginf(glse), np.isneginf(ref_lse))
        empty = (b.seq_lens == 0).nonzero().flatten().tolist()
        assert all(float(out[e].abs().max()) == 0.0 for e in empty[:8])
    # run to run and under a page permutation: bit-identical (default grid)
    o2, l2 = gpu_run(b, workspace=ws)
    o3, l3 = gpu_run(W.permute_pages(b, seed=batch))
    assert torch.equal(bits(base[0]), bits(o2)) and torch.equal(bits(base[0]), bits(o3))
    assert torch.equal(base[1].nan_to_num(neginf=-1e30), l3.nan_to_num(neginf=-1e30))
    # the two-call form (K1 un-fused, then the stand-alone K2) at this batch
    two = torch.full_like(b.q, float("nan"))
    for ph in (comem.COMEM_PHASE_SPLIT, comem.COMEM_PHASE_COMBINE):
        comem.comem_decode_attn_phases_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                             two, ws, phases=ph)
    torch.cuda.synchronize()
    assert_parity(errors(two, ref, pairs), f"batch {batch} two-phase")


def test_max_batch_fp8_and_window(oracle):
    """COMEM_MAX_BATCH with the FP8 cache and with a sliding window (the same prologue, other tile maps)."""
    rng = np.random.default_rng(7999)
    lens = _ragged(rng, 4096, 70)
    b = W.make_batch(lens, 16, 4, 128, 16, seed=7998, device=DEV, poison_unused=True)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    out = torch.full_like(b.q, float("nan"))
    comem.comem_decode_attn_window_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out,
                                         ws, 24, 2)
    torch.cuda.synchronize()
    c = b.to("cpu")
    ref, _ = oracle.decode_attn_window(c.q, c.k_pages, c.v_pages, c.block_table, c.seq_lens, c.softmax_scale, 24, 2)
    assert_parity(_err_dense(out, ref), "window at max batch")
    f = W.quantize_batch_fp8(b)
    out8 = torch.full_like(f.q, float("nan"))
    comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                      f.softmax_scale, out8, ws)
    torch.cuda.synchronize()
    cf = f.to("cpu")
    ref8, _ = oracle.decode_attn_fp8(cf.q, cf.k_pages, cf.v_pages, cf.k_scale, cf.v_scale, cf.block_table, cf.seq_lens,
                                     cf.softmax_scale)
    assert_parity(_err_dense(out8, ref8), "fp8 at max batch")


def _err_dense(gpu_out, ref):
    g = gpu_out.double().cpu().numpy().reshape(-1, gpu_out.shape[-1])
    r = np.asarray(ref).reshape(-1, gpu_out.shape[-1])
    d = np.abs(g - r)
    return {"max_abs": float(d.max()), "mean_abs": float(d.mean()),
            "rel_l2": float(np.linalg.norm(g - r) / max(np.linalg.norm(r), 1e-300)),
            "max_ref": float(np.abs(r).max()), "finite": bool(np.isfinite(g).all())}
