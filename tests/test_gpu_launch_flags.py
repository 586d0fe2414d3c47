"""GPU parity of the launch flags (include/comem_decode_attn.h, comem_launch_opts.flags):
COMEM_LAUNCH_KV_PREFIX_IMMUTABLE (the ring is filled before the PDL wait) must not change a bit;
COMEM_LAUNCH_SPLIT_COMBINE (the merge runs as a small dependent kernel) is checked against the oracle like any
other path, is bit-identical to itself under reruns and page permutation, and falls back to the fused kernel for
steps of many segments."""
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import check_batch, gpu_run

pytestmark = pytest.mark.gpu
DEV = "cuda"
IMM = comem.COMEM_LAUNCH_KV_PREFIX_IMMUTABLE
SC = comem.COMEM_LAUNCH_SPLIT_COMBINE
QS = comem.COMEM_LAUNCH_Q_STABLE
EARLY = [IMM, IMM | QS]


def bits(t):
    return t.contiguous().view(torch.int16)


CASES = [
    ([32768], 64, 8, 128, 16),            # C2's shape: 8 segments x 18-19 CTAs
    ([20000, 37, 0, 50001, 8191, 16, 300], 64, 8, 128, 16),
    ([5000, 1, 17], 32, 8, 128, 32),
    ([700, 64, 4097], 12, 3, 64, 32),
    ([9000, 33, 0, 2500, 17], 10, 2, 128, 16),   # G = 5
    ([15], 8, 1, 128, 16), ([16], 8, 1, 128, 16), ([17], 8, 1, 128, 16), ([33], 4, 1, 64, 16),
]


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("flags", EARLY)
def test_early_mode_is_bit_identical(oracle, case, flags):
    lens, hq, hkv, d, ps = case
    b = W.make_batch(lens, hq, hkv, d, ps, seed=501, device=DEV, poison_unused=True)
    out0, lse0 = gpu_run(b)
    res = [gpu_run(b, flags=flags) for _ in range(6)]  # back to back: each launch streams under the previous one
    torch.cuda.synchronize()
    for out1, lse1 in res:
        assert torch.equal(bits(out0), bits(out1))
        assert torch.equal(lse0.view(torch.int32), lse1.view(torch.int32))
    check_batch(oracle, b, flags=flags, what=f"early {flags} {case}")


@pytest.mark.parametrize("flags", EARLY)
def test_early_mode_fp8_and_grids(oracle, flags):
    f = W.quantize_batch_fp8(W.make_batch([3000, 17, 0, 640, 9000], 32, 8, 128, 16, seed=8, device=DEV, poison_unused=True))
    for fb in (f, W.to_hnd(f)):
        ws = comem.alloc_workspace(fb.q, fb.k_pages, fb.block_table, kv_layout=fb.kv_layout)
        for grid in (None, 5, 64):
            o0, o1 = torch.full_like(fb.q, float("nan")), torch.full_like(fb.q, float("nan"))
            comem.comem_decode_attn_fp8_async(fb.q, fb.k_pages, fb.v_pages, fb.k_scale, fb.v_scale, fb.block_table,
                                              fb.seq_lens, fb.softmax_scale, o0, ws, kv_layout=fb.kv_layout, grid_ctas=grid)
            for _ in range(3):
                comem.comem_decode_attn_fp8_async(fb.q, fb.k_pages, fb.v_pages, fb.k_scale, fb.v_scale, fb.block_table,
                                                  fb.seq_lens, fb.softmax_scale, o1, ws, kv_layout=fb.kv_layout,
                                                  grid_ctas=grid, flags=flags)
            torch.cuda.synchronize()
            assert torch.isfinite(o0.float()).all() and torch.equal(bits(o0), bits(o1)), (fb.kv_layout, grid)


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("flags", [SC, SC | IMM, SC | IMM | QS])
def test_split_combine_parity(oracle, case, flags):
    lens, hq, hkv, d, ps = case
    b = W.make_batch(lens, hq, hkv, d, ps, seed=502, device=DEV, poison_unused=True)
    out, lse, err = check_batch(oracle, b, flags=flags, what=f"split-combine {case}")
    for _ in range(4):
        out2, lse2 = gpu_run(b, flags=flags)
        torch.cuda.synchronize()
        assert torch.equal(bits(out), bits(out2)) and torch.equal(lse.view(torch.int32), lse2.view(torch.int32))
    bp = W.permute_pages(b, seed=77)
    out3, lse3 = gpu_run(bp, flags=flags)
    torch.cuda.synchronize()
    assert torch.equal(bits(out), bits(out3)) and torch.equal(lse.view(torch.int32), lse3.view(torch.int32))


@pytest.mark.parametrize("grid", [1, 7, 37, 148, 296])
def test_split_combine_grids(oracle, grid):
    b = W.make_batch([12000, 600, 0, 31], 32, 4, 128, 16, seed=503, device=DEV, poison_unused=True)
    out = torch.full_like(b.q, float("nan"))
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out, ws,
                                  grid_ctas=grid, flags=SC | IMM)
    ref = torch.full_like(b.q, float("nan"))
    comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, ref, ws,
                                  grid_ctas=grid)
    torch.cuda.synchronize()
    assert torch.isfinite(out.float()).all()
    # the two merges sum in different fixed orders: within a bf16 ulp of each other
    assert (out.float() - ref.float()).abs().max() <= 2.0 ** -7 * ref.float().abs().max()


def test_split_combine_many_segments_falls_back_to_fused():
    b = W.make_batch([300 + 17 * i for i in range(40)], 16, 2, 128, 16, seed=504, device=DEV, poison_unused=True)
    out0, _ = gpu_run(b)
    out1, _ = gpu_run(b, flags=SC)   # 80 segments > 64: the fused kernel runs, same bits
    torch.cuda.synchronize()
    assert torch.equal(bits(out0), bits(out1))


@pytest.mark.parametrize("flags", EARLY + [IMM | QS | SC])
def test_early_mode_with_growing_context(flags):
    """A decode loop (append, attend) enqueued WITHOUT host synchronisation: the append kernel releases its dependents
    at entry, so the attention kernel's early part runs while seq_lens still holds the previous length; whenever a
    length then crosses a tile boundary the guessed schedule is wrong and the early attempt is aborted and redone.
    Every step must match a run without the flags bit for bit (SPLIT_COMBINE: its own un-flagged run)."""
    lens = [4090, 33, 15, 250]
    b = W.make_batch(lens, 16, 2, 128, 16, seed=505, device=DEV, spare_tokens=48)
    ref = W.make_batch(lens, 16, 2, 128, 16, seed=505, device=DEV, spare_tokens=48)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    ws2 = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    steps = 40
    rows = [W.decode_step_rows(b, step, 9000) for step in range(steps)]
    o1 = [torch.empty_like(rows[0][0]) for _ in range(steps)]
    o2 = [torch.empty_like(rows[0][0]) for _ in range(steps)]
    torch.cuda.synchronize()
    for step, (q, nk, nv) in enumerate(rows):
        comem.comem_kv_append_async(b.k_pages, b.v_pages, b.block_table, b.seq_lens, nk, nv)
        comem.comem_decode_attn_async(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, o1[step], ws,
                                      flags=flags & ~QS)  # q rows are stable here (pre-generated), but keep QS for the 2nd pass
    torch.cuda.synchronize()
    for step, (q, nk, nv) in enumerate(rows):
        comem.comem_kv_append_async(ref.k_pages, ref.v_pages, ref.block_table, ref.seq_lens, nk, nv)
        comem.comem_decode_attn_async(q, ref.k_pages, ref.v_pages, ref.block_table, ref.seq_lens, ref.softmax_scale,
                                      o2[step], ws2, flags=flags & SC)
        torch.cuda.synchronize()
    for step in range(steps):
        assert torch.equal(bits(o1[step]), bits(o2[step])), step
    assert torch.equal(b.seq_lens, ref.seq_lens)
    # once more with the consumers starting early too (q is pre-generated: stable)
    b2 = W.make_batch(lens, 16, 2, 128, 16, seed=505, device=DEV, spare_tokens=48)
    o3 = [torch.empty_like(rows[0][0]) for _ in range(steps)]
    for step, (q, nk, nv) in enumerate(rows):
        comem.comem_kv_append_async(b2.k_pages, b2.v_pages, b2.block_table, b2.seq_lens, nk, nv)
        comem.comem_decode_attn_async(q, b2.k_pages, b2.v_pages, b2.block_table, b2.seq_lens, b2.softmax_scale, o3[step], ws,
                                      flags=flags)
    torch.cuda.synchronize()
    for step in range(steps):
        assert torch.equal(bits(o3[step]), bits(o2[step])), step


def test_recovery_paths_forced_by_a_stale_schedule_guess():
    """COMEM_DEBUG_STALE_GUESS=1 makes every launch compute its first schedule from lengths 16 tokens short: the
    validation after the wait fails on every launch, so the classic re-computation and the early mode's abort (drain,
    barrier re-initialisation, rerun in the classic order) run deterministically.  In a fresh process (the switch is
    read once), every flag combination must give the bits of an un-flagged run of THIS process."""
    import os
    import subprocess
    import sys
    code = r'''
import torch
import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
def bits(t): return t.contiguous().view(torch.int16)
ok = True
for lens, hq, hkv, d, ps in [([32768], 64, 8, 128, 16), ([20000, 37, 0, 50001, 8191, 16, 300], 64, 8, 128, 16), ([700, 64, 4097], 12, 3, 64, 32), ([17], 8, 1, 128, 16)]:
    b = W.make_batch(lens, hq, hkv, d, ps, seed=901, device="cuda", poison_unused=True)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    outs = {}
    for flags in (0, 1, 5, 7, 2):
        o = torch.full_like(b.q, float("nan"))
        for _ in range(3):
            comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, o, ws, flags=flags)
        torch.cuda.synchronize()
        outs[flags] = o
    ok = ok and torch.isfinite(outs[0].float()).all().item()
    ok = ok and torch.equal(bits(outs[0]), bits(outs[1])) and torch.equal(bits(outs[0]), bits(outs[5]))
    ok = ok and torch.equal(bits(outs[2]), bits(outs[7]))
    f = W.quantize_batch_fp8(b) if d == 128 else None
    if f is not None:
        ws8 = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
        o8 = {}
        for flags in (0, 5):
            o = torch.full_like(f.q, float("nan"))
            comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens, f.softmax_scale, o, ws8, flags=flags)
            torch.cuda.synchronize()
            o8[flags] = o
        ok = ok and torch.equal(bits(o8[0]), bits(o8[5]))
print("RESULT", ok)
'''
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    ref = {}
    for stale in ("0", "1"):
        env = dict(os.environ, COMEM_DEBUG_STALE_GUESS=stale, PYTHONPATH=root)
        r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        assert "RESULT True" in r.stdout, (stale, r.stdout[-500:], r.stderr[-1500:])


def test_all_flags_on_the_fp8_cache_and_the_two_tier_cache(oracle):
    """KV_PREFIX_IMMUTABLE | Q_STABLE | SPLIT_COMBINE on the other instances of the kernel: the FP8 cache (NHD and HND)
    against its oracle and its own un-flagged SPLIT_COMBINE run, and the two-tier cache against the all-HBM bits."""
    import numpy as np
    ALL = IMM | QS | SC
    f = W.quantize_batch_fp8(W.make_batch([9000, 17, 0, 640], 32, 8, 128, 16, seed=31, device=DEV, poison_unused=True))
    for fb in (f, W.to_hnd(f)):
        ws = comem.alloc_workspace(fb.q, fb.k_pages, fb.block_table, kv_layout=fb.kv_layout)
        outs = {}
        for flags in (SC, ALL):
            o = torch.full_like(fb.q, float("nan"))
            for _ in range(3):
                comem.comem_decode_attn_fp8_async(fb.q, fb.k_pages, fb.v_pages, fb.k_scale, fb.v_scale, fb.block_table,
                                                  fb.seq_lens, fb.softmax_scale, o, ws, kv_layout=fb.kv_layout, flags=flags)
            torch.cuda.synchronize()
            outs[flags] = o
        assert torch.equal(bits(outs[SC]), bits(outs[ALL])), fb.kv_layout
        c = fb.to("cpu")
        ref, _ = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table, c.seq_lens,
                                        c.softmax_scale, kv_layout=c.kv_layout)
        d = np.abs(outs[ALL].double().cpu().numpy() - ref)
        assert d.max() <= 2e-2 and d.mean() <= 2e-3 and np.linalg.norm(d) / np.linalg.norm(ref) <= 5e-3
    b = W.make_batch([30000], 64, 8, 128, 16, seed=32, device=DEV, poison_unused=True)
    ref_out, _ = gpu_run(b, flags=SC)
    ob = W.offload_pages(b, 0.2, seed=3, coldest_first=False)
    bb = ob.base
    out = torch.full_like(bb.q, float("nan"))
    ws = comem.alloc_workspace(bb.q, bb.k_pages, bb.block_table)
    for _ in range(3):
        comem.comem_decode_attn_offload_async(bb.q, bb.k_pages, bb.v_pages, ob.k_host, ob.v_host, bb.block_table, bb.seq_lens,
                                              bb.softmax_scale, out, ws, flags=ALL)
    torch.cuda.synchronize()
    assert torch.equal(bits(out), bits(ref_out))
