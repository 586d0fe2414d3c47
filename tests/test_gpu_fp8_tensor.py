"""GPU parity of the tcgen05 split kernel for the FP8 cache (COMEM_LAUNCH_FP8_TENSOR, csrc/decode_fp8_tc.cu) against
oracle.decode_attn_fp8 on the same bytes, at the tolerances of the default FP8 kernel, plus the properties that fix
bits (reruns, page placement, pool layout) and the error codes of what the kernel does not take."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from test_gpu_fp8 import bits, fp8_batch, gate

pytestmark = pytest.mark.gpu
DEV = "cuda"
TENSOR = comem.COMEM_LAUNCH_FP8_TENSOR


def run_tc(f, grid=None, flags=TENSOR, window=0, sinks=0):
    out = torch.full_like(f.q, float("nan"))
    lse = torch.full((f.batch, f.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
    ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
    comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                      f.softmax_scale, out, ws, window, sinks, lse_out=lse, kv_layout=f.kv_layout,
                                      grid_ctas=grid, flags=flags)
    torch.cuda.synchronize()
    return out, lse


def check_tc(oracle, f, what, grid=None, flags=TENSOR):
    out, lse = run_tc(f, grid, flags)
    c = f.to("cpu")
    ref, ref_lse = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table,
                                          c.seq_lens, c.softmax_scale, 0, 0, kv_layout=c.kv_layout)
    gate(out.double().cpu().numpy(), ref, lse.double().cpu().numpy(), ref_lse, what)
    return out, lse


@pytest.mark.parametrize("G,ps", [(1, 16), (4, 32), (8, 16), (3, 32), (5, 16), (8, 32)])
def test_tensor_small_ragged(oracle, G, ps):
    lens = [1, 15, 16, 17, 31, 33, 127, 128, 129, 512, 1000, 0, 2049]
    f = fp8_batch(lens, 2 * G, 2, ps, seed=700 + G + ps)
    check_tc(oracle, f, f"tensor G{G} ps{ps}")


def test_tensor_long_ragged_grids_permutation_layout(oracle):
    lens = [20000, 37, 0, 50001, 8191, 16, 300]
    f = fp8_batch(lens, 64, 8, 16, seed=721)
    base, base_lse = check_tc(oracle, f, "tensor ragged default grid")
    again, again_lse = run_tc(f)
    assert torch.equal(bits(base), bits(again)) and torch.equal(base_lse, again_lse)        # run to run
    po, pl = run_tc(W.permute_pages_fp8(f, seed=9))
    assert torch.equal(bits(base), bits(po)) and torch.equal(base_lse, pl)                  # page placement
    ho, hl = check_tc(oracle, W.to_hnd(f), "tensor ragged HND")
    assert torch.equal(bits(base), bits(ho)) and torch.equal(base_lse, hl)                  # pool layout
    for grid in (1, 7, 61, 148, 296):
        check_tc(oracle, f, f"tensor ragged grid {grid}", grid=grid)
    # the other launch flags are accepted and change nothing
    fo, fl = run_tc(f, flags=TENSOR | 7)
    assert torch.equal(bits(base), bits(fo)) and torch.equal(base_lse, fl)


def test_tensor_single_long_sequence(oracle):
    f = fp8_batch([32768], 64, 8, 16, seed=722, k_scale=0.5)
    check_tc(oracle, f, "tensor c2-shaped")
    check_tc(oracle, W.to_hnd(f), "tensor c2-shaped HND")


@pytest.mark.parametrize("nats,v_mean", [(12.0, 0.3), (14.0, 0.15)])
def test_tensor_sink_token_small_v_scale(oracle, nats, v_mean):
    """One sink token far above a flat 32K tail with page scales <= 2e-3: the tail's p * v_scale must keep its bits
    through the E4M3 split (only the scale's mantissa and a relative power of two ride on p)."""
    f = W.quantize_batch_fp8(W.sink_batch(32768, 32, 8, 128, 16, seed=730, device=DEV, sink_nats=nats, v_mean=v_mean,
                                          v_std=v_mean / 3))
    check_tc(oracle, f, f"tensor sink {nats} nats")


def test_tensor_mixed_page_scales(oracle):
    """v_scale exponents spread over 2^-12 .. 2^6 within a sequence: the running reference exponent moves, O is rescaled."""
    b = W.make_batch([3000, 777], 32, 8, 128, 16, seed=731, device=DEV, poison_unused=True)
    gen = torch.Generator(device=DEV)
    gen.manual_seed(5)
    expo = torch.randint(-12, 7, (b.v_pages.shape[0], 1, 8, 1), generator=gen, device=DEV).float()
    b.v_pages.copy_((b.v_pages.float() * torch.exp2(expo)).to(torch.bfloat16))
    check_tc(oracle, W.quantize_batch_fp8(b), "tensor mixed page scales")


def test_tensor_rising_logits(oracle):
    """Keys whose scores grow along the sequence: every super tile raises the running maximum (the slow path each time)."""
    b = W.make_batch([4096, 1500], 16, 2, 128, 16, seed=732, device=DEV, poison_unused=True)
    f = W.quantize_batch_fp8(b)
    ramp = torch.linspace(0.2, 3.0, 4096, device=DEV)
    for s in range(2):
        n = int(f.seq_lens[s])
        for t0 in range(0, n, 16):
            pid = int(f.block_table[s, t0 // 16])
            f.k_scale[pid] *= float(ramp[t0])
    check_tc(oracle, f, "tensor rising logits")


def test_tensor_all_byte_codes_exact(oracle):
    """L = 1, unit scales: the weight is exactly 1 (hi = 128 * 2, lo = 0 after the split), so out = bf16(e4m3(V byte))
    exactly for every finite byte code, and lse = scale * q . k checks the K side and the exact split of q."""
    f = fp8_batch([1, 1], 8, 1, 16, seed=724)
    codes = torch.arange(256, dtype=torch.uint8, device=DEV)
    codes = torch.where((codes & 0x7f) == 0x7f, torch.zeros_like(codes), codes)
    for b in range(2):
        pid = int(f.block_table[b, 0])
        f.v_pages[pid, 0, 0] = codes[128 * b:128 * (b + 1)]
        f.k_pages[pid, 0, 0] = codes[128 * b:128 * (b + 1)].flip(0)
        f.k_scale[pid, 0] = 1.0
        f.v_scale[pid, 0] = 1.0
    f = dataclasses.replace(f, q=(f.q.float() / 64).to(torch.bfloat16))
    out, lse = run_tc(f)
    want = codes.view(torch.float8_e4m3fn).float()
    for b in range(2):
        for h in range(8):
            assert torch.equal(out[b, h].float(), want[128 * b:128 * (b + 1)]), (b, h)
    c = f.to("cpu")
    _, ref_lse = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table, c.seq_lens,
                                        c.softmax_scale)
    assert np.max(np.abs(lse.double().cpu().numpy() - ref_lse) / np.maximum(1.0, np.abs(ref_lse))) <= 1e-5


@pytest.mark.parametrize("batch", [33, 64, 256, 1024])
def test_tensor_large_batches(oracle, batch):
    """The paper's batch sizes: many short segments per CTA, whole and cut, zeros mixed in."""
    rng = np.random.default_rng(7400 + batch)
    lens = [0 if rng.random() < 0.05 else int(rng.integers(1, 700)) for _ in range(batch)]
    f = fp8_batch(lens, 16, 4, 16, seed=7400 + batch)
    out, lse = check_tc(oracle, f, f"tensor batch {batch}")
    po, pl = run_tc(W.permute_pages_fp8(f, seed=batch))
    assert torch.equal(bits(out), bits(po))
    assert torch.equal(lse.nan_to_num(neginf=-1e30), pl.nan_to_num(neginf=-1e30))


@pytest.mark.parametrize("case", range(10))
def test_tensor_randomised_shapes(oracle, case):
    rng = np.random.default_rng(9700 + case)
    G, hkv, ps = int(rng.integers(1, 9)), int(rng.integers(1, 9)), int(rng.choice([16, 32]))
    batch = int(rng.integers(1, 11))
    special = [0, 1, 15, 16, 17, ps - 1, ps, ps + 1, 127, 128, 129, 255, 256, 257]
    lens = [int(rng.choice(special)) if rng.random() < 0.3 else int(rng.integers(1, 6000)) for _ in range(batch)]
    if case % 4 == 0:
        lens[0] = int(rng.integers(20000, 60000))
    grid = int(rng.choice([0, 0, 3, 17, 61, 148, 211, 600]))
    f = fp8_batch(lens, G * hkv, hkv, ps, seed=9800 + case)
    if rng.random() < 0.5:
        f = W.to_hnd(f)
    what = f"tensor case {case}: G{G} hkv{hkv} ps{ps} {f.kv_layout} lens{lens} grid{grid}"
    out, lse = check_tc(oracle, f, what, grid=grid or None)
    out2, lse2 = run_tc(W.permute_pages_fp8(f, seed=case), grid=grid or None)
    assert torch.equal(bits(out), bits(out2)), what
    assert torch.equal(lse.nan_to_num(neginf=-1e30), lse2.nan_to_num(neginf=-1e30)), what


def test_tensor_flag_rejections():
    """The flag belongs to the FP8 entry points; head_dim 64, a sliding window and batch > 1024 are not taken."""
    b = W.make_batch([100], 8, 2, 128, 16, seed=1, device=DEV)
    out = torch.empty_like(b.q)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    with pytest.raises(comem.ComemError) as e:
        comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, out, ws,
                                      flags=TENSOR)
    assert e.value.status == comem.COMEM_ERR_INVALID_ARG
    f = fp8_batch([300, 20], 8, 2, 16, seed=2)
    with pytest.raises(comem.ComemError) as e:
        run_tc(f, window=64, sinks=2)
    assert e.value.status == comem.COMEM_ERR_UNSUPPORTED
    f64 = W.quantize_batch_fp8(W.make_batch([300], 8, 2, 64, 16, seed=3, device=DEV))
    with pytest.raises(comem.ComemError) as e:
        run_tc(f64)
    assert e.value.status == comem.COMEM_ERR_UNSUPPORTED
    big = fp8_batch([5] * 1025, 4, 1, 16, seed=4)
    with pytest.raises(comem.ComemError) as e:
        run_tc(big)
    assert e.value.status == comem.COMEM_ERR_UNSUPPORTED
    torch.cuda.synchronize()


def test_tensor_append_then_attend_loop(oracle):
    """40 decode steps enqueued without host synchronisation: quantising append, then the tensor kernel, which computes
    its schedule speculatively while the append kernel may still be bumping seq_lens (a length crosses a tile boundary
    once in 16 steps: the validation after the wait must catch it).  Outputs against the oracle on the final cache at
    the steps kept, and against the default kernel within the attention tolerances at every step."""
    ps = 16
    lens = [ps - 3, 5000, 0, 2 * ps - 1, 777, 12000]
    b = W.make_batch(lens, 16, 4, 128, ps, seed=761, device=DEV, spare_tokens=48)
    f = W.quantize_batch_fp8(b)
    f.k_scale.copy_(torch.where(torch.isnan(f.k_scale) | (f.k_scale == 1.0), torch.full_like(f.k_scale, 0.011), f.k_scale))
    f.v_scale.copy_(torch.where(torch.isnan(f.v_scale) | (f.v_scale == 1.0), torch.full_like(f.v_scale, 0.009), f.v_scale))
    f = dataclasses.replace(f, seq_lens=f.seq_lens.clone())
    ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
    ws2 = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
    outs_t, outs_d, qs = [], [], []
    for step in range(40):
        q, nk, nv = W.decode_step_rows(b, step, seed_base=7700)
        comem.comem_kv_append_fp8_async(f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens, nk, nv,
                                        kv_layout=f.kv_layout)
        ot, od = torch.full_like(q, float("nan")), torch.full_like(q, float("nan"))
        comem.comem_decode_attn_fp8_async(q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                          f.softmax_scale, ot, ws, kv_layout=f.kv_layout, flags=TENSOR)
        comem.comem_decode_attn_fp8_async(q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                          f.softmax_scale, od, ws2, kv_layout=f.kv_layout)
        outs_t.append(ot), outs_d.append(od), qs.append(q)
    torch.cuda.synchronize()
    assert f.seq_lens.tolist() == [l + 40 for l in lens]
    for step in range(40):
        a, d = outs_t[step].double().cpu().numpy(), outs_d[step].double().cpu().numpy()
        assert np.isfinite(a).all(), step
        assert np.abs(a - d).max() <= 2 * 2e-2 and np.linalg.norm(a - d) <= 2 * 5e-3 * np.linalg.norm(d), step
    # the last step against the oracle on the final cache
    c = dataclasses.replace(f, q=qs[-1]).to("cpu")
    ref, _ = oracle.decode_attn_fp8(c.q, c.k_pages, c.v_pages, c.k_scale, c.v_scale, c.block_table, c.seq_lens,
                                    c.softmax_scale, 0, 0, kv_layout=c.kv_layout)
    gate(outs_t[-1].double().cpu().numpy(), ref, np.full(ref.shape[:2], 0.0), np.full(ref.shape[:2], 0.0), "tensor loop, last step")


def test_tensor_recovery_path_forced_by_a_stale_schedule_guess():
    """COMEM_DEBUG_STALE_GUESS=1 (fresh process): the tensor kernel's first schedule comes from lengths 16 tokens short,
    so its validation after the wait fails on every launch and the schedule is recomputed; same bits as without."""
    import os
    import subprocess
    import sys
    code = r'''
import torch, hashlib
import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
h = hashlib.sha256()
for lens, hq, hkv, ps in [([32768], 64, 8, 16), ([20000, 37, 0, 50001, 8191, 16, 300], 64, 8, 16), ([700, 64, 4097], 12, 3, 32), ([17], 8, 1, 16)]:
    f = W.quantize_batch_fp8(W.make_batch(lens, hq, hkv, 128, ps, seed=902, device="cuda", poison_unused=True))
    ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
    o = torch.full_like(f.q, float("nan"))
    for _ in range(3):
        comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                          f.softmax_scale, o, ws, kv_layout=f.kv_layout, flags=comem.COMEM_LAUNCH_FP8_TENSOR)
    torch.cuda.synchronize()
    assert torch.isfinite(o.float()).all().item()
    h.update(o.contiguous().view(torch.int16).cpu().numpy().tobytes())
print("RESULT", h.hexdigest())
'''
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    digests = []
    for stale in ("0", "1"):
        env = dict(os.environ, COMEM_DEBUG_STALE_GUESS=stale, PYTHONPATH=root)
        r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        assert "RESULT" in r.stdout, (stale, r.stdout[-500:], r.stderr[-1500:])
        digests.append(r.stdout.split("RESULT")[1].strip())
    assert digests[0] == digests[1]


@pytest.mark.parametrize("batch,hkv,hi", [(1000, 8, 40), (517, 2, 130), (64, 8, 16)])
def test_tensor_many_one_tile_portions(oracle, batch, hkv, hi):
    """Sequences of one to a few tiles: a CTA walks dozens of portions of a single super tile each, so the eight Qs buffers
    and the eight S buffers cycle as fast as they can (their reuse is covered by the ring's hand-off, not by a barrier)."""
    rng = np.random.default_rng(8800 + batch)
    lens = [int(rng.integers(1, hi + 1)) for _ in range(batch)]
    f = fp8_batch(lens, 4 * hkv, hkv, 16, seed=8800 + batch)
    out, lse = check_tc(oracle, f, f"tensor tiny sequences {batch}")
    again, again_lse = run_tc(f)
    assert torch.equal(bits(out), bits(again)) and torch.equal(lse, again_lse)
    for grid in (37, 148):
        check_tc(oracle, f, f"tensor tiny sequences {batch} grid {grid}", grid=grid)


@pytest.mark.parametrize("G,hkv", [(8, 8), (4, 2), (3, 5)])
def test_tensor_hnd_32_token_pages(oracle, G, hkv):
    """HND pools with 32-token pages (two tiles per page, config 4's layout): grids that cut the segments at odd tiles,
    ragged ends inside a page's first and second tile, page permutation, reruns."""
    lens = [20000, 37, 0, 50001, 8191, 16, 17, 300, 48, 49, 4097]
    f = W.to_hnd(fp8_batch(lens, G * hkv, hkv, 32, seed=880 + G))
    base, base_lse = check_tc(oracle, f, f"tensor HND ps32 G{G} hkv{hkv}")
    again, again_lse = run_tc(f)
    assert torch.equal(bits(base), bits(again)) and torch.equal(base_lse, again_lse)
    po, pl = run_tc(W.permute_pages_fp8(f, seed=11))
    assert torch.equal(bits(base), bits(po)) and torch.equal(base_lse, pl)
    for grid in (1, 3, 7, 61, 147, 148, 149, 296, 601):
        check_tc(oracle, f, f"tensor HND ps32 grid {grid}", grid=grid)


def test_tensor_c4_shape_sampled(oracle):
    """Config 4's geometry (32q / 8kv, 32-token pages, HND), 4 x 131072 tokens: two whole sequences against the oracle."""
    bf = W.make_batch([131072, 131072, 100000, 65537], 32, 8, 128, 32, seed=890, device=DEV, poison_unused=True)
    f = W.to_hnd(W.quantize_batch_fp8(bf))
    del bf
    out, lse = run_tc(f)
    ps = f.page_size
    for b in (1, 3):
        n = W.pages_needed(int(f.seq_lens[b]), ps)
        ids = f.block_table[b, :n].long()
        sub = W.Fp8DecodeBatch(q=f.q[b:b + 1].cpu(), k_pages=f.k_pages[ids].cpu(), v_pages=f.v_pages[ids].cpu(),
                               k_scale=f.k_scale[ids].cpu(), v_scale=f.v_scale[ids].cpu(),
                               block_table=torch.arange(n, dtype=torch.int32).view(1, n),
                               seq_lens=f.seq_lens[b:b + 1].cpu(), softmax_scale=f.softmax_scale, kv_layout="HND")
        ref, ref_lse = oracle.decode_attn_fp8(sub.q, sub.k_pages, sub.v_pages, sub.k_scale, sub.v_scale, sub.block_table,
                                              sub.seq_lens, sub.softmax_scale, kv_layout="HND")
        gate(out[b:b + 1].double().cpu().numpy(), ref, lse[b:b + 1].double().cpu().numpy(), ref_lse, f"tensor c4 shape seq {b}")


def test_tensor_against_the_default_kernel_over_random_shapes():
    """Sixty seeded shapes (hundreds of one-tile sequences, ragged mid-size batches, one long sequence among short ones;
    group 1..8, 1..8 kv heads, both page sizes and pool layouts, grids 1..1000): the tensor kernel's output is finite,
    the same on a second run, and within twice the attention tolerances of the default FP8 kernel's on the same bytes."""
    rng = np.random.default_rng(2024)

    def run(f, flags, grid):
        out = torch.full_like(f.q, float("nan"))
        ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, kv_layout=f.kv_layout)
        comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table, f.seq_lens,
                                          f.softmax_scale, out, ws, 0, 0, kv_layout=f.kv_layout, flags=flags, grid_ctas=grid)
        torch.cuda.synchronize()
        return out.double()

    for case in range(60):
        G, hkv, ps = int(rng.integers(1, 9)), int(rng.integers(1, 9)), int(rng.choice([16, 32]))
        kind = case % 4
        if kind == 0:
            lens = [int(rng.integers(0, 40)) for _ in range(int(rng.integers(1, 900)))]
        elif kind == 1:
            lens = [int(rng.integers(1, 3000)) for _ in range(int(rng.integers(1, 40)))]
        elif kind == 2:
            lens = [int(rng.integers(100, 140)) for _ in range(int(rng.integers(1, 300)))]
        else:
            lens = [int(rng.integers(20000, 70000))] + [int(rng.integers(0, 300)) for _ in range(int(rng.integers(0, 20)))]
        grid = int(rng.choice([0, 1, 2, 5, 37, 148, 149, 300, 1000])) or None
        f = fp8_batch(lens, G * hkv, hkv, ps, seed=5000 + case)
        if rng.random() < 0.5:
            f = W.to_hnd(f)
        what = (case, G, hkv, ps, f.kv_layout, len(lens), grid)
        a, a2, b = run(f, TENSOR, grid), run(f, TENSOR, grid), run(f, 0, grid)
        assert torch.isfinite(a).all(), what
        assert torch.equal(a, a2), what
        assert (a - b).abs().max().item() <= 2 * 2e-2, what
        assert ((a - b).norm() / b.norm().clamp_min(1e-30)).item() <= 2 * 5e-3, what
