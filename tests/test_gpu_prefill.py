"""GPU parity of the paged causal prefill kernel (reading R20; comem_prefill_attn_async, the tcgen05
kernel) against oracle_prefill_attn on the same bits, through the C-ABI.  Tolerances: tests/parity_util.py."""
import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W

from parity_util import MAX_ABS, MEAN_ABS, REL_L2

pytestmark = pytest.mark.gpu


def gpu_prefill(pb, want_lse=True, stream=None):
    out = torch.full_like(pb.q, float("nan"))
    lse = torch.full((pb.total_q, pb.num_q_heads), float("nan"), dtype=torch.float32, device=pb.q.device) if want_lse else None
    comem.comem_prefill_attn_async(pb.q, pb.k_pages, pb.v_pages, pb.block_table, pb.seq_lens, pb.q_start,
                                   pb.softmax_scale, out, lse_out=lse, stream=stream)
    return out, lse


def check(oracle, pb, what=""):
    out, lse = gpu_prefill(pb)
    torch.cuda.synchronize()
    c = pb.to("cpu")
    ref, ref_lse = oracle.prefill_attn(c.q, c.k_pages, c.v_pages, c.block_table, c.seq_lens, c.q_start, c.softmax_scale)
    g = out.double().cpu().numpy()
    assert np.isfinite(g).all(), what
    d = np.abs(g - ref)
    err = {"max_abs": float(d.max()), "mean_abs": float(d.mean()),
           "rel_l2": float(np.linalg.norm(g - ref) / max(np.linalg.norm(ref), 1e-300)), "max_ref": float(np.abs(ref).max())}
    assert err["max_abs"] <= MAX_ABS and err["mean_abs"] <= MEAN_ABS and err["rel_l2"] <= REL_L2, (what, err)
    assert err["max_abs"] <= 4 * 2.0 ** -9 * err["max_ref"] + 1e-6, (what, err)
    gl = lse.double().cpu().numpy()
    assert np.max(np.abs(gl - ref_lse) / np.maximum(1.0, np.abs(ref_lse))) <= 2e-4, what
    return out, err


@pytest.mark.parametrize("n", [1, 15, 16, 17, 128, 512])
@pytest.mark.parametrize("prefix", [0, 1, 31, 4096])
def test_chunk_over_prefix(oracle, n, prefix):
    pb = W.make_prefill_batch([prefix + n], [n], 64, 8, 128, 16, seed=100 + n + prefix, device="cuda", poison_unused=True)
    check(oracle, pb, f"n={n} prefix={prefix}")


@pytest.mark.parametrize("hq,hkv,d,ps", [(32, 8, 128, 32), (4, 1, 64, 16), (8, 8, 128, 16), (16, 8, 64, 32), (16, 1, 128, 16)])
def test_geometries_ragged_batch(oracle, hq, hkv, d, ps):
    lens = [700, 33, 1, 2050, 129]
    qn = [300, 33, 1, 17, 0]
    pb = W.make_prefill_batch(lens, qn, hq, hkv, d, ps, seed=5, device="cuda", poison_unused=True)
    check(oracle, pb, f"{hq}/{hkv}/{d}/{ps}")


def test_uncached_full_prefill_4096(oracle):
    pb = W.make_prefill_batch([4096], [4096], 32, 8, 128, 16, seed=9, device="cuda", poison_unused=True)
    check(oracle, pb, "full 4096")


def test_page_permutation_bit_identical():
    pb = W.make_prefill_batch([1500, 640], [900, 640], 64, 8, 128, 16, seed=11, device="cuda")
    out0, _ = gpu_prefill(pb, want_lse=False)
    g = torch.Generator().manual_seed(3)
    perm = torch.randperm(pb.k_pages.shape[0], generator=g).to(pb.q.device)
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(perm.numel(), device=perm.device)
    import dataclasses
    pb2 = dataclasses.replace(pb, k_pages=pb.k_pages[perm].contiguous(), v_pages=pb.v_pages[perm].contiguous(),
                              block_table=inv[pb.block_table.long().clamp_min(0)].to(torch.int32))
    out1, _ = gpu_prefill(pb2, want_lse=False)
    torch.cuda.synchronize()
    assert torch.equal(out0.view(torch.int16), out1.view(torch.int16))
    out2, _ = gpu_prefill(pb, want_lse=False)
    torch.cuda.synchronize()
    assert torch.equal(out0.view(torch.int16), out2.view(torch.int16))


@pytest.mark.parametrize("grid", [1, 3, 16, 100, 100000])
def test_persistent_grid_is_bit_identical(grid):
    """comem_launch_opts.grid_ctas on the prefill call: the kernel becomes persistent on that many SMs (each CTA takes every
    grid-th work item, re-initialising its barriers in between).  A row is computed by one thread in a fixed order
    whatever CTA runs it, so the bits are those of the default launch; with and without lse_out."""
    pb = W.make_prefill_batch([700, 4100, 33, 1], [700, 300, 33, 1], 32, 4, 128, 16, seed=811, device="cuda", poison_unused=True)
    ref, ref_lse = gpu_prefill(pb)
    out = torch.full_like(pb.q, float("nan"))
    lse = torch.full((pb.total_q, pb.num_q_heads), float("nan"), dtype=torch.float32, device="cuda")
    comem.comem_prefill_attn_async(pb.q, pb.k_pages, pb.v_pages, pb.block_table, pb.seq_lens, pb.q_start, pb.softmax_scale,
                                   out, lse_out=lse, grid_ctas=grid)
    out2 = torch.full_like(pb.q, float("nan"))
    comem.comem_prefill_attn_async(pb.q, pb.k_pages, pb.v_pages, pb.block_table, pb.seq_lens, pb.q_start, pb.softmax_scale,
                                   out2, grid_ctas=grid)
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int16), ref.view(torch.int16))
    assert torch.equal(out2.view(torch.int16), ref.view(torch.int16))
    assert torch.equal(lse.view(torch.int32), ref_lse.view(torch.int32))
