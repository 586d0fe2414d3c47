"""GPU parity of the two-tier cache (CPU offloading):
comem_decode_attn_offload_async with 0 / 10 / 50 / 100 % of the pages in pinned host memory must give the bits of the
all-HBM call (placement never enters the arithmetic) and match the oracle, which is given the same cache as one pool
(pure data movement: workloads.combined_pool_cpu; the oracle's indifference to placement is pin O9).
comem_pages_copy_async (the migration step) is checked byte for byte."""
import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import all_pairs, assert_parity, errors, gpu_run

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t):
    return t.contiguous().view(torch.int16)


def run_offload(ob, flags=0, grid=None):
    b = ob.base
    out = torch.full_like(b.q, float("nan"))
    lse = torch.full((b.batch, b.num_q_heads), float("nan"), dtype=torch.float32, device=b.q.device)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    comem.comem_decode_attn_offload_async(b.q, b.k_pages, b.v_pages, ob.k_host, ob.v_host, b.block_table, b.seq_lens,
                                          b.softmax_scale, out, ws, lse_out=lse, grid_ctas=grid, flags=flags)
    torch.cuda.synchronize()
    return out, lse


CASES = [
    ([9000, 33, 0, 2500, 17], 64, 8, 128, 16),
    ([700, 64, 4097], 12, 3, 64, 32),
    ([20000], 32, 8, 128, 32),
    ([1, 15, 16, 17, 31], 8, 2, 128, 16),
]


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("frac", [0.0, 0.1, 0.5, 1.0])
@pytest.mark.parametrize("coldest", [True, False])
def test_offload_parity_and_placement_bit_identity(oracle, case, frac, coldest):
    lens, hq, hkv, d, ps = case
    b = W.make_batch(lens, hq, hkv, d, ps, seed=601, device=DEV, poison_unused=True)
    ref_out, ref_lse = gpu_run(b)
    torch.cuda.synchronize()
    ob = W.offload_pages(b, frac, seed=17, coldest_first=coldest)
    out, lse = run_offload(ob)
    assert torch.equal(bits(out), bits(ref_out)), "placement changed the bits"
    assert torch.equal(lse.view(torch.int32), ref_lse.view(torch.int32))
    c = W.combined_pool_cpu(ob)
    ref, ref_l = oracle.decode_attn(c.q, c.k_pages, c.v_pages, c.block_table, c.seq_lens, c.softmax_scale)
    pairs = all_pairs(b)
    err = errors(out, ref.reshape(len(pairs), -1), pairs)
    assert_parity(err, f"offload {frac} {case}")


@pytest.mark.parametrize("flags", [0, comem.COMEM_LAUNCH_KV_PREFIX_IMMUTABLE | comem.COMEM_LAUNCH_Q_STABLE])
@pytest.mark.parametrize("grid", [None, 7, 64])
def test_offload_grids_and_early_mode(grid, flags):
    b = W.make_batch([12000, 600, 0, 31], 32, 4, 128, 16, seed=602, device=DEV, poison_unused=True)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    ref = torch.empty_like(b.q)
    comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, ref, ws, grid_ctas=grid)
    ob = W.offload_pages(b, 0.3, seed=5, coldest_first=False)
    for _ in range(3):
        out, _ = run_offload(ob, flags=flags, grid=grid)
        assert torch.equal(bits(out), bits(ref))


def test_offload_rejects_unpinned_host_pool():
    b = W.make_batch([100], 8, 2, 128, 16, seed=603, device=DEV)
    ob = W.offload_pages(b, 0.5, seed=1)
    lib = comem.load_library()
    import ctypes
    kh = torch.zeros_like(ob.k_host)  # pageable
    out = torch.empty_like(b.q)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table)
    st = lib.comem_decode_attn_offload_async(
        b.q.data_ptr(), b.k_pages.data_ptr(), b.v_pages.data_ptr(), kh.data_ptr(), ob.v_host.data_ptr(),
        b.block_table.data_ptr(), b.seq_lens.data_ptr(), 8, 2, 128, 16, ctypes.c_float(b.softmax_scale), out.data_ptr(), 1,
        b.block_table.shape[1], b.num_pages, kh.shape[0], None, ws.data_ptr(), ws.numel() * ws.element_size(), None, None)
    assert st == comem.COMEM_ERR_INVALID_ARG


def test_pages_copy_roundtrip_and_offload_then_attend(oracle):
    """Offload the coldest pages with the library's migration kernel, attend over the two tiers, bring them back."""
    b = W.make_batch([6000, 900], 32, 8, 128, 16, seed=604, device=DEV, poison_unused=True)
    ref_out, _ = gpu_run(b)
    ps = b.page_size
    n0 = 100  # coldest pages of sequence 0
    src = b.block_table[0, :n0].clone()
    dst = torch.arange(n0, dtype=torch.int32, device=DEV)
    k_host = torch.zeros((n0,) + tuple(b.k_pages.shape[1:]), dtype=torch.bfloat16).pin_memory()
    v_host = torch.zeros_like(k_host).pin_memory()
    comem.comem_pages_copy_async(b.k_pages, b.v_pages, k_host, v_host, src, dst)
    torch.cuda.synchronize()
    assert torch.equal(bits(k_host), bits(b.k_pages[src.long()].cpu())) and torch.equal(bits(v_host), bits(b.v_pages[src.long()].cpu()))
    bt = b.block_table.clone()
    bt[0, :n0] = -1 - dst
    kd, vd = b.k_pages.clone(), b.v_pages.clone()
    kd[src.long()] = float("nan")
    vd[src.long()] = float("nan")
    out = torch.empty_like(b.q)
    ws = comem.alloc_workspace(b.q, kd, bt)
    comem.comem_decode_attn_offload_async(b.q, kd, vd, k_host, v_host, bt, b.seq_lens, b.softmax_scale, out, ws)
    torch.cuda.synchronize()
    assert torch.equal(bits(out), bits(ref_out))
    comem.comem_pages_copy_async(k_host, v_host, kd, vd, dst, src)   # bring them back
    torch.cuda.synchronize()
    assert torch.equal(bits(kd[src.long()]), bits(b.k_pages[src.long()])) and torch.equal(bits(vd[src.long()]), bits(b.v_pages[src.long()]))
