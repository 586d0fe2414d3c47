"""Shared helpers for the GPU parity tests: run the CUDA path through the C-ABI binding, run the
fp64 oracle on THE SAME BITS, and measure the error against the written tolerances.

Tolerances:
  contract gate (BASELINE.json north_star): max|d| <= 2e-2 and mean|d| <= 2e-3;
  scale-aware gate (the contract gate alone would accept an all-zero output at 32K+ context):
      rel_l2 = ||gpu - oracle||_2 / ||oracle||_2 <= 5e-3
      max|d| <= 4 * 2^-9 * max|oracle| + 1e-6
"""
import numpy as np
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W

MAX_ABS, MEAN_ABS, REL_L2 = 2e-2, 2e-3, 5e-3


def gpu_run(batch: W.DecodeBatch, want_lse: bool = True, stream=None, workspace=None, flags: int = 0):
    """One decode-attention step through the C-ABI on the current device. Returns (out, lse) tensors."""
    assert batch.q.is_cuda
    out = torch.full_like(batch.q, float("nan"))
    lse = torch.full((batch.batch, batch.num_q_heads), float("nan"), dtype=torch.float32,
                     device=batch.q.device) if want_lse else None
    ws = workspace if workspace is not None else comem.alloc_workspace(batch.q, batch.k_pages, batch.block_table,
                                                                        stream=stream)
    comem.comem_decode_attn_async(batch.q, batch.k_pages, batch.v_pages, batch.block_table,
                                  batch.seq_lens, batch.softmax_scale, out, ws, lse_out=lse, stream=stream, flags=flags)
    return out, lse


def compact_rows_to_cpu(batch: W.DecodeBatch, seqs):
    """Gather the pages of the sequences in `seqs` into a small pool (identity block table) on the
    CPU, so the oracle can run on full-size configs without an 18 GB copy.  Pure data movement; the
    oracle's indifference to physical placement is pin O9."""
    ps = batch.page_size
    lens = batch.seq_lens.cpu()
    ids, rows, off = [], [], 0
    maxp = max(1, max(W.pages_needed(int(lens[b]), ps) for b in seqs))
    bt = torch.zeros((len(seqs), maxp), dtype=torch.int32)
    for i, b in enumerate(seqs):
        n = W.pages_needed(int(lens[b]), ps)
        ids.append(batch.block_table[b, :n].to(torch.int64))
        bt[i, :n] = torch.arange(off, off + n, dtype=torch.int32)
        off += n
    ids = torch.cat(ids) if ids else torch.zeros(0, dtype=torch.int64)
    if ids.numel() == 0:
        kp = torch.zeros((1, ps, batch.num_kv_heads, batch.head_dim), dtype=torch.bfloat16)
        vp = kp.clone()
    else:
        kp = batch.k_pages[ids.to(batch.k_pages.device)].cpu()
        vp = batch.v_pages[ids.to(batch.v_pages.device)].cpu()
    sel = torch.tensor(list(seqs), dtype=torch.int64)
    return W.DecodeBatch(q=batch.q.cpu()[sel], k_pages=kp, v_pages=vp, block_table=bt,
                         seq_lens=lens[sel].contiguous(), softmax_scale=batch.softmax_scale)


def oracle_rows(oracle, batch: W.DecodeBatch, pairs):
    """Oracle out/lse for the (b, h) rows in `pairs` (list) on the same bits as `batch`."""
    seqs = sorted({b for b, _ in pairs})
    sub = compact_rows_to_cpu(batch, seqs)
    remap = {b: i for i, b in enumerate(seqs)}
    sub_pairs = [(remap[b], h) for b, h in pairs]
    return oracle.decode_attn(sub.q, sub.k_pages, sub.v_pages, sub.block_table, sub.seq_lens,
                              sub.softmax_scale, pairs=sub_pairs)


def all_pairs(batch):
    return [(b, h) for b in range(batch.batch) for h in range(batch.num_q_heads)]


def errors(gpu_out: torch.Tensor, ref: np.ndarray, pairs):
    g = np.stack([gpu_out[b, h].double().cpu().numpy() for b, h in pairs])
    d = np.abs(g - ref)
    return {"max_abs": float(d.max()), "mean_abs": float(d.mean()),
            "rel_l2": float(np.linalg.norm(g - ref) / max(np.linalg.norm(ref), 1e-300)),
            "max_ref": float(np.abs(ref).max()), "finite": bool(np.isfinite(g).all())}


def assert_parity(err, what=""):
    assert err["finite"], (what, err)
    assert err["max_abs"] <= MAX_ABS, (what, err)
    assert err["mean_abs"] <= MEAN_ABS, (what, err)
    assert err["rel_l2"] <= REL_L2, (what, err)
    assert err["max_abs"] <= 4 * 2.0 ** -9 * err["max_ref"] + 1e-6, (what, err)


def check_batch(oracle, batch: W.DecodeBatch, pairs=None, what="", lse_tol=2e-4, flags: int = 0):
    out, lse = gpu_run(batch, flags=flags)
    torch.cuda.synchronize()
    pairs = pairs if pairs is not None else all_pairs(batch)
    ref, ref_lse = oracle_rows(oracle, batch, pairs)
    err = errors(out, ref, pairs)
    assert_parity(err, what)
    glse = np.array([float(lse[b, h]) for b, h in pairs])
    live = np.isfinite(ref_lse)
    assert np.array_equal(np.isneginf(glse), np.isneginf(ref_lse)), what
    if live.any():
        assert np.max(np.abs(glse[live] - ref_lse[live]) / np.maximum(1.0, np.abs(ref_lse[live]))) <= lse_tol, what
    return out, lse, err
