"""GPU parity at BASELINE.json's FULL sizes (configs C2..C5), in the launch configuration bench.py
times (default persistent grid, fused combine).  The oracle runs on sampled whole sequences (all
their query heads) -- it computes each row one by one from the same bits -- and the properties that
hold at any size (page-permutation bit-identity, run-to-run bit-identity, overlap == serial replay)
are checked on the complete outputs.  Input recipes: DESIGN.md "Input recipe"."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import compact_rows_to_cpu, assert_parity, errors, gpu_run, oracle_rows

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t: torch.Tensor) -> torch.Tensor:
    return t.contiguous().view(torch.int16)


def seq_pairs(batch, seqs):
    return [(b, h) for b in seqs for h in range(batch.num_q_heads)]


def sample_seqs(lens, k):
    """shortest, longest and k-2 evenly spaced others (deterministic)."""
    order = sorted(range(len(lens)), key=lambda i: (lens[i], i))
    if len(order) <= k:
        return sorted(order)
    pick = {order[0], order[-1]}
    for j in range(1, k - 1):
        pick.add(order[j * (len(order) - 1) // (k - 1)])
    return sorted(pick)


def check_sampled(oracle, batch, seqs, what):
    out, lse = gpu_run(batch)
    torch.cuda.synchronize()
    pairs = seq_pairs(batch, seqs)
    ref, ref_lse = oracle_rows(oracle, batch, pairs)
    err = errors(out, ref, pairs)
    assert_parity(err, what)
    glse = np.array([float(lse[b, h]) for b, h in pairs])
    assert np.max(np.abs(glse - ref_lse) / np.maximum(1.0, np.abs(ref_lse))) <= 2e-4, what
    assert torch.isfinite(out.float()).all(), what
    print(what, err)
    return out, lse


def test_c2_full(oracle):
    """C2: all 64 rows against the oracle; unused half of the 4096-page pool NaN-poisoned;
    bit-identical under two physical page permutations and over 5 repeats."""
    b = W.config2_agent_single(DEV, poison_unused=True)
    out, lse = check_sampled(oracle, b, [0], "C2")
    for _ in range(5):
        o, l = gpu_run(b)
        assert torch.equal(bits(o), bits(out)) and torch.equal(l, lse)
    for s in (11, 12):
        o, l = gpu_run(W.permute_pages(b, seed=s))
        assert torch.equal(bits(o), bits(out)) and torch.equal(l, lse)


def test_c3_full(oracle):
    """C3: 32 ragged sequences in one shuffled pool; ALL 32 sequences (2 048 rows) against the oracle;
    the complete output bit-identical under a page permutation."""
    b = W.config3_agent_ragged(DEV, poison_unused=True)
    lens = b.seq_lens.cpu().tolist()
    assert len(lens) == 32 and min(lens) >= 8192 and max(lens) <= 65536
    out, lse = check_sampled(oracle, b, list(range(32)), "C3")
    o, l = gpu_run(W.permute_pages(b, seed=13))
    assert torch.equal(bits(o), bits(out)) and torch.equal(l, lse)


def test_c4_full(oracle):
    """C4: 16 x 131072 tokens, page 32, K pool > 4 GiB (64-bit offsets), 1 % peaked keys;
    ALL 16 sequences (512 rows) against the oracle; run-to-run bit-identity on all rows."""
    b = W.config4_memory_long(DEV, poison_unused=True)
    assert b.k_pages.numel() * 2 > 2 ** 32
    out, lse = check_sampled(oracle, b, list(range(16)), "C4")
    o, l = gpu_run(b)
    assert torch.equal(bits(o), bits(out)) and torch.equal(l, lse)


# ---- C5: k-step-off overlap, two batches on two streams, 64 decode steps with appends -------------
ORACLE_STEPS = (0, 1, 2, 15, 16, 17, 31, 32, 63)
N_STEPS = 64


def _c5_batches():
    agent = W.config3_agent_ragged(DEV, spare_tokens=N_STEPS)
    memory = W.config5_memory_ragged(DEV, spare_tokens=N_STEPS)
    return agent, memory


def _c5_rows(batch, seed_base):
    return [W.decode_step_rows(batch, i, seed_base) for i in range(N_STEPS)]


def _c5_run(agent, memory, rows_a, rows_m, stream_a, stream_m):
    """64 steps of (append, attend) per batch; the two batches on the given streams (the same
    stream twice = serial replay).  Returns per-step outputs [64][B, Hq, D] for both."""
    torch.cuda.synchronize()
    ws_a = comem.alloc_workspace(agent.q, agent.k_pages, agent.block_table, stream=stream_a)
    ws_m = comem.alloc_workspace(memory.q, memory.k_pages, memory.block_table, stream=stream_m)
    outs_a = torch.empty((N_STEPS,) + tuple(agent.q.shape), dtype=torch.bfloat16, device=DEV)
    outs_m = torch.empty((N_STEPS,) + tuple(memory.q.shape), dtype=torch.bfloat16, device=DEV)
    torch.cuda.synchronize()
    for i in range(N_STEPS):
        for b, rows, outs, ws, st in ((agent, rows_a, outs_a, ws_a, stream_a),
                                      (memory, rows_m, outs_m, ws_m, stream_m)):
            q, nk, nv = rows[i]
            comem.comem_kv_append_async(b.k_pages, b.v_pages, b.block_table, b.seq_lens, nk, nv, stream=st)
            comem.comem_decode_attn_async(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                          b.softmax_scale, outs[i], ws, stream=st)
    torch.cuda.synchronize()
    return outs_a, outs_m


def test_c5_overlap_two_streams(oracle):
    agent, memory = _c5_batches()
    len_a0, len_m0 = agent.seq_lens.clone(), memory.seq_lens.clone()
    rows_a, rows_m = _c5_rows(agent, 1005_000), _c5_rows(memory, 1005_500)
    sa, sm = torch.cuda.Stream(), torch.cuda.Stream()
    outs_a, outs_m = _c5_run(agent, memory, rows_a, rows_m, sa, sm)
    assert torch.equal(agent.seq_lens, len_a0 + N_STEPS) and torch.equal(memory.seq_lens, len_m0 + N_STEPS)

    # oracle at the steps that straddle page boundaries, on sampled sequences.  The final cache
    # holds every appended row; step i's attention saw the first L_b + i + 1 tokens of it (the
    # oracle ignores what lies past seq_len: pin O12).
    for name, b, l0, rows, outs, k in (("agent", agent, len_a0, rows_a, outs_a, 32),
                                       ("memory", memory, len_m0, rows_m, outs_m, 8)):
        seqs = list(range(k))        # all 40 sequences at every listed step
        pairs = seq_pairs(b, seqs)
        sub = compact_rows_to_cpu(b, seqs)          # the final cache, gathered to the CPU once
        for i in ORACLE_STEPS:
            ref, _ = oracle.decode_attn(rows[i][0].cpu(), sub.k_pages, sub.v_pages, sub.block_table,
                                        (l0.cpu() + i + 1).to(torch.int32), b.softmax_scale)
            ref = ref.reshape(len(pairs), -1)
            assert_parity(errors(outs[i], ref, pairs), f"C5 {name} step {i}")

    # all 64 steps of all 40 sequences: the overlapped run equals a serial single-stream replay, bit for bit
    del agent, memory
    torch.cuda.empty_cache()
    agent2, memory2 = _c5_batches()
    s1 = torch.cuda.Stream()
    outs_a2, outs_m2 = _c5_run(agent2, memory2, rows_a, rows_m, s1, s1)
    assert torch.equal(bits(outs_a), bits(outs_a2))
    assert torch.equal(bits(outs_m), bits(outs_m2))
