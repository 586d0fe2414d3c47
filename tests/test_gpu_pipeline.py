"""SURVEY.md §8(f).4 on the GPU: two batches sharing the device by SM partition (per-call comem_launch_opts:
grid_ctas from comem_sm_partition, programmatic launch off) give, bit for bit, what each gives alone with the same
grid, and agree with the oracle; the plan's context lengths drive the agent's seq_lens; two host threads enqueueing
different grids concurrently do not disturb each other."""
import threading

import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from paper_2605_30842_b200 import workloads as W
from parity_util import assert_parity, errors, oracle_rows

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t):
    return t.contiguous().view(torch.int16)


def test_sm_partitioned_streams_match_serial_and_oracle(oracle):
    arr, ev = comem.comem_kstep_plan(12, 3, 0)
    ctx, full, mem = comem.comem_kstep_context_lengths(arr, 12, 160, 700)
    agent = W.make_batch([max(full)] * 4, 64, 8, 128, 16, seed=901, device=DEV)
    memory = W.make_batch([max(full)] * 4, 32, 8, 128, 16, seed=902, device=DEV)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ws_a = comem.alloc_workspace(agent.q, agent.k_pages, agent.block_table, stream=sa)
    ws_m = comem.alloc_workspace(memory.q, memory.k_pages, memory.block_table, stream=sb)
    sms = comem.comem_grid_ctas(128)
    ga, gm = comem.comem_sm_partition(agent.algorithmic_bytes(), memory.algorithmic_bytes(), sms)
    assert ga + gm == sms and ga >= gm >= 8       # the agent batch (64 query heads' Q, same KV bytes) is no smaller
    steps = [t for t in range(12) if mem[t]]
    assert steps, "the plan launches memory jobs"

    def run(step, concurrent):
        la = torch.full((4,), ctx[min(step + 1, 11)], dtype=torch.int32, device=DEV)
        lm = torch.full((4,), mem[step], dtype=torch.int32, device=DEV)
        oa, om = torch.full_like(agent.q, float("nan")), torch.full_like(memory.q, float("nan"))
        torch.cuda.synchronize()
        comem.comem_decode_attn_async(memory.q, memory.k_pages, memory.v_pages, memory.block_table, lm,
                                      memory.softmax_scale, om, ws_m, stream=sb, grid_ctas=gm, programmatic_launch=False)
        if not concurrent:
            torch.cuda.synchronize()
        comem.comem_decode_attn_async(agent.q, agent.k_pages, agent.v_pages, agent.block_table, la,
                                      agent.softmax_scale, oa, ws_a, stream=sa, grid_ctas=ga, programmatic_launch=False)
        torch.cuda.synchronize()
        return oa, om, la

    for step in steps:
        a1, m1, la = run(step, concurrent=False)
        a2, m2, _ = run(step, concurrent=True)
        assert torch.equal(bits(a1), bits(a2)) and torch.equal(bits(m1), bits(m2)), step
        import dataclasses
        pairs = [(0, 0), (1, 17), (3, 63)]
        ref, _ = oracle_rows(oracle, dataclasses.replace(agent, seq_lens=la), pairs)
        assert_parity(errors(a2, ref, pairs), f"agent step {step}")


def test_two_host_threads_with_different_grids_bit_identical_to_serial():
    """Launch options are per call (comem_launch_opts), not process state: two engines' threads (the paper's
    deployment) enqueue 40 steps each with DIFFERENT grid sizes at the same time; every output is
    bit-identical to the same call made alone with that grid."""
    a = W.make_batch([5000, 1200, 77], 64, 8, 128, 16, seed=911, device=DEV)
    m = W.make_batch([9000, 300], 32, 8, 128, 16, seed=912, device=DEV)
    sms = comem.comem_grid_ctas(128)
    jobs = [(a, 37, torch.cuda.Stream()), (m, sms - 37, torch.cuda.Stream())]
    want = []
    for b, grid, st in jobs:
        ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table, stream=st)
        o = torch.empty_like(b.q)
        comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale, o, ws,
                                      stream=st, grid_ctas=grid, programmatic_launch=False)
        torch.cuda.synchronize()
        want.append((o, ws))
    outs = [[torch.empty_like(b.q) for _ in range(40)] for b, _, _ in jobs]
    errs = []

    def worker(i):
        try:
            b, grid, st = jobs[i]
            torch.cuda.set_device(b.q.device)
            for o in outs[i]:
                comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                              o, want[i][1], stream=st, grid_ctas=grid, programmatic_launch=False)
        except Exception as e:  # noqa: BLE001
            errs.append(e)

    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    assert not errs, errs
    for i in range(2):
        for o in outs[i]:
            assert torch.equal(bits(o), bits(want[i][0]))
