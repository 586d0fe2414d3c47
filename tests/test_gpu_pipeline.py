"""SURVEY.md §8(f).4 on the GPU: two batches sharing the device by SM partition (comem_set_grid_ctas per
enqueue, programmatic launch off) give, bit for bit, what each gives alone with the same grid, and agree with
the oracle; the plan's context lengths drive the agent's seq_lens."""
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
    ga, gm = sms // 2, sms - sms // 2
    steps = [t for t in range(12) if mem[t]]
    assert steps, "the plan launches memory jobs"

    def run(step, concurrent):
        la = torch.full((4,), ctx[min(step + 1, 11)], dtype=torch.int32, device=DEV)
        lm = torch.full((4,), mem[step], dtype=torch.int32, device=DEV)
        oa, om = torch.full_like(agent.q, float("nan")), torch.full_like(memory.q, float("nan"))
        torch.cuda.synchronize()
        comem.comem_set_grid_ctas(gm)
        comem.comem_decode_attn_async(memory.q, memory.k_pages, memory.v_pages, memory.block_table, lm,
                                      memory.softmax_scale, om, ws_m, stream=sb)
        if not concurrent:
            torch.cuda.synchronize()
        comem.comem_set_grid_ctas(ga)
        comem.comem_decode_attn_async(agent.q, agent.k_pages, agent.v_pages, agent.block_table, la,
                                      agent.softmax_scale, oa, ws_a, stream=sa)
        torch.cuda.synchronize()
        return oa, om, la

    try:
        comem.comem_set_programmatic_launch(False)
        for step in steps:
            a1, m1, la = run(step, concurrent=False)
            a2, m2, _ = run(step, concurrent=True)
            assert torch.equal(bits(a1), bits(a2)) and torch.equal(bits(m1), bits(m2)), step
            import dataclasses
            pairs = [(0, 0), (1, 17), (3, 63)]
            ref, _ = oracle_rows(oracle, dataclasses.replace(agent, seq_lens=la), pairs)
            assert_parity(errors(a2, ref, pairs), f"agent step {step}")
    finally:
        comem.comem_set_grid_ctas(0)
        comem.comem_set_programmatic_launch(True)
