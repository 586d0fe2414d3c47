"""The library's Algorithm-1 step scheduler (comem_kstep_step_async):
  * the context it gives the agent at every step is the oracle's (oracle/kstep_pipeline.py: eq. 4), and the prefill
    it enqueues is cached / uncached as the oracle's plan says;
  * what it computes is bit-identical to the same sequence of plain API calls (the scheduler holds no arithmetic);
  * the attention outputs of the last step match the fp64 attention oracles on the final cache state;
  * a memory job runs on the second stream behind the agent's step and both models' results are unchanged by it."""
import numpy as np
import pytest
import torch

import paper_2605_30842_b200 as comem
from oracle import kstep_pipeline as KP
from paper_2605_30842_b200 import workloads as W
from parity_util import MAX_ABS, MEAN_ABS

pytestmark = pytest.mark.gpu
DEV = "cuda"


def bits(t):
    return t.contiguous().view(torch.int16)


def build_model(batch, hq, hkv, d, ps, max_ctx, seed):
    b = W.make_batch([max_ctx] * batch, hq, hkv, d, ps, seed, DEV)
    gen = torch.Generator(device=DEV)
    gen.manual_seed(seed + 1)
    t = {"b": b,
         "q_decode": b.q, "out_decode": torch.zeros_like(b.q),
         "q_prefill": (torch.randn((batch * max_ctx, hq, d), generator=gen, device=DEV)).to(torch.bfloat16),
         "new_k": torch.randn((batch, hkv, d), generator=gen, device=DEV).to(torch.bfloat16),
         "new_v": torch.randn((batch, hkv, d), generator=gen, device=DEV).to(torch.bfloat16),
         "q_start": torch.zeros(batch + 1, dtype=torch.int32, device=DEV),
         "ws": comem.alloc_workspace(b.q, b.k_pages, b.block_table)}
    t["out_prefill"] = torch.zeros_like(t["q_prefill"])
    t["model"] = comem.kstep_model(t["q_decode"], t["out_decode"], t["q_prefill"], t["out_prefill"], t["new_k"], t["new_v"],
                                   b.k_pages, b.v_pages, b.block_table, b.seq_lens, t["q_start"], t["ws"], b.softmax_scale)
    return t


@pytest.mark.parametrize("k", [1, 3])
def test_scheduler_follows_the_oracle_plan_and_equals_plain_calls(oracle, k):
    T, TURN, SUMM, Y, YM, B = 7, 48, 40, 3, 2, 2
    max_ctx = T * TURN + 16
    agent = build_model(B, 16, 2, 128, 16, max_ctx, 701)
    memory = build_model(B, 8, 2, 128, 16, max_ctx, 702)
    twin = build_model(B, 16, 2, 128, 16, max_ctx, 701)       # same bits: re-enacted with plain API calls
    arr, events = comem.comem_kstep_plan(T, k, 0)
    want = KP.kstep_plan(T, k)
    ctx_want, _, mem_want = KP.context_lengths(want, TURN, SUMM)
    sa, sm = torch.cuda.Stream(), torch.cuda.Stream()
    ev_done, ev_step = torch.cuda.Event(), torch.cuda.Event()
    ev_done.record(sm)
    ev_step.record(sa)
    torch.cuda.synchronize()
    for i, e in enumerate(events):
        stats = comem.comem_kstep_step_async(e, TURN, SUMM, Y, YM, agent["model"], memory["model"], sa, sm, ev_done, ev_step)
        torch.cuda.synchronize()
        assert stats.agent_ctx == ctx_want[i]
        assert stats.agent_prefill_tokens == (ctx_want[i] if want[i].prefill_uncached else min(TURN, ctx_want[i]))
        assert stats.memory_ctx == mem_want[i]
        assert agent["b"].seq_lens.tolist() == [ctx_want[i] + Y] * B        # the Y decoded tokens were appended
        if mem_want[i]:
            assert memory["b"].seq_lens.tolist() == [mem_want[i] + YM] * B
        # the same step with plain calls on the twin
        tb = twin["b"]
        n_new = stats.agent_prefill_tokens
        tb.seq_lens.fill_(ctx_want[i])
        twin["q_start"].copy_(torch.arange(B + 1, dtype=torch.int32, device=DEV) * n_new)
        comem.comem_prefill_attn_async(twin["q_prefill"][: B * n_new], tb.k_pages, tb.v_pages, tb.block_table, tb.seq_lens,
                                       twin["q_start"], tb.softmax_scale, twin["out_prefill"][: B * n_new])
        for _ in range(Y):
            comem.comem_kv_append_async(tb.k_pages, tb.v_pages, tb.block_table, tb.seq_lens, twin["new_k"], twin["new_v"])
            comem.comem_decode_attn_async(twin["q_decode"], tb.k_pages, tb.v_pages, tb.block_table, tb.seq_lens,
                                          tb.softmax_scale, twin["out_decode"], twin["ws"])
        torch.cuda.synchronize()
        assert torch.equal(bits(agent["out_decode"]), bits(twin["out_decode"])), i
        assert torch.equal(bits(agent["out_prefill"][: B * n_new]), bits(twin["out_prefill"][: B * n_new])), i
        assert torch.equal(bits(agent["b"].k_pages), bits(tb.k_pages))
    # oracle parity of the last step's outputs on the final cache state
    ab = agent["b"]
    ref, _ = oracle.decode_attn(ab.q.cpu(), ab.k_pages.cpu(), ab.v_pages.cpu(), ab.block_table.cpu(), ab.seq_lens.cpu(),
                                ab.softmax_scale)
    d = np.abs(agent["out_decode"].double().cpu().numpy() - ref)
    assert d.max() <= MAX_ABS and d.mean() <= MEAN_ABS


def test_scheduler_rejects_bad_arguments():
    agent = build_model(1, 8, 2, 128, 16, 64, 703)
    arr, events = comem.comem_kstep_plan(4, 2, 0)
    s = torch.cuda.Stream()
    with pytest.raises(comem.ComemError) as ei:   # the context does not fit the block-table row
        comem.comem_kstep_step_async(events[3], 48, 40, 1, 0, agent["model"], None, s)
    assert ei.value.status == comem.COMEM_ERR_INVALID_ARG
    with pytest.raises(comem.ComemError):
        comem.comem_kstep_step_async(events[0], 0, 40, 1, 0, agent["model"], None, s)
