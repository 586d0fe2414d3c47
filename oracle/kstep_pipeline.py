"""oracle/kstep_pipeline.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain Python statement of the paper's k-step-off pipeline schedule (Algorithm 1) and of
its latency model (eq. 5-7), followed line by line in the paper's order and notation.
Only tests/ and bench.py's reference legs may import this; it shares nothing with the C-ABI library.

Readings (R19, where the paper is silent):
  * "P_mem is complete" (Alg. 1 line 4): the job launched after step t0 is complete at the synchronisation
    point of step t0 + d, d = `mem_delay` agent steps.  The text fixes the default: "Upon completion, the new
    summary becomes available at the start of the next cycle" (L122) -> d = k.  1 <= d <= k is required, so
    that line 20 never overwrites a job still in flight (the paper does not say what happens then).
  * KV cache validity (Alg. 1 lines 9-13): invalid before the first step (nothing is cached) and after every
    adoption of a new summary (line 5); valid after any prefill.
  * what the agent's context holds at step t (eq. 4): the summary s = f(tau_{<=u}) (u = the step after
    which the adopted job was launched; s = {} while u = 0) plus the raw turns tau_{u+1 : t}.

Pins (tests/test_oracle_pipeline_pins.py): the paper's own statements about 1-step-off and 2-step-off
(L176, Fig. 4 caption), eq. 4's summary / buffer split at every adoption step, the case study's printed numbers
(L199: ratio < 0.23, 7.36K tokens of a 32K prefix), eq. 6 <=> eq. 7 on a grid.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Sequence


@dataclass
class StepEvent:
    step: int               # t, 1-based as in Algorithm 1
    adopt_summary: bool     # lines 4-7: P_mem complete -> s <- result, KV cache invalidated
    summary_upto: int       # u: the summary in use covers tau_{<= u}; 0 = no summary yet
    prefill_uncached: bool  # lines 9-13: False = cached (new tokens only), True = full context (s, tau_{u+1:t})
    launch_memory: bool     # lines 19-21: t mod k = 0 -> P_mem <- async f(tau_{<= t})


def kstep_plan(num_steps: int, k: int, mem_delay: int | None = None) -> List[StepEvent]:
    """Algorithm 1 for t = 1 .. num_steps."""
    if num_steps < 0 or k < 1:
        raise ValueError("num_steps >= 0 and k >= 1")
    d = k if mem_delay is None else mem_delay
    if not 1 <= d <= k:
        raise ValueError("1 <= mem_delay <= k")
    events = []
    summary_upto = 0          # line 1: s <- {}
    p_mem = None              # line 1: P_mem <- None; else (launched_after_step, covers_upto)
    kv_valid = False
    t = 1
    while t <= num_steps:     # line 2
        adopt = False
        if p_mem is not None and t >= p_mem[0] + d:   # line 4: P_mem is complete
            summary_upto = p_mem[1]                   # line 5: s <- result(P_mem); invalidate KV cache
            kv_valid = False
            p_mem = None                              # line 6
            adopt = True
        uncached = not kv_valid                       # lines 9-13
        kv_valid = True
        # lines 14-17: decode a_t, execute, tau_{t+1} <- tau_t U {a_t, o_{t+1}}: nothing to schedule
        launch = (t % k == 0)                         # line 19
        if launch:
            p_mem = (t, t)                            # line 20: async f(tau_{<= t})
        events.append(StepEvent(t, adopt, summary_upto, uncached, launch))
        t += 1                                        # line 22
    return events


def context_lengths(events: Sequence[StepEvent], turn_tokens: int, summary_tokens: int):
    """Token counts per step, with every turn tau_i worth `turn_tokens` tokens and every summary
    `summary_tokens` tokens.  Returns (comem_ctx, full_ctx, memory_input): the agent's context under CoMem
    (summary + raw turns tau_{u+1 : t}, eq. 4), under the full-context baseline (tau_{<= t}), and the memory
    model's input when it is launched after step t (tau_{<= t}; 0 if no launch)."""
    comem, full, mem = [], [], []
    for e in events:
        s = summary_tokens if e.summary_upto > 0 else 0
        comem.append(s + (e.step - e.summary_upto) * turn_tokens)
        full.append(e.step * turn_tokens)
        mem.append(e.step * turn_tokens if e.launch_memory else 0)
    return comem, full, mem


# ---- eq. 5-7: S in GB per token, W in GB/s, P in tokens/s -------------------------------
def decode_saving_s(l_full: float, l_sum: float, s_gb: float, w_gbs: float) -> float:
    """eq. 5: per-token decode latency saved, (L_full - L_sum) * S / W."""
    return (l_full - l_sum) * s_gb / w_gbs


def net_speedup(y: float, l_full: float, l_sum: float, s_gb: float, w_gbs: float, p_tok_s: float) -> bool:
    """eq. 6: Y * (L_full - L_sum) * S / W  >  L_sum / P."""
    return y * decode_saving_s(l_full, l_sum, s_gb, w_gbs) > l_sum / p_tok_s


def max_compression_ratio(w_gbs: float, y: float, s_gb: float, p_tok_s: float) -> float:
    """eq. 7: L_sum / L_full  <  1 / (1 + W / (Y * S * P))."""
    return 1.0 / (1.0 + w_gbs / (y * s_gb * p_tok_s))
