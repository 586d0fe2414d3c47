"""Pins of oracle/kstep_pipeline.py (Algorithm 1 and eq. 5-7 of the paper; reading R19) against
what the paper itself prints:
  P1  1-step-off: "every step after the first requires uncached prefilling" (Fig. 4 caption)
  P2  2-step-off: "the uncached prefill occurs only once per cycle, with the intermediate step reusing the
      cached KV prefix" (same caption); k-step-off: one uncached prefill per cycle of k steps (L122)
  P3  eq. 4 (L126) at every adoption step t: summary = f(tau_{<= t-k}), buffer = tau_{t-k+1 : t}; the memory
      model is launched every k steps on tau_{<= t} (Alg. 1 lines 19-20)
  P4  the case study (L199): W = 2 TB/s, P = 3000 tok/s, S = 2e-4 GB, Y = 1000 -> L_sum / L_full < 0.23,
      i.e. 7.36K tokens of a 32K prefix
  P5  eq. 6 holds exactly when L_sum / L_full is below eq. 7's bound (grid; the rearrangement, L195-197)
  P6  eq. 5 is linear in L_full - L_sum and equals one token's KV bytes over the bandwidth
  P7  context lengths: CoMem's prompt stays bounded (summary + at most 2k - 1 raw turns) while the
      full-context prompt grows linearly (section 4.5)
"""
import math

import pytest

from oracle import kstep_pipeline as KP


def test_p1_one_step_off_every_step_uncached():
    ev = KP.kstep_plan(20, 1)
    assert all(e.prefill_uncached for e in ev)
    assert all(e.adopt_summary for e in ev[1:]) and not ev[0].adopt_summary
    assert all(e.launch_memory for e in ev)


@pytest.mark.parametrize("k", [2, 3, 4, 7])
def test_p2_one_uncached_prefill_per_cycle(k):
    ev = KP.kstep_plan(10 * k, k)
    assert ev[0].prefill_uncached                                  # nothing cached before the first step
    for c in range(2, 10):                                         # first launch after step k -> adopted at step 2k
        cyc = ev[c * k - 1:(c + 1) * k - 1]                        # steps c*k .. (c+1)*k - 1
        assert [e.prefill_uncached for e in cyc] == [True] + [False] * (k - 1)
    assert sum(e.prefill_uncached for e in ev[1:2 * k - 1]) == 0   # steps 2 .. 2k-1: no summary yet, cache reused


@pytest.mark.parametrize("k", [1, 2, 3, 5])
def test_p3_eq4_summary_and_buffer_split(k):
    ev = KP.kstep_plan(6 * k + 2, k)
    for e in ev:
        assert e.launch_memory == (e.step % k == 0)
        if e.adopt_summary:
            assert e.step % k == 0 and e.summary_upto == e.step - k   # f(tau_{<= t-k}); buffer tau_{t-k+1 : t}
            assert e.prefill_uncached
        assert 0 <= e.summary_upto <= max(0, e.step - k)
        assert e.step - e.summary_upto <= 2 * k - 1 or e.summary_upto == 0


def test_p3_shorter_memory_job_is_adopted_earlier():
    ev = KP.kstep_plan(12, 3, mem_delay=1)
    adopt = [e.step for e in ev if e.adopt_summary]
    assert adopt == [4, 7, 10] and [ev[s - 1].summary_upto for s in adopt] == [3, 6, 9]
    with pytest.raises(ValueError):
        KP.kstep_plan(12, 3, mem_delay=4)


def _golden_case_study():
    """tests/golden/eq7_case_study.txt: the values the paper prints, key=value lines."""
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "eq7_case_study.txt")) as fh:
        for line in fh:
            if "=" in line and not line.startswith("#"):
                k, v = line.strip().split("=")
                vals[k] = float(v)
    return vals


def test_p4_case_study_numbers():
    g = _golden_case_study()
    r = KP.max_compression_ratio(w_gbs=g["W_GBps"], y=g["Y_tokens"], s_gb=g["S_GB_per_tok"], p_tok_s=g["P_tok_s"])
    assert abs(r - 1.0 / (1.0 + 2000.0 / 600.0)) < 1e-15
    assert round(r, 2) == g["ratio_printed"]                        # "L_sum / L_full < 0.23"
    assert abs(g["ratio_printed"] * 32000 - g["summary_tokens_printed"]) < 1e-9   # "within 7.36K tokens"
    assert g["summary_tokens_printed"] < r * 32768 < 7600
    # eq. 6 at the printed operating point: a 7.36K summary of a 32K prefix is just inside the bound
    assert KP.net_speedup(g["Y_tokens"], 32000.0, g["summary_tokens_printed"], g["S_GB_per_tok"], g["W_GBps"], g["P_tok_s"])
    assert not KP.net_speedup(g["Y_tokens"], 32000.0, 7500.0, g["S_GB_per_tok"], g["W_GBps"], g["P_tok_s"])


def test_p5_eq6_iff_below_eq7_bound():
    for w in (2000.0, 3350.0, 7100.0):
        for y in (100.0, 1000.0, 4000.0):
            for p in (1000.0, 3000.0, 30000.0):
                s = 2e-4
                bound = KP.max_compression_ratio(w, y, s, p)
                for l_full in (8192.0, 32768.0, 131072.0):
                    for frac in (0.01, 0.5, 0.9, 0.999, 1.001, 1.1, 2.0):
                        l_sum = frac * bound * l_full
                        assert KP.net_speedup(y, l_full, l_sum, s, w, p) == (frac < 1.0), (w, y, p, l_full, frac)


def test_p6_eq5_closed_form():
    assert KP.decode_saving_s(32768, 32768, 2e-4, 2000.0) == 0.0
    a = KP.decode_saving_s(32768, 8192, 2e-4, 2000.0)
    assert math.isclose(a, 24576 * 2e-4 / 2000.0, rel_tol=1e-15)
    assert math.isclose(KP.decode_saving_s(65536, 16384, 2e-4, 2000.0), 2 * a, rel_tol=1e-15)
    assert math.isclose(KP.decode_saving_s(32768, 8192, 2e-4, 4000.0), a / 2, rel_tol=1e-15)


def test_p7_bounded_vs_linear_context():
    k, turn, summ = 3, 512, 2048
    ev = KP.kstep_plan(64, k)
    comem, full, mem = KP.context_lengths(ev, turn, summ)
    assert full == [turn * t for t in range(1, 65)]
    assert max(comem) <= summ + (2 * k - 1) * turn
    assert comem[:k + 2] == [turn * t for t in range(1, k + 3)]     # no summary yet: same as full context
    assert [m for m in mem if m] == [turn * t for t in range(k, 65, k)]
