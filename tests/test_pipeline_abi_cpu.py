"""The library's host-side k-step-off plan and latency model (comem_kstep_plan, comem_kstep_context_lengths,
eq. 5-7) against oracle/kstep_pipeline.py: integer events bit-exact on a sweep of (steps, k, delay), doubles
to the last bit or 1 ulp.  CPU only: these entry points do no device work."""
import math

import pytest

import paper_2605_30842_b200 as comem
from oracle import kstep_pipeline as KP


@pytest.mark.parametrize("k", [1, 2, 3, 4, 8])
def test_plan_matches_oracle(k):
    for steps in (0, 1, k, 2 * k + 1, 64):
        for delay in [0] + list(range(1, k + 1)):
            arr, ev = comem.comem_kstep_plan(steps, k, delay)
            want = KP.kstep_plan(steps, k, None if delay == 0 else delay)
            assert len(ev) == len(want) == steps
            for a, b in zip(ev, want):
                assert (a.step, a.summary_upto, bool(a.adopt_summary), bool(a.prefill_uncached), bool(a.launch_memory)) == \
                       (b.step, b.summary_upto, b.adopt_summary, b.prefill_uncached, b.launch_memory)
            got = comem.comem_kstep_context_lengths(arr, steps, 512, 2048)
            exp = KP.context_lengths(want, 512, 2048)
            assert tuple(got) == tuple(exp)


def test_plan_rejects_bad_arguments():
    for args in ((10, 0, 0), (-1, 2, 0), (10, 3, 4)):
        with pytest.raises(comem.ComemError) as ei:
            comem.comem_kstep_plan(*args)
        assert ei.value.status == comem.COMEM_ERR_INVALID_ARG


def test_latency_model_matches_oracle_and_case_study():
    r = comem.comem_max_compression_ratio(2000.0, 1000.0, 2e-4, 3000.0)
    assert r == KP.max_compression_ratio(2000.0, 1000.0, 2e-4, 3000.0) and round(r, 2) == 0.23
    for l_full, l_sum in ((32768.0, 7360.0), (131072.0, 2048.0), (4096.0, 4096.0)):
        a = comem.comem_decode_saving_seconds(l_full, l_sum, 2e-4, 2000.0)
        b = KP.decode_saving_s(l_full, l_sum, 2e-4, 2000.0)
        assert a == b or math.isclose(a, b, rel_tol=2e-16)
        for y in (10.0, 1000.0):
            assert comem.comem_net_speedup(y, l_full, l_sum, 2e-4, 2000.0, 3000.0) == \
                   KP.net_speedup(y, l_full, l_sum, 2e-4, 2000.0, 3000.0)


def test_sm_partition_policy():
    """comem_sm_partition: shares proportional to the bytes, a floor on each side, always the whole GPU."""
    assert comem.comem_sm_partition(1.0, 1.0, 148, 8) == (74, 74)
    assert comem.comem_sm_partition(4.83e9, 3.22e9, 148, 8) == (89, 59)          # config 5: agent C3 + memory batch
    assert comem.comem_sm_partition(1e9, 0.0, 148, 8) == (140, 8)
    assert comem.comem_sm_partition(0.0, 0.0, 148, 8) == (74, 74)
    assert comem.comem_sm_partition(1.0, 1e6, 148, 200) == (74, 74)              # a floor above half is clamped to half
    for a, b in ((1.0, 3.0), (5.0, 2.0), (1e12, 7.0)):
        x, y = comem.comem_sm_partition(a, b, 148, 8)
        assert x + y == 148 and min(x, y) >= 8
        assert abs(x - 148 * a / (a + b)) <= max(1.0, 8 - 148 * min(a, b) / (a + b) + 1)
    for bad in ((-1.0, 1.0, 148, 8), (1.0, float("nan"), 148, 8), (1.0, 1.0, 1, 1)):
        with pytest.raises(comem.ComemError):
            comem.comem_sm_partition(*bad)
