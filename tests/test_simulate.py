"""CPU-only: the policy simulator (second half).

oracle/sim_oracle.py (the flat Python restatement of the event rules) is pinned by scenarios worked out by hand; libkairos'
kairos_simulate (csrc/simulate.cpp) must then reproduce it exactly -- deflection counts, step counts, every TTFT -- on seeded
bursty arrivals under all four policies."""
import math

import numpy as np
import pytest

from oracle import sim_oracle as S
from paper_2607_02043_b200 import workloads as W

A0, B0 = [0.0, 0.0, 0.0], [0.0, 0.0, 0.0, 0.0]


def _run(a, b, p, reqs, **kw):
    d = dict(n_prefill=1, n_decode=1, chi_p=100, policy=S.BASELINE, param=0, static_chi=128, candidates=[128, 64], tau=1e30,
             beta=1.0, alpha=1.0, ttft_slo=1e30, transfer_per_token=0.0)
    d.update(kw)
    return S.simulate(a, b, p, reqs, **d)


def test_baseline_single_and_queued_requests_by_hand():
    # prefill step = 10 per chunk of 100 tokens; transfer 0.01 per token; decode step = 2 (constant)
    a, b, p = [2.0, 0, 0], B0, [10.0, 0, 0, 0]
    res, ttft = _run(a, b, p, [(0.0, 250, 3)], transfer_per_token=0.01)
    assert ttft == [pytest.approx(3 * 10 + 2.5)]                      # 3 chunks (Eq. 3) + KV transfer of 250 tokens
    assert res["decode_steps"] == 3 and res["makespan"] == pytest.approx(32.5 + 3 * 2.0) and res["n_deflected"] == 0
    # FIFO: the second request waits for the first (arrives at 5, first leaves the prefill node at 30)
    res, ttft = _run(a, b, p, [(0.0, 250, 1), (5.0, 100, 1)])
    assert ttft == [pytest.approx(30.0), pytest.approx(30.0 + 10.0 - 5.0)]
    # two prefill nodes: the second request takes the idle one
    res, ttft = _run(a, b, p, [(0.0, 250, 1), (5.0, 100, 1)], n_prefill=2)
    assert ttft == [pytest.approx(30.0), pytest.approx(10.0)]
    # the two decodes overlap in one batch on the least-loaded decode node: 1 + 1 tokens -> steps at 30..32 (B=1) ... count them
    res, _ = _run(a, b, p, [(0.0, 100, 2), (0.0, 100, 2)], n_prefill=2)
    assert res["decode_steps"] == 2                                    # both ready at 10, one node, B = 2 for two steps


def test_static_length_deflection_and_tbt_violations_by_hand():
    # T_step = 1 + 0.01 * C (+ nothing else); prefill node slow (100 per chunk)
    a, b, p = [1.0, 0, 0], [0.0, 0.01, 0.0, 0.0], [100.0, 0, 0, 0]
    # SL(300): the 250-token prompt is deflected; no decodes in flight -> C = min(max(128 - 0, 1), left) = 128, 122
    res, ttft = _run(a, b, p, [(0.0, 250, 2)], policy=S.SL, param=300)
    assert res["n_deflected"] == 1
    assert ttft == [pytest.approx((1 + 1.28) + (1 + 1.22))]
    assert res["decode_steps"] == 2                                    # then it decodes 2 tokens on the same node
    # SL(200): too long -> prefill path
    res, ttft = _run(a, b, p, [(0.0, 250, 2)], policy=S.SL, param=200)
    assert res["n_deflected"] == 0 and ttft == [pytest.approx(300.0)]
    # a decode in flight shrinks the chunk (chi counts B + C) and its steps are TBT-checked: tau = 2.2 < 1 + 0.01 * 127
    reqs = [(0.0, 400, 80), (450.5, 254, 1)]
    res, ttft = _run(a, b, p, reqs, policy=S.SL, param=300, tau=2.2, ttft_slo=1e9)
    # request 0 (400 tokens: not deflected): prefill 4 x 100 -> decoding from t = 400, one step per 1.0; request 1 arrives at
    # 450.5 while the step 450..451 runs, then two mixed steps with C = 127 each (2.27 > tau): two violated steps, both hit request 0
    assert res["n_deflected"] == 1 and res["tbt_violations"] == 2
    assert ttft[1] == pytest.approx((451.0 - 450.5) + 2 * 2.27)
    assert res["slo_attainment"] == pytest.approx(0.5)                 # request 0 decoded in a violated step


def test_static_queue_policy_fires_only_when_every_prefill_queue_is_long():
    a, b, p = [1.0, 0, 0], [0.0, 0.01, 0.0, 0.0], [100.0, 0, 0, 0]
    reqs = [(0.0, 100, 1), (1.0, 100, 1), (2.0, 100, 1), (3.0, 100, 1)]
    # one prefill node, theta = 1: request 2 finds 1 waiting (not > 1) -> queued; request 3 finds 2 waiting -> deflected
    res, ttft = _run(a, b, p, reqs, policy=S.SQ, param=1)
    assert res["n_deflected"] == 1 and ttft[3] == pytest.approx(1 + 1.0)
    res, _ = _run(a, b, p, reqs, policy=S.SQ, param=1, n_prefill=2)     # two nodes share the queue: never both > 1
    assert res["n_deflected"] == 0


def test_oracle_policy_follows_algorithm1_schedule():
    a, b, p = [0.0, 0, 0], [0.0, 1.0, 0.0, 0.0], [1000.0, 0, 0, 0]     # T_step = C; prefill node hopeless
    res, ttft = _run(a, b, p, [(0.0, 250, 0)], policy=S.ORACLE, candidates=[512, 256, 128, 64], tau=128.0, ttft_slo=1e9)
    assert res["n_deflected"] == 1 and ttft == [pytest.approx(128 + 122)]   # largest safe chi = 128, two steps (second trimmed)
    res, ttft = _run(a, b, p, [(0.0, 250, 0)], policy=S.ORACLE, candidates=[512, 256, 128, 64], tau=10.0)
    assert res["n_deflected"] == 0                                          # nothing is TBT-safe -> KEEP


def _models():
    a = [19.0, 0.006, 2.2e-4]
    b = [3.5, 0.026, 1.9e-5, -2.5e-5]
    p = [20.0, 0.03, 1e-3, 2e-5]
    return a, b, p


@pytest.mark.parametrize("policy,param", [("baseline", 0), ("sq", 1), ("sq", 4), ("sl", 1024), ("sl", 4096), ("oracle", 0)])
def test_library_reproduces_the_restatement(policy, param):
    from paper_2607_02043_b200 import kairos as K
    a, b, p = _models()
    reqs = W.make_arrivals(11, 160, rate=1 / 900.0, burst_every=20000.0, burst_size=10, out_median=60.0)
    kw = dict(n_prefill=2, n_decode=2, chi_p=2048, static_chi=128, candidates=[2048, 1024, 512, 256, 128], tau=160.0, beta=0.9,
              alpha=1.3, ttft_slo=6000.0, transfer_per_token=0.02)
    want, want_ttft = S.simulate(a, b, p, reqs, policy=K.POLICIES[policy], param=param, **kw)
    got, got_ttft = K.simulate(K.step_model(a, b), K.prefill_model(p), reqs, kw["n_prefill"], kw["n_decode"], kw["chi_p"], policy, param,
                               kw["static_chi"], kw["candidates"], kw["tau"], kw["beta"], kw["alpha"], kw["ttft_slo"], kw["transfer_per_token"])
    for k in ("n_requests", "n_deflected", "decode_steps", "tbt_violations"):
        assert got[k] == want[k], k
    assert np.allclose(got_ttft, want_ttft, rtol=1e-12, atol=0)
    for k in ("p95_ttft", "mean_ttft", "slo_attainment", "makespan"):
        assert got[k] == pytest.approx(want[k], rel=1e-12), k
    if policy == "baseline":
        assert got["n_deflected"] == 0
    if policy == "oracle":
        assert got["n_deflected"] > 0 and got["tbt_violations"] == 0     # PAPER.md:296 carried into the simulator: never an unsafe step it planned


def test_argument_errors():
    from paper_2607_02043_b200 import kairos as K
    m, pm = K.step_model([1, 0, 0], [0, 0, 0, 0]), K.prefill_model([1, 0, 0, 0])
    with pytest.raises(K.KairosError):
        K.simulate(m, pm, [(1.0, 10, 1), (0.5, 10, 1)], 1, 1, 8, "baseline")   # not sorted
    with pytest.raises(K.KairosError):
        K.simulate(m, pm, [(0.0, 0, 1)], 1, 1, 8, "baseline")                  # empty prompt
    res, ttft = K.simulate(m, pm, [], 1, 1, 8, "baseline")
    assert res["n_requests"] == 0
