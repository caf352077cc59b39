"""CPU-only: SURVEY.md 8(f) row 1 -- the latency model, chunk schedule and deflection decision.

First the plain Python restatement (oracle/decide_oracle.py) is pinned against values worked out by hand from PAPER.md's
equations; then libkairos' kairos_fit_latency_model / kairos_decide (csrc/decide.cpp) are compared with it, and checked
for the paper's own claims: never an unsafe schedule, sum of chunks >= l_r, < 1 ms per
decision on one core, MAPE < 10 % on held-out points of the measured table.
"""
import json
import math
import os
import time

import numpy as np
import pytest

from oracle import decide_oracle as D

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------ pins of the restatement (hand-worked)
def test_eq2_eq3_closed_forms():
    # constant step time t: W_queue = (sum l / chi_p) * t; T_pf = ceil(l_r / chi_p) * t   (Eq. 2, Eq. 3 with G19's limit)
    p = [10.0, 0, 0, 0]
    assert D.w_queue(p, [1000, 3000], 500) == pytest.approx(8 * 10.0)
    assert D.t_pf(p, 1001, 500) == pytest.approx(3 * 10.0)   # 3 chunks, not 4: the printed upper limit would give 40
    # step time = cached tokens: T_pf = chi_p * (0 + 1 + ... + (n-1)) = chi_p * n (n-1) / 2
    p = [0, 0, 1.0, 0]
    assert D.t_pf(p, 2000, 500) == pytest.approx(500 * (0 + 1 + 2 + 3))
    # Eq. 2 evaluates the step at HALF of the outstanding tokens
    assert D.w_queue(p, [600, 400], 100) == pytest.approx(10 * 500.0)
    assert D.ttft_pf([1.0, 0, 0, 0], 100, [], 100) == pytest.approx(1.0)  # empty queue: Eq. 1 = T_pf alone


def test_largest_safe_and_greedy_schedule_by_hand():
    # T_step = C (prefill tokens): beta * tau = 100 -> the largest chi with chi - B <= 100
    a, b = [0, 0, 0], [0, 1.0, 0, 0]
    cands = [512, 256, 128, 64]
    assert D.largest_safe(a, b, 28, 0, 0, cands, 100.0, 1.0) == 128       # C = 100 is safe, C = 228 is not
    assert D.largest_safe(a, b, 28, 0, 0, cands, 200.0, 0.5) == 128       # beta scales tau (Eq. 5)
    assert D.largest_safe(a, b, 28, 0, 0, cands, 30.0, 1.0) == 0          # C = 36 > 30: infeasible
    assert D.largest_safe(a, b, 64, 0, 0, cands, 1e9, 1.0) == 512
    assert D.largest_safe(a, b, 600, 0, 0, cands, 1e9, 1.0) == 0          # no candidate carries a prefill token (G19)
    X, ttft = D.build_schedule(a, b, 28, 0, 250, cands, 100.0, 1.0)
    assert X == [128, 128, 128] and ttft == pytest.approx(300.0)          # served 100, 200, 300 >= 250
    # later chunks cost more: T = C * (P + (C+1)/2) / 100, limit 1500, B = 0, candidates 400/200/100
    b = [0, 0, 0.01, 0]
    t = lambda C, P: 0.01 * C * (P + (C + 1) / 2)
    assert t(400, 0) == pytest.approx(802.0) and t(400, 400) > 1500 and t(200, 400) == pytest.approx(1001.0)
    assert t(200, 600) == pytest.approx(1401.0) and t(200, 800) > 1500 and t(100, 800) == pytest.approx(850.5)
    X, ttft = D.build_schedule([0, 0, 0], b, 0, 0, 900, [400, 200, 100], 1500.0, 1.0)
    assert X == [400, 200, 200, 100]                                      # "larger chunks early and smaller chunks later"
    assert ttft == pytest.approx(802.0 + 1001.0 + 1401.0 + 850.5)
    # the decodes' own tokens enter T0 step by step: T = Kd, K_n = 10, B = 5 -> steps see 10, 15, 20
    X, ttft = D.build_schedule([0, 0, 1.0], [0, 0, 0, 0], 5, 10, 30, [15], 1e9, 1.0)
    assert X == [15, 15, 15] and ttft == pytest.approx(10 + 15 + 20)


def test_algorithm1_by_hand():
    a, b, p = [0, 0, 0], [0, 1.0, 0, 0], [50.0, 0, 0, 0]
    cands = [128, 64]
    # prefill node: queue of 4 chunks ahead (200 us) + 2 own chunks (100 us) = 300 us
    kw = dict(prompt_len=200, queue_lens=[400], chi_p=100, candidates=cands, tau=100.0, beta=1.0, ttft_slo=1e9)
    # node 0: B = 28 -> C = 100 per step -> 2 steps, TTFT_dec = 200;  node 1: B = 60 -> 68, 68, 68 -> 204
    r = D.decide(a, b, p, nodes=[(28, 0), (60, 0)], alpha=1.0, **kw)
    assert r == ("DEFLECT", 0, [128, 128], pytest.approx(300.0), pytest.approx(200.0))
    # Eq. 7, margin: empty queue -> TTFT_pf = 100; 200 <= 1.3 * 100 fails, 200 <= 2 * 100 holds
    kw["queue_lens"] = []
    assert D.decide(a, b, p, nodes=[(28, 0)], alpha=1.3, **kw)[0] == "KEEP"
    assert D.decide(a, b, p, nodes=[(28, 0)], alpha=2.0, **kw)[0] == "DEFLECT"
    kw["ttft_slo"] = 150.0                                               # Eq. 7, second condition
    assert D.decide(a, b, p, nodes=[(28, 0)], alpha=2.0, **kw)[0] == "KEEP"
    # no feasible node -> KEEP with ttft_dec = inf
    r = D.decide(a, b, p, nodes=[(28, 0)], alpha=2.0, **{**kw, "tau": 10.0})
    assert r[0] == "KEEP" and math.isinf(r[4])


def test_fit_recovers_known_coefficients():
    rng = np.random.default_rng(0)
    a, b = [20.0, 0.01, 2e-4], [3.0, 0.03, 2e-5, -1e-5]
    B = rng.integers(1, 300, 200); K = rng.integers(64, 9000, 200); Kd = B * K
    C = rng.choice([0, 0, 128, 512, 2048, 4096], 200); P = rng.choice([0, 1000, 5000], 200) * (C > 0)
    T = np.array([D.t_step(a, b, *r) for r in zip(B, Kd, C, P)])
    fa, fb = D.fit_mixed_model(B, Kd, C, P, T)
    assert np.allclose(fa, a, rtol=1e-6) and np.allclose(fb, b, rtol=1e-5, atol=1e-9)
    assert D.mape(fa, fb, B, Kd, C, P, T) < 1e-9


# ------------------------------------------------------------------ libkairos vs the restatement
def _random_instance(rng):
    a = [rng.uniform(5, 50), rng.uniform(0, 0.05), rng.uniform(0, 5e-4)]
    b = [rng.uniform(0, 10), rng.uniform(0.005, 0.06), rng.uniform(0, 4e-5), rng.uniform(-3e-5, 1e-5)]
    p = [rng.uniform(5, 40), rng.uniform(0.005, 0.05), rng.uniform(0, 1e-3), rng.uniform(0, 2e-6)]
    nodes = [(int(rng.integers(0, 200)), int(rng.integers(0, 2_000_000))) for _ in range(int(rng.integers(0, 6)))]
    cands = sorted({int(c) for c in rng.choice([64, 128, 256, 384, 512, 1024, 2048, 4096], int(rng.integers(1, 6)))}, reverse=True)
    kw = dict(prompt_len=int(rng.integers(1, 20000)), queue_lens=[int(x) for x in rng.integers(1, 8000, int(rng.integers(0, 5)))],
              chi_p=int(rng.choice([512, 2048, 8192])), nodes=nodes, candidates=cands,
              tau=float(rng.uniform(20, 600)), beta=float(rng.uniform(0.5, 1.0)), alpha=float(rng.uniform(1.0, 2.0)),
              ttft_slo=float(rng.choice([1e3, 1e4, 1e9])))
    return a, b, p, kw


def test_decide_matches_restatement_and_is_never_unsafe():
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(7)
    n_deflect = 0
    for _ in range(400):
        a, b, p, kw = _random_instance(rng)
        want = D.decide(a, b, p, **kw)
        m, pm = K.step_model(a, b), K.prefill_model(p)
        got = K.decide(m, pm, kw["prompt_len"], kw["queue_lens"], kw["chi_p"], kw["nodes"], kw["candidates"], kw["tau"],
                       kw["beta"], kw["alpha"], kw["ttft_slo"])
        assert got[0] == want[0] and got[1] == want[1] and got[2] == want[2]
        assert got[3] == pytest.approx(want[3], rel=1e-12)
        assert (math.isinf(got[4]) and math.isinf(want[4])) or got[4] == pytest.approx(want[4], rel=1e-12)
        if got[0] == "DEFLECT":
            n_deflect += 1
            B_n, K_n = kw["nodes"][got[1]]
            served, Kd = 0, K_n
            for i, chi in enumerate(got[2]):
                assert chi in kw["candidates"] and chi > B_n
                assert served < kw["prompt_len"]                                    # no step after the prompt is done
                assert K.predict_step(m, B_n, Kd, chi - B_n, served) <= kw["beta"] * kw["tau"] * (1 + 1e-12)
                served += chi - B_n
                Kd += B_n
            assert served >= kw["prompt_len"]
            assert got[4] <= kw["alpha"] * got[3] * (1 + 1e-12) and got[4] <= kw["ttft_slo"] * (1 + 1e-12)  # Eq. 7
    assert 20 < n_deflect < 380  # the random instances exercise both outcomes


def test_decide_argument_errors():
    from paper_2607_02043_b200 import kairos as K
    m, pm = K.step_model([1, 0, 0], [0, 1, 0, 0]), K.prefill_model([1, 0, 0, 0])
    ok = dict(prompt_len=10, queue_lens=[], chi_p=8, nodes=[(1, 0)], candidates=[8, 4], tbt_slo=100.0, beta=1.0, alpha=1.0, ttft_slo=1e9)
    assert K.decide(m, pm, **ok)[0] in ("KEEP", "DEFLECT")
    for bad in [dict(candidates=[4, 8]), dict(candidates=[8, 8]), dict(alpha=0.5), dict(beta=0.0), dict(prompt_len=0), dict(chi_p=0)]:
        with pytest.raises(K.KairosError) as ei:
            K.decide(m, pm, **{**ok, **bad})
        assert ei.value.code == -1
    with pytest.raises(K.KairosError) as ei:   # schedule longer than the caller's buffer
        K.decide(m, pm, **{**ok, "prompt_len": 1000, "tbt_slo": 1e9, "alpha": 100.0}, max_schedule=3)
    assert ei.value.code == -3


def test_fit_matches_restatement():
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(3)
    B = rng.integers(1, 300, 120); Kc = rng.integers(64, 9000, 120); Kd = B * Kc
    C = rng.choice([0, 0, 128, 512, 2048, 4096], 120); P = rng.choice([0, 1000, 5000], 120) * (C > 0)
    T = 25 + 0.01 * B + 2.2e-4 * Kd + (C > 0) * (2 + 0.03 * C + 2e-5 * C * (P + (C + 1) / 2)) * rng.uniform(0.9, 1.1, 120)
    fa, fb = D.fit_mixed_model(B, Kd, C, P, T)
    m, mape = K.fit_latency_model(B, Kd, C, P, T)
    assert np.allclose(list(m.a), fa, rtol=1e-6, atol=1e-9) and np.allclose(list(m.b), fb, rtol=1e-5, atol=1e-9)
    assert mape == pytest.approx(D.mape(fa, fb, B, Kd, C, P, T), rel=1e-6)
    with pytest.raises(K.KairosError):  # every sample with the same B and Kd: singular
        K.fit_latency_model([4] * 8, [400] * 8, [0] * 8, [0] * 8, [1.0] * 8)


def _table_samples():
    path = os.path.join(ROOT, "profiles", "r02_latency_table.json.txt")
    d = json.load(open(path))
    rows = []
    for key in ("grid", "grid_prefix", "configs3"):
        g = d.get(key)
        if g is None:
            continue
        m = np.array(g["median_us"])
        for i, B in enumerate(g["Bs"]):
            for j, Kc in enumerate(g["Ks"]):
                for k, C in enumerate(g["Cs"]):
                    if B == 0 and C == 0:
                        continue
                    rows.append((B, B * Kc, C, g["prefix_len"] if C > 0 else 0, m[i, j, k]))
    return np.array(rows, dtype=np.float64)


def test_model_fitted_on_the_measured_table_holds_out_under_10_percent():
    """'on held-out traces ... MAPE < 10 %'.  The table is the committed output of kairos_step_latency_table
    on a B200 (profiles/r02_latency_table.json.txt); every third point is held out of the fit."""
    from paper_2607_02043_b200 import kairos as K
    rows = _table_samples()
    held = np.arange(len(rows)) % 3 == 1
    tr, te = rows[~held], rows[held]
    m, mape_in = K.fit_latency_model(tr[:, 0], tr[:, 1], tr[:, 2], tr[:, 3], tr[:, 4])
    pred = np.array([K.predict_step(m, *(int(x) for x in r[:4])) for r in te])
    mape_out = float(np.mean(np.abs(pred - te[:, 4]) / te[:, 4]))
    assert mape_in < 0.10 and mape_out < 0.10, (mape_in, mape_out)


def test_decision_takes_under_a_millisecond():
    """'the scheduling delay is under 1 ms on a single CPU core' (their setup: 2 decode nodes)."""
    from paper_2607_02043_b200 import kairos as K
    m = K.step_model([19.0, 0.006, 2.2e-4], [3.5, 0.026, 1.9e-5, -2.5e-5])
    pm = K.prefill_model([20.0, 0.03, 1e-3, 2e-5])
    nodes = [(64 + 8 * i, 100_000 * (i + 1)) for i in range(8)]
    args = (m, pm, 16384, [4000, 9000, 2000], 2048, nodes, [2048, 1024, 512, 256, 128], 400.0, 0.9, 1.3, 1e9)
    K.decide(*args)
    t0 = time.perf_counter()
    n = 200
    for _ in range(n):
        r = K.decide(*args)
    dt = (time.perf_counter() - t0) / n
    assert r[0] in ("KEEP", "DEFLECT") and dt < 1e-3, dt
