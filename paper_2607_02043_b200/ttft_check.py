"""Measured TTFT_dec of a deflected request against Eq. 6's prediction, end to end on one B200:

  kairos_step_latency_table -> kairos_fit_latency_model (Eq. 4) -> kairos_decide (Algorithm 1: the greedy TBT-safe
  schedule X*, Eq. 5) -> kairos_run_schedule(X*) -> measured per-step latencies and TTFT_dec vs the model's.

Latencies are ONE attention layer's, in microseconds (include/kairos.h units note), so tau here is a per-layer TBT budget.

  python -m paper_2607_02043_b200.ttft_check --out profiles/r02_ttft_vs_model.json.txt
"""
from __future__ import annotations

import argparse
import json

import numpy as np
import torch

from . import kairos as K
from . import latency_table as LT

CASES = [  # (B decodes, K tokens each, prompt length, tau us, beta)
    dict(B=64, K=2048, prompt=6000, tau=150.0, beta=0.9),
    dict(B=256, K=2048, prompt=8192, tau=260.0, beta=0.9),
    dict(B=16, K=8192, prompt=4000, tau=120.0, beta=0.9),
]
CANDIDATES = [4096, 2048, 1024, 512, 256]


def run_case(ctx, model, case, device="cuda"):
    B, Kc, L = case["B"], case["K"], case["prompt"]
    pm = K.prefill_model([1e9, 0, 0, 0])  # the prefill node is out of the picture here: Eq. 7 always prefers the decode node
    decision, node, X, _, ttft_pred = K.decide(model, pm, L, [], 4096, [(B, B * Kc)], CANDIDATES, case["tau"], case["beta"], 1.0, 1e18)
    if decision != "DEFLECT":
        return dict(case=case, decision=decision, note="no TBT-safe schedule under this tau")
    chunks, left = [], L
    for chi in X:  # prefill tokens per step = chi - B, the last one trimmed to what is left of the prompt
        c = min(chi - B, left)
        chunks.append(c)
        left -= c
    m = len(chunks)
    g = torch.Generator(device=device).manual_seed(1)
    rnd = lambda *s: (0.1 * torch.randn(s, generator=g, device=device)).to(torch.bfloat16)
    pages_per = -(-(Kc + m) // 64)
    dec_pt = torch.arange(B * pages_per, dtype=torch.int32, device=device).view(B, pages_per)
    prompt_pt = torch.arange(B * pages_per, B * pages_per + -(-L // 64), dtype=torch.int32, device=device)
    args = (rnd(m, B, 16, 576), dec_pt, [Kc] * B, 10 * rnd(m, B, 512), 10 * rnd(m, B, 64), chunks, rnd(L, 16, 576), 10 * rnd(L, 512),
            10 * rnd(L, 64), prompt_pt)
    ctx.run_schedule(*args)                                   # capture
    ttfts = [ctx.run_schedule(*args)[4] for _ in range(5)]    # graph replays
    steps = ctx.run_schedule(*args, time_steps=True)[5]
    pred_steps, served = [], 0
    for i, c in enumerate(chunks):
        pred_steps.append(K.predict_step(model, B, B * Kc + i * B, c, served))
        served += c
    ttft_meas = float(np.median(ttfts))
    pred_trimmed = float(np.sum(pred_steps))
    return dict(case=case, decision=decision, schedule_chi=X, prefill_tokens_per_step=chunks,
                ttft_pred_eq6_us=ttft_pred, ttft_pred_trimmed_last_chunk_us=pred_trimmed, ttft_measured_graph_us=ttft_meas,
                rel_err=abs(pred_trimmed - ttft_meas) / ttft_meas, step_us_measured=np.round(steps, 1).tolist(),
                step_us_predicted=np.round(pred_steps, 1).tolist(), beta_tau=case["beta"] * case["tau"],
                max_step_measured_us=float(np.max(steps)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    args = ap.parse_args()
    torch.cuda.set_device(0)
    n = max(LT.pages_needed(**LT.GRID), LT.pages_needed(**LT.GRID_PREFIX), 256 * 34 + 200)
    ctx = LT.make_context(n, 256, 8192)
    table = {"grid": LT.run_table(ctx, **LT.GRID, flush=False), "grid_prefix": LT.run_table(ctx, **LT.GRID_PREFIX, flush=False)}
    rows = LT.table_samples(table)
    model, mape = K.fit_latency_model(rows[:, 0], rows[:, 1], rows[:, 2], rows[:, 3], rows[:, 4])
    out = {"library": K.version(), "table": "kairos_step_latency_table, grid + grid_prefix of latency_table.py, L2 not flushed "
           "(the steps of a schedule run back to back)", "model": {"a": list(model.a), "b": list(model.b), "mape_in_sample": mape},
           "cases": [run_case(ctx, model, c) for c in CASES]}
    with open(args.out, "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out["cases"], indent=1))


if __name__ == "__main__":
    main()
