"""Deployment-time profiling: kairos_step_latency_table over a (B, K, C) grid, written as JSON.

The table is the input of the latency model of Eq. 4 that `kairos_fit_latency_model` fits and
`kairos_decide` consumes.  Default grid: BASELINE.json configs[3] (B = 256, K = 2048, C in {0 .. 8192}, 20 timed reps
after 5 warm-ups) plus a B x K x C grid around it.  The pool is synthetic (N(0,1) bf16): this is a timing tool.

  python -m paper_2607_02043_b200.latency_table --out profiles/r02_latency_table.json.txt [--grid paper] [--no-flush]
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np
import torch

from . import kairos as K

CONFIG3 = dict(Bs=[256], Ks=[2048], Cs=[0, 256, 512, 1024, 2048, 4096, 8192])
GRID = dict(Bs=[16, 64, 256], Ks=[512, 2048, 8192], Cs=[0, 256, 512, 1024, 2048, 4096])
GRID_PREFIX = dict(Bs=[16, 64, 256], Ks=[2048], Cs=[256, 1024, 2048], prefix=4096)  # later chunks of a request
# the paper's own microbenchmark grid (Fig. 1 caption PAPER.md:159): its chi counts B + C tokens
PAPER_GRID = dict(Bs=[4, 8, 16, 32], Ks=[842, 998, 3569, 13968, 14013], chis=[128, 256, 512, 1024, 2048])


def make_context(num_pages: int, max_b: int, max_c: int, device="cuda"):
    g = torch.Generator(device=device).manual_seed(0)
    pool = torch.randn((num_pages, 64, 576), generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    ws = torch.empty(K.workspace_bytes(max_b, max_c), dtype=torch.uint8, device=device)
    return K.Kairos(pool, ws)


def pages_needed(Bs, Ks, Cs, prefix=0) -> int:
    return max(b * -(-k // 64) for b in Bs for k in Ks) + -(-(prefix + max(Cs)) // 64) + 1


def run_table(ctx, Bs, Ks, Cs, prefix=0, warmup=5, reps=20, flush=True) -> dict:
    t0 = time.time()
    med, mn = ctx.step_latency_table(Bs, Ks, Cs, prefix_len=prefix, warmup=warmup, reps=reps, flush_l2=flush)
    return {"Bs": list(Bs), "Ks": list(Ks), "Cs": list(Cs), "prefix_len": prefix, "warmup": warmup, "reps": reps,
            "l2": "256 MiB rewritten before every step, outside the timed interval" if flush else "not flushed",
            "median_us": np.round(med, 2).tolist(), "min_us": np.round(mn, 2).tolist(), "index": "[iB][iK][iC]",
            "wall_s": round(time.time() - t0, 2)}


def table_samples(table: dict, keys=("grid", "grid_prefix", "configs3")):
    """Rows (B, Kd, C, P, T_us) of a table written by this module: the samples kairos_fit_latency_model takes."""
    rows = []
    for key in keys:
        g = table.get(key)
        if g is None:
            continue
        m = np.array(g["median_us"])
        for i, B in enumerate(g["Bs"]):
            for j, Kc in enumerate(g["Ks"]):
                for k, C in enumerate(g["Cs"]):
                    if B == 0 and C == 0:
                        continue
                    rows.append((B, B * Kc, C, g["prefix_len"] if C > 0 else 0, float(m[i, j, k])))
    return np.array(rows, dtype=np.float64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    ap.add_argument("--grid", default="default", choices=["default", "paper"])
    ap.add_argument("--no-flush", action="store_true")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    args = ap.parse_args()
    torch.cuda.set_device(0)
    out = {"library": K.version(), "device": torch.cuda.get_device_name(0),
           "units": "one layer's attention, microseconds; K = per-decode context; C = prefill tokens only (include/kairos.h)"}
    if args.grid == "default":
        n = max(pages_needed(**CONFIG3), pages_needed(**GRID), pages_needed(**GRID_PREFIX))
        ctx = make_context(n, 256, 8192)
        out["configs3"] = run_table(ctx, **CONFIG3, warmup=args.warmup, reps=args.reps, flush=not args.no_flush)
        out["grid"] = run_table(ctx, **GRID, warmup=args.warmup, reps=args.reps, flush=not args.no_flush)
        out["grid_prefix"] = run_table(ctx, **GRID_PREFIX, warmup=args.warmup, reps=args.reps, flush=not args.no_flush)
    else:
        # Fig. 1's setting, attention only: B decodes with K cached tokens each, a batch of chi tokens of which chi - B are
        # prefill, five successive chunks of the same request (the prefix grows by one chunk each time)
        g = PAPER_GRID
        import os
        pk = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
        peaks = json.load(open(pk)) if os.path.exists(pk) else {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}
        peaks = {"hbm_gbs": peaks["hbm_gbs"], "bf16_tflops": peaks["bf16_tflops"]}
        n = max(b * -(-k // 64) for b in g["Bs"] for k in g["Ks"]) + -(-(5 * max(g["chis"])) // 64) + 1
        ctx = make_context(n, max(g["Bs"]), max(g["chis"]))
        rows = []
        for chi in g["chis"]:
            for B in g["Bs"]:
                C = chi - B
                for j in range(5):
                    t = run_table(ctx, [B], g["Ks"], [0, C], prefix=j * C, warmup=args.warmup, reps=args.reps, flush=not args.no_flush)
                    for iK, Kc in enumerate(g["Ks"]):
                        mixed = t["median_us"][0][iK][1]
                        P = j * C
                        nbytes = B * Kc * 1152 + B * 34816 + (P + C) * 1152 + C * 34816      # SURVEY.md 8(d) algorithmic work
                        flops = 34816 * (B * Kc + C * P + C * (C + 1) // 2)
                        roof = max(nbytes / (peaks["hbm_gbs"] * 1e3), flops / (peaks["bf16_tflops"] * 1e6))
                        rows.append({"chi": chi, "B": B, "K": Kc, "C": C, "chunk_index": j, "prefix": P,
                                     "decode_only_us": t["median_us"][0][iK][0], "mixed_us": mixed,
                                     "delta_us": round(mixed - t["median_us"][0][iK][0], 2), "roofline_us": round(roof, 2),
                                     "frac_of_roofline": round(roof / mixed, 3)})
        out["paper_grid"] = {"note": "PAPER.md:143 grid (B x K x chi, five successive chunks), attention only, one layer; "
                             "delta_us = the step-latency increase Fig. 1 plots (PAPER.md:159)", "peaks": peaks, "rows": rows}
    with open(args.out, "w") as f:
        json.dump(out, f, indent=1)
    print(f"wrote {args.out}")


if __name__ == "__main__":
    main()
