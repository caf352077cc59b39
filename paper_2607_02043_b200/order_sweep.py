"""Launch orders of the two grids on a (B, K, C, P) grid: the planner's own choice against forced orders (a sweep tool).

For every point, `kairos_step_latency_table([B], [K], [C], prefix_len=P)` once with the planner deciding and once per forced
order through the test-only `kairos_debug_set("pairs", c)`: c > 0 = the decode grid first on 148 - 2c SMs beside c clusters
(the other clusters join when decode CTAs exit), c >= 74 = every cluster first.  It shows where `kairos_tune_step` pays.

  python -m paper_2607_02043_b200.order_sweep --out profiles/r02_order_sweep.json.txt
"""
from __future__ import annotations

import argparse
import itertools
import json

import torch

from . import kairos as K

BS, KS, CS, PS = [64, 128, 256], [1024, 2048, 4096], [1536, 2048, 3072, 4096, 6144], [0, 4096]
MODES = [-1, 20, 28, 36, 44, 52, 60, 74]


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    ap.add_argument("--reps", type=int, default=8)
    args = ap.parse_args()
    num_pages = max(BS) * (max(KS) // 64) + (max(PS) + max(CS)) // 64 + 2
    g = torch.Generator(device="cuda").manual_seed(0)
    pool = torch.randn((num_pages, 64, 576), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
    ws = torch.empty(K.workspace_bytes(max(BS), max(CS)), dtype=torch.uint8, device="cuda")
    rows = []
    for P in PS:
        for B, Kc, C in itertools.product(BS, KS, CS):
            row = dict(B=B, K=Kc, C=C, P=P, us={})
            for m in MODES:
                ctx = K.Kairos(pool, ws)  # a fresh context per order: no plan of another order in its cache
                if m != -1:
                    ctx.debug_set("pairs", m)
                med, _ = ctx.step_latency_table([B], [Kc], [C], prefix_len=P, warmup=3, reps=args.reps, flush_l2=True)
                row["us"][str(m)] = round(float(med[0, 0, 0]), 1)
                if m == -1:
                    info = ctx.last_plan_info()
                    row["planner"] = dict(clusters=info["chunk_pairs"], dec_ctas_first=info["dec_ctas_first"])
                del ctx
            row["best"] = min(row["us"], key=lambda k: row["us"][k])
            row["planner_over_best"] = round(row["us"]["-1"] / row["us"][row["best"]], 3)
            rows.append(row)
            print(row, flush=True)
    with open(args.out, "w") as f:
        json.dump(dict(modes=MODES, note="-1 = planner; c = decode grid first beside c clusters; 74 = every cluster first; us = median of reps, L2 flushed",
                       rows=rows), f)


if __name__ == "__main__":
    main()
