"""Plain restatement of the paper's policy simulator -- TEST INFRASTRUCTURE, not the product.

Only tests/ may import this.  PAPER.md:183 ("we wrap the three predictors in an event-based simulator with support for PD
disaggregation") and section 3.4 (Baseline, Static-queue SQ(theta), Static-length SL(l), Oracle; Table 4's
columns).  The paper gives no pseudo-code for the simulator, so the event rules below ARE the reading (G22); they are
written as one flat loop in float64 Python, with the latency models and Algorithm 1 taken from oracle/decide_oracle.py.
It shares no code with csrc/simulate.cpp.

Rules (G22):
  * N_p prefill nodes, each a FIFO server: a request occupies its node for T_pf (Eq. 3).  An arriving request that is not
    deflected goes to the prefill node with the fewest outstanding prompt tokens (in service + queued; ties: lowest index).
    When its prefill ends at time f it is ready on a decode node at f + transfer_per_token * l_r (KV transfer = bytes over
    bandwidth); TTFT = that time - arrival (PAPER.md:171-172 counts queue wait and KV transfer in TTFT).  It joins
    the decode node with the fewest (in-flight + pending) requests at time f (ties: lowest index).
  * N_d decode nodes run steps back to back while they have work.  At a step start the node admits every pending request
    whose ready time has passed, then runs ONE mixed batch: B in-flight decodes caching Kd tokens in total, plus -- if a
    deflected request is in its prefill phase on this node (at most one per node) -- a chunk of
    C = min(max(chi - B, 1), tokens left) prefill tokens over the P already served (chi counts B + C).  The step
    lasts T_step(B, Kd, C, P) (Eq. 4).  At its end every in-flight decode has produced one token (context + 1) and leaves
    when its output is complete; the chunk is served; a deflected request whose prompt is complete has TTFT = step end -
    arrival and is pending on the same node from that instant.
  * A step with B > 0 that lasts longer than tau is a TBT violation of the step and of every request decoding in it.
  * Deflection target of the static policies: the decode node with the fewest in-flight decodes among those that host no
    deflected request in its prefill phase (ties: lowest index); if there is none the request takes the prefill path.
    SQ(theta): deflect when the number of WAITING requests exceeds theta on all prefill nodes.  SL(l): deflect when l_r < l.
    Both use the fixed chi given (128 in the paper).  Oracle: Algorithm 1 (decide_oracle.decide) on the simulator's own state:
    the queue of the prefill node the request would go to, and (B, Kd) of every eligible decode node; the schedule X* it
    returns is followed step by step (its last chi is repeated if in-flight decodes grew meanwhile).
  * Events at equal times: decode step ends (node order), prefill completions (node order), the arrival; then idle nodes start.
  * P95 = nearest rank: sorted[ceil(0.95 n) - 1].  SLO attainment = share of requests with TTFT <= ttft_slo and no violated step.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

from oracle import decide_oracle as D

BASELINE, SQ, SL, ORACLE = 0, 1, 2, 3


def simulate(a, b, p, reqs: Sequence[Tuple[float, int, int]], n_prefill: int, n_decode: int, chi_p: int, policy: int,
             param: int, static_chi: int, candidates, tau: float, beta: float, alpha: float, ttft_slo: float,
             transfer_per_token: float):
    """reqs: (arrival, prompt_len, output_len) sorted by arrival.  Returns (result dict, ttft list)."""
    n = len(reqs)
    inf = math.inf
    # prefill nodes
    pf_queue: List[List[int]] = [[] for _ in range(n_prefill)]
    pf_cur = [-1] * n_prefill
    pf_end = [inf] * n_prefill
    # decode nodes
    active: List[List[List[int]]] = [[] for _ in range(n_decode)]      # [req, context, remaining]
    pending: List[List[Tuple[int, float]]] = [[] for _ in range(n_decode)]  # (req, ready time)
    defl = [None] * n_decode       # [req, served P, schedule (list of chi or None), step index, C of the running step]
    step_end = [inf] * n_decode
    step_reqs: List[List[int]] = [[] for _ in range(n_decode)]
    ttft = [inf] * n
    violated = [False] * n
    n_deflected = decode_steps = violations = 0
    finished = 0
    next_arr = 0
    t = 0.0

    def t_pf(l):
        return D.t_pf(p, l, chi_p)

    def outstanding(i):
        s = sum(reqs[r][1] for r in pf_queue[i])
        return s + (reqs[pf_cur[i]][1] if pf_cur[i] >= 0 else 0)

    def eligible_nodes():
        return [d for d in range(n_decode) if defl[d] is None]

    while finished < n:
        # ---- next event time
        t_next = reqs[next_arr][0] if next_arr < n else inf
        t_next = min([t_next] + pf_end + step_end)
        for d in range(n_decode):  # an idle node wakes when a pending request becomes ready
            if step_end[d] == inf and pending[d]:
                t_next = min(t_next, max(t, min(rt for _, rt in pending[d])))
        assert t_next < inf, "simulation stalled"
        t = t_next
        # ---- decode step ends
        for d in range(n_decode):
            if step_end[d] == t:
                step_end[d] = inf
                keep = []
                for e in active[d]:
                    e[1] += 1
                    e[2] -= 1
                    if e[2] > 0:
                        keep.append(e)
                    else:
                        finished += 1
                active[d] = keep
                if defl[d] is not None:
                    r = defl[d][0]
                    defl[d][1] += defl[d][4]
                    defl[d][3] += 1
                    if defl[d][1] >= reqs[r][1]:
                        ttft[r] = t - reqs[r][0]
                        pending[d].append((r, t))
                        defl[d] = None
        # ---- prefill completions
        for i in range(n_prefill):
            if pf_end[i] == t:
                r = pf_cur[i]
                pf_cur[i], pf_end[i] = -1, inf
                ready = t + transfer_per_token * reqs[r][1]
                ttft[r] = ready - reqs[r][0]
                load = [len(active[d]) + len(pending[d]) for d in range(n_decode)]
                d = load.index(min(load))
                pending[d].append((r, ready))
        # ---- the arrival(s) at this instant
        while next_arr < n and reqs[next_arr][0] == t:
            r = next_arr
            next_arr += 1
            l = reqs[r][1]
            out = [outstanding(i) for i in range(n_prefill)]
            pn = out.index(min(out))
            target, sched = -1, None
            elig = eligible_nodes()
            if policy == SQ:
                if all(len(pf_queue[i]) > param for i in range(n_prefill)) and elig:
                    target = min(elig, key=lambda d: (len(active[d]), d))
            elif policy == SL:
                if l < param and elig:
                    target = min(elig, key=lambda d: (len(active[d]), d))
            elif policy == ORACLE and elig:
                qlens = ([reqs[pf_cur[pn]][1]] if pf_cur[pn] >= 0 else []) + [reqs[q][1] for q in pf_queue[pn]]
                nodes = [(len(active[d]), float(sum(e[1] for e in active[d]))) for d in elig]
                dec, ns, X, _, _ = D.decide(a, b, p, l, qlens, chi_p, nodes, candidates, tau, beta, alpha, ttft_slo)
                if dec == "DEFLECT":
                    target, sched = elig[ns], X
            if target >= 0:
                n_deflected += 1
                defl[target] = [r, 0, sched, 0, 0]
            else:
                pf_queue[pn].append(r)
        # ---- idle nodes start work
        for i in range(n_prefill):
            if pf_cur[i] < 0 and pf_queue[i]:
                pf_cur[i] = pf_queue[i].pop(0)
                pf_end[i] = t + t_pf(reqs[pf_cur[i]][1])
        for d in range(n_decode):
            if step_end[d] != inf:
                continue
            still = []
            for (r, rt) in pending[d]:
                if rt <= t:
                    if reqs[r][2] > 0:
                        active[d].append([r, reqs[r][1], reqs[r][2]])
                    else:
                        finished += 1
                else:
                    still.append((r, rt))
            pending[d] = still
            B = len(active[d])
            C, P = 0, 0
            if defl[d] is not None:
                r, P, sched, k = defl[d][0], defl[d][1], defl[d][2], defl[d][3]
                chi = static_chi if sched is None else sched[min(k, len(sched) - 1)]
                C = min(max(chi - B, 1), reqs[r][1] - P)
                defl[d][4] = C
            if B == 0 and C == 0:
                continue
            Kd = float(sum(e[1] for e in active[d]))
            T = D.t_step(a, b, B, Kd, C, P)
            step_end[d] = t + T
            if B > 0:
                decode_steps += 1
                if T > tau:
                    violations += 1
                    for e in active[d]:
                        violated[e[0]] = True
    s = sorted(ttft)
    ok = sum(1 for r in range(n) if ttft[r] <= ttft_slo and not violated[r])
    res = dict(n_requests=n, n_deflected=n_deflected, p95_ttft=s[max(0, math.ceil(0.95 * n) - 1)], mean_ttft=sum(ttft) / n,
               decode_steps=decode_steps, tbt_violations=violations, slo_attainment=ok / n, makespan=t)
    return res, ttft
