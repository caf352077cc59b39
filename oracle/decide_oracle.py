"""Plain restatement of the paper's decision logic -- TEST INFRASTRUCTURE, not the product.

Only tests/ may import this.  It follows PAPER.md step by step, in the paper's order and notation, in float64 Python:
Eq. 1-3 (section 4.2), Eq. 4 (section 4.3.1), Eq. 5-6 (section
4.3.2), Eq. 7 (section 4.4) and Algorithm 1.  The least-squares fit of the two
regressors of Eq. 4 ("simple linear regressors") calls numpy.linalg.lstsq.  It shares no code with
csrc/decide.cpp.

Readings (G19-G21):
  G19  Eq. 3's sum runs i = 0 .. ceil(l_r/chi_p) - 1 (the printed upper limit is one term too many); Algorithm 1 serves
       chi - B_n prefill tokens per step ("injecting chi - B_n prefill tokens") and skips candidates <= B_n;
       F starts empty; LargestSafe tests against beta * tau (Eq. 5) although Algorithm 1's call omits beta.
  G20  The paper lumps every cached token into K_n.  One attention layer treats them differently (a decode's token is read
       once per step; a prefix token of the deflected request meets every query token of the chunk), so the model keeps
       them apart: Kd = tokens cached by the in-flight decodes, P = tokens of the deflected request already cached.
       T0(B, Kd) = a0 + a1*B + a2*Kd;  dT(C, P, Kd) = b0 + b1*C + b2*C*(P + (C+1)/2) + b3*Kd for C > 0, 0 for C = 0.
       Step i of a schedule on node n: Kd_i = K_n + (i-1)*B_n (each decode appends one token per step), P_i = sum_{j<i} C_j,
       C_i = chi_i - B_n.  Linear in its parameters: closed-form least squares, as in the paper.
  G21  The fit minimises RELATIVE error (rows weighted by 1/T), because the criterion the paper states is MAPE < 10 %
       (PAPER.md:181); scikit-learn's unweighted fit is the special case of equal weights.
"""
from __future__ import annotations

import math
from typing import List, Optional, Sequence, Tuple

import numpy as np


# ---------------------------------------------------------------------------------------------- Eq. 4
def t0(a: Sequence[float], B: float, Kd: float) -> float:
    """Decode-only step latency T_step^(0)(B_n, K_n) of Eq. 4."""
    return a[0] + a[1] * B + a[2] * Kd


def delta_pf(b: Sequence[float], C: float, P: float, Kd: float) -> float:
    """Latency increase Delta T_pf of Eq. 4 from injecting C prefill tokens whose request has P tokens cached (G20)."""
    if C <= 0:
        return 0.0
    return b[0] + b[1] * C + b[2] * C * (P + (C + 1) / 2.0) + b[3] * Kd


def t_step(a, b, B: float, Kd: float, C: float, P: float) -> float:
    """Eq. 4: T_step = T^(0) + Delta T_pf."""
    return t0(a, B, Kd) + delta_pf(b, C, P, Kd)


def t_prefill_step(p: Sequence[float], tokens: float, cached: float) -> float:
    """Prefill-node step latency: 'a function of the number of tokens in the batch and the number of cached KV tokens'
    (PAPER.md:310); p[3] is an optional tokens*cached term (0 gives the paper's plain form)."""
    return p[0] + p[1] * tokens + p[2] * cached + p[3] * tokens * cached


def fit_mixed_model(B, Kd, C, P, T) -> Tuple[List[float], List[float]]:
    """Two regressors as in PAPER.md:312: first the pure-decode latency from the C = 0 rows, then the additional prefill
    time from the residual of the C > 0 rows.  Weighted by 1/T (G21)."""
    B, Kd, C, P, T = (np.asarray(x, dtype=np.float64) for x in (B, Kd, C, P, T))
    dec = C == 0
    X0 = np.stack([np.ones(dec.sum()), B[dec], Kd[dec]], axis=1)
    w0 = 1.0 / T[dec]
    a, *_ = np.linalg.lstsq(X0 * w0[:, None], T[dec] * w0, rcond=None)
    mix = C > 0
    resid = T[mix] - (a[0] + a[1] * B[mix] + a[2] * Kd[mix])
    X1 = np.stack([np.ones(mix.sum()), C[mix], C[mix] * (P[mix] + (C[mix] + 1) / 2.0), Kd[mix]], axis=1)
    w1 = 1.0 / T[mix]
    b, *_ = np.linalg.lstsq(X1 * w1[:, None], resid * w1, rcond=None)
    return [float(v) for v in a], [float(v) for v in b]


def mape(a, b, B, Kd, C, P, T) -> float:
    pred = np.array([t_step(a, b, *row) for row in zip(B, Kd, C, P)])
    T = np.asarray(T, dtype=np.float64)
    return float(np.mean(np.abs(pred - T) / T))


# ---------------------------------------------------------------------------------------------- Eq. 1-3
def w_queue(p, queue_lens: Sequence[int], chi_p: int) -> float:
    """Eq. 2: number of chunks ahead times the average chunk time with half the outstanding tokens cached."""
    s = float(sum(queue_lens))
    return (s / chi_p) * t_prefill_step(p, chi_p, s / 2.0)


def t_pf(p, prompt_len: int, chi_p: int) -> float:
    """Eq. 3 with the upper limit of G19: i = 0 .. ceil(l_r/chi_p) - 1."""
    return sum(t_prefill_step(p, chi_p, chi_p * i) for i in range(math.ceil(prompt_len / chi_p)))


def ttft_pf(p, prompt_len: int, queue_lens: Sequence[int], chi_p: int) -> float:
    """Eq. 1."""
    return w_queue(p, queue_lens, chi_p) + t_pf(p, prompt_len, chi_p)


# ---------------------------------------------------------------------------------------------- Eq. 5-6, Algorithm 1
def largest_safe(a, b, B_n: int, Kd: float, P: float, candidates: Sequence[int], tau: float, beta: float) -> int:
    """First chi in X (sorted decreasing) that satisfies Eq. 5; 0 if none.  Candidates that carry no
    prefill token (chi <= B_n) are skipped (G19)."""
    for chi in candidates:
        if chi <= B_n:
            continue
        if t_step(a, b, B_n, Kd, chi - B_n, P) <= beta * tau:
            return chi
    return 0


def build_schedule(a, b, B_n: int, K_n: float, prompt_len: int, candidates, tau, beta) -> Tuple[Optional[List[int]], float]:
    """The while loop of Algorithm 1 for one decode node, then Eq. 6."""
    X: List[int] = []
    Kd, served, ttft = float(K_n), 0, 0.0
    while served < prompt_len:
        chi = largest_safe(a, b, B_n, Kd, served, candidates, tau, beta)
        if chi == 0:
            return None, math.inf  # node n infeasible
        ttft += t_step(a, b, B_n, Kd, chi - B_n, served)
        X.append(chi)
        Kd += B_n                 # every in-flight decode appends its new token
        served += chi - B_n       # the chunk's prefill tokens (they become the request's cached prefix)
    return X, ttft


def decide(a, b, p, prompt_len: int, queue_lens, chi_p: int, nodes: Sequence[Tuple[int, float]], candidates, tau: float,
           beta: float, alpha: float, ttft_slo: float):
    """Algorithm 1.  Returns (decision, n_star, X_star, ttft_pf, ttft_dec)."""
    est_pf = ttft_pf(p, prompt_len, queue_lens, chi_p)
    F = []
    for n, (B_n, K_n) in enumerate(nodes):
        X, est = build_schedule(a, b, B_n, K_n, prompt_len, candidates, tau, beta)
        if X is not None:
            F.append((est, n, X))
    if not F:
        return "KEEP", -1, [], est_pf, math.inf
    est, n_star, X_star = min(F, key=lambda f: (f[0], f[1]))  # ties: the lowest node index
    if est <= alpha * est_pf and est <= ttft_slo:  # Eq. 7
        return "DEFLECT", n_star, X_star, est_pf, est
    return "KEEP", -1, [], est_pf, est
