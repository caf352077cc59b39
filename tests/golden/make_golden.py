"""Writes tests/golden/closed_form_case.txt: expected outputs of a hand-derivable mixed step.

Uses only Python's `math` (no oracle, no CUDA path): the case is built so that every score is known in closed
form from the definition in SURVEY.md 8(c) / include/kairos.h (absorbed MLA: s_t = sigma (qC.c_t + qR.kR_t),
p = softmax, o = sum p_t c_t, lse = ln sum exp s_t; decode sees L keys, chunk row j sees P + j + 1 keys):

  sequence of T = 66 tokens (positions 0..65: crosses the page boundary at 64, ragged last page)
  c_t    = a_t * e_{t mod 512}            (one non-zero latent coordinate per token, value a_t = 1 + (t mod 4)/2)
  kR_t   = b_t * e_0                      (b_t = (t mod 3) - 1)
  head h query: qC = 0, qR = g_h * e_0    (g_h = 4 (h + 1)), the same for every query token
  => s_t = sigma * g_h * b_t,  o[t mod 512 coordinate] += p_t * a_t

Every input value is exactly representable in bf16.  Run: python tests/golden/make_golden.py
"""
import math
import os

SIGMA = 1.0 / math.sqrt(192.0)
T = 66
P = 60          # chunk: prefix 60, chunk 6 tokens (rows see 61..66 keys)
DEC_L = [1, 64, 65, 66]


def row(h, n):
    g = 4.0 * (h + 1)
    s = [SIGMA * g * ((t % 3) - 1) for t in range(n)]
    m = max(s)
    e = [math.exp(x - m) for x in s]
    z = math.fsum(e)
    out = {}
    for t in range(n):
        out[t % 512] = out.get(t % 512, 0.0) + e[t] / z * (1.0 + (t % 4) / 2.0)
    return out, m + math.log(z)


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_form_case.txt")
    with open(path, "w") as f:
        f.write("# kind index head n_keys lse then T values o[0..T-1] (coordinates >= T are 0); see make_golden.py\n")
        for kind, ns in (("dec", DEC_L), ("chunk", [P + j + 1 for j in range(T - P)])):
            for i, n in enumerate(ns):
                for h in (0, 7, 15):
                    o, lse = row(h, n)
                    vals = " ".join(repr(o.get(d, 0.0)) for d in range(T))
                    f.write(f"{kind} {i} {h} {n} {lse!r} {vals}\n")
    print(path)


if __name__ == "__main__":
    main()
