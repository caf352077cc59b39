"""tests/golden/closed_form_case.txt (written by tests/golden/make_golden.py from the definition with Python's
`math` only) against the oracle (CPU) and against the CUDA path (-m gpu)."""
import os

import numpy as np
import pytest

from paper_2607_02043_b200 import workloads as W

T, P = 66, 60
DEC_L = [1, 64, 65, 66]
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "closed_form_case.txt")


def _load():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#"):
                continue
            p = line.split()
            rows.append((p[0], int(p[1]), int(p[2]), int(p[3]), float(p[4]), np.array([float(x) for x in p[5:]])))
    assert len(rows) == 3 * (len(DEC_L) + T - P)
    return rows


def _inputs():
    """The case of make_golden.py as pool / page tables / queries (all values bf16-exact)."""
    rng = np.random.default_rng(123)
    num_pages = 5
    pt = rng.permutation(num_pages).astype(np.int32)[:2]
    pool_f = rng.standard_normal((num_pages, 64, 576)).astype(np.float32)  # stale slots: finite garbage
    lat = np.zeros((T, 512), np.float32)
    rope = np.zeros((T, 64), np.float32)
    for t in range(T):
        lat[t, t % 512] = 1.0 + (t % 4) / 2.0
        rope[t, 0] = (t % 3) - 1
    for t in range(P):  # prefix already cached; the chunk's own tokens go through append
        pool_f[pt[t // 64], t % 64, :512] = lat[t]
        pool_f[pt[t // 64], t % 64, 512:] = rope[t]
    q = np.zeros((16, 576), np.float32)
    q[:, 512] = 4.0 * (np.arange(16) + 1)
    C = T - P
    bits = W.f32_to_bf16_bits
    for a in (lat, rope, q):
        assert np.array_equal(W.bf16_bits_to_f32(bits(a)), a)  # exactly representable
    return dict(pool=bits(pool_f), pt=pt, lat=bits(lat[P:]), rope=bits(rope[P:]),
                q_dec=bits(np.broadcast_to(q, (len(DEC_L), 16, 576)).copy()), q_chunk=bits(np.broadcast_to(q, (C, 16, 576)).copy()),
                dec_pt=np.broadcast_to(pt, (len(DEC_L), 2)).copy(), lens=np.array(DEC_L, np.int32), C=C)


def _check(od, oc, ld, lc, atol, ltol):
    for kind, i, h, n, lse, vals in _load():
        o, l = (od, ld) if kind == "dec" else (oc, lc)
        assert abs(float(l[i, h]) - lse) <= ltol, (kind, i, h)
        assert np.abs(o[i, h, :T].astype(np.float64) - vals).max() <= atol, (kind, i, h)
        assert np.abs(o[i, h, T:]).max() == 0.0


def test_oracle_matches_closed_form_golden():
    from oracle import oracle
    x = _inputs()
    pool = x["pool"].copy()
    oracle.append(pool, x["lat"], x["rope"], x["pt"], P)
    od, oc, ld, lc = oracle.mixed_step(pool, x["q_dec"], x["dec_pt"], x["lens"], x["C"], P, x["q_chunk"], x["pt"],
                                       W.SOFTMAX_SCALE)
    _check(od, oc, ld, lc, atol=2e-6, ltol=5e-6)


@pytest.mark.gpu
def test_cuda_matches_closed_form_golden():
    import torch
    from paper_2607_02043_b200 import kairos as K
    x = _inputs()
    pool = K.bf16_tensor(x["pool"])
    ws = torch.empty(K.workspace_bytes(8, 8), dtype=torch.uint8, device="cuda")
    ctx = K.Kairos(pool, ws, W.SOFTMAX_SCALE)
    pt = torch.from_numpy(x["pt"]).cuda()
    ctx.append_latent(K.bf16_tensor(x["lat"]), K.bf16_tensor(x["rope"]), pt, P)
    od, oc, ld, lc = ctx.mixed_step(K.bf16_tensor(x["q_dec"]), torch.from_numpy(x["dec_pt"]).cuda(), x["lens"],
                                    K.bf16_tensor(x["q_chunk"]), pt, x["C"], P)
    torch.cuda.synchronize()
    f = lambda t: W.bf16_bits_to_f32(K.bf16_bits(t))
    _check(f(od), f(oc), ld.cpu().numpy(), lc.cpu().numpy(), atol=2e-2, ltol=1e-3)
