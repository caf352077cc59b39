"""-m gpu: kairos_absorb_q / kairos_project_out against oracle/proj_oracle.py, every element, and the
chain absorb -> kairos_mixed_step -> project_out against ordinary multi-head attention in float64."""
import numpy as np
import pytest

from paper_2607_02043_b200 import workloads as W
from tests import helpers as Hp

pytestmark = pytest.mark.gpu


def _bits(rng, shape, scale=1.0):
    return W.f32_to_bf16_bits(np.float32(scale) * rng.standard_normal(shape, dtype=np.float32))


@pytest.mark.parametrize("n", [1, 127, 128, 129, 700, 3, 255, 257, 1031, 2048])
def test_projections_every_element(n):
    from oracle import proj_oracle as P
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(n)
    run = Hp.GpuRun(W.make_inputs("p", 1, [64], 0, 0))
    qn, qr = _bits(rng, (n, 16, 128)), _bits(rng, (n, 16, 64))
    wk, wv = _bits(rng, (16, 512, 128), 0.1), _bits(rng, (16, 128, 512), 0.05)
    o = _bits(rng, (n, 16, 512))
    q_gpu = K.bf16_bits(run.ctx.absorb_q(K.bf16_tensor(qn), K.bf16_tensor(qr), K.bf16_tensor(wk)))
    want = P.absorb_q(qn, qr, wk)
    assert np.array_equal(q_gpu[:, :, 512:], qr), "RoPE part must pass through bit-exact"
    got = W.bf16_bits_to_f32(q_gpu).astype(np.float64)
    # bf16 result of an fp32-accumulated 128-term dot product: half an ulp of bf16 (2^-9 relative) plus accumulation noise
    assert np.abs(got - want).max() <= 2e-2 and np.linalg.norm(got - want) / np.linalg.norm(want) <= 5e-3
    assert np.all(np.abs(got - want) <= 2.0 ** -8 * np.abs(want) + 1e-3)
    v_gpu = W.bf16_bits_to_f32(K.bf16_bits(run.ctx.project_out(K.bf16_tensor(o), K.bf16_tensor(wv)))).astype(np.float64)
    want_v = P.project_out(o, wv)
    assert np.linalg.norm(v_gpu - want_v) / np.linalg.norm(want_v) <= 5e-3
    assert np.all(np.abs(v_gpu - want_v) <= 2.0 ** -8 * np.abs(want_v) + 2e-3)


def test_chain_equals_ordinary_multi_head_attention():
    """absorb_q -> kairos_mixed_step (decode rows over a paged cache) -> project_out vs float64 MHA with un-absorbed keys/values."""
    import torch
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(5)
    lens = [70, 200, 333]
    inp = W.make_inputs("chain", 9, lens, 0, 0, extra_pages=2)
    run = Hp.GpuRun(inp)
    B = len(lens)
    qn, qr = _bits(rng, (B, 16, 128), 0.3), _bits(rng, (B, 16, 64), 0.3)
    wk, wv = _bits(rng, (16, 512, 128), 0.05), _bits(rng, (16, 128, 512), 0.05)
    q = run.ctx.absorb_q(K.bf16_tensor(qn), K.bf16_tensor(qr), K.bf16_tensor(wk))
    e = torch.empty((0, 16, 576), dtype=torch.bfloat16, device="cuda")
    od, _, _, _ = run.ctx.mixed_step(q, run.dec_pt, inp.dec_ctx_lens, e, run.chunk_pt, 0, 0)
    v = W.bf16_bits_to_f32(K.bf16_bits(run.ctx.project_out(od, K.bf16_tensor(wv)))).astype(np.float64)
    f = lambda b: W.bf16_bits_to_f32(b).astype(np.float64)
    want = np.zeros((B, 16, 128))
    for i, L in enumerate(lens):
        t = np.arange(L)
        rows = f(inp.pool[inp.dec_page_tables[i][t // 64], t % 64])   # [L, 576]
        c, kr = rows[:, :512], rows[:, 512:]
        for h in range(16):
            k_h = np.concatenate([c @ f(wk)[h], kr], axis=1)
            v_h = c @ f(wv)[h].T
            s = inp.softmax_scale * (np.concatenate([f(qn)[i, h], f(qr)[i, h]]) @ k_h.T)
            p = np.exp(s - s.max()); p /= p.sum()
            want[i, h] = p @ v_h
    # three bf16 roundings in the chain (q, o_lat, v): a few times the single-step budget
    assert np.linalg.norm(v - want) / np.linalg.norm(want) <= 1.5e-2
