"""CPU-only: pins of oracle/proj_oracle.py against what the mathematics fixes."""
import numpy as np

from oracle import proj_oracle as P
from paper_2607_02043_b200 import workloads as W


def test_identity_and_one_hot_weights_by_hand():
    rng = np.random.default_rng(0)
    qn = rng.standard_normal((3, 16, 128))
    qr = rng.standard_normal((3, 16, 64))
    w = np.zeros((16, 512, 128))
    for h in range(16):
        w[h, np.arange(128) + h, np.arange(128)] = 1.0      # head h copies its 128 inputs to outputs h .. h+127
    q = P.absorb_q(qn, qr, w)
    assert q.shape == (3, 16, 576)
    for h in range(16):
        assert np.array_equal(q[:, h, h:h + 128], qn[:, h]) and np.count_nonzero(q[:, h, :512]) == 3 * 128
    assert np.array_equal(q[:, :, 512:], qr)                 # the RoPE part passes through
    w2 = np.zeros((16, 128, 512)); w2[5, 7, 300] = 2.0       # one weight: v[j,5,7] = 2 * o[j,5,300]
    o = rng.standard_normal((4, 16, 512))
    v = P.project_out(o, w2)
    assert v.shape == (4, 16, 128) and np.count_nonzero(v) == 4 and np.allclose(v[:, 5, 7], 2 * o[:, 5, 300])
    # a transposed weight would read w[h,k,d]: the one-hot test above fails for it (shape 512 x 128 vs 128 x 512 differ)


def test_bf16_bit_patterns_are_decoded_exactly():
    x = np.array([[[1.5] * 128] * 16], np.float32)
    bits = W.f32_to_bf16_bits(x)
    w = np.zeros((16, 512, 128)); w[:, 0, :] = 1.0
    assert np.allclose(P.absorb_q(bits, W.f32_to_bf16_bits(np.zeros((1, 16, 64), np.float32)), w)[0, :, 0], 1.5 * 128)


def test_absorbed_attention_equals_ordinary_mha():
    """W_UV . softmax(q_abs . [c | kR]) c  ==  softmax([q_nope | q_rope] . [W_UK c | kR]) (W_UV c): the 576/512 form the
    library computes is the cited model's attention (SURVEY.md 8(c) pin 'absorbed = un-absorbed')."""
    rng = np.random.default_rng(1)
    n_keys, sigma = 37, 1.0 / np.sqrt(192.0)
    c = rng.standard_normal((n_keys, 512)); kr = rng.standard_normal((n_keys, 64))
    qn = rng.standard_normal((2, 16, 128)) * 0.3; qr = rng.standard_normal((2, 16, 64)) * 0.3
    w_uk_t = rng.standard_normal((16, 512, 128)) * 0.05   # [h][d][k]: k_nope[t,h,k] = sum_d c[t,d] w[h,d,k]
    w_uv_t = rng.standard_normal((16, 128, 512)) * 0.05   # [h][e][d]: v[t,h,e] = sum_d c[t,d] w[h,e,d]
    # ordinary multi-head attention, written out with explicit loops over heads and a dense softmax
    want = np.zeros((2, 16, 128))
    for h in range(16):
        k_h = np.concatenate([c @ w_uk_t[h], kr], axis=1)            # [t, 128 + 64]
        v_h = c @ w_uv_t[h].T                                        # [t, 128]
        for j in range(2):
            s = sigma * (np.concatenate([qn[j, h], qr[j, h]]) @ k_h.T)
            p = np.exp(s - s.max()); p /= p.sum()
            want[j, h] = p @ v_h
    # absorbed form through the oracle's two projections
    q = P.absorb_q(qn, qr, w_uk_t)
    o = np.zeros((2, 16, 512))
    keys = np.concatenate([c, kr], axis=1)
    for h in range(16):
        for j in range(2):
            s = sigma * (q[j, h] @ keys.T)
            p = np.exp(s - s.max()); p /= p.sum()
            o[j, h] = p @ c
    got = P.project_out(o, w_uv_t)
    assert np.allclose(got, want, rtol=1e-10, atol=1e-12)
