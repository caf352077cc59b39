"""CPU-only pins of oracle/fp8_oracle.py (G23): the e4m3 codec against the format's printed constants, brute force
and torch's own float8_e4m3fn cast; the quantiser against its bounds; the attention against the already pinned bf16 oracle on
inputs the fp8 cache represents exactly, and against a closed form."""
import numpy as np
import pytest
import torch

from oracle import fp8_oracle as F
from oracle import oracle as O
from paper_2607_02043_b200 import workloads as W


def test_e4m3_decode_known_values():
    # OCP 8-bit floating point specification (E4M3): bias 7, max 448 = S.1111.110, min normal 2^-6, min subnormal 2^-9, NaN = S.1111.111
    known = {0x00: 0.0, 0x01: 2.0 ** -9, 0x07: 7 * 2.0 ** -9, 0x08: 2.0 ** -6, 0x38: 1.0, 0x3C: 1.5, 0x40: 2.0, 0x7E: 448.0,
             0xB8: -1.0, 0xFE: -448.0, 0x77: 240.0, 0x30: 0.5}
    codes = np.array(sorted(known), dtype=np.uint8)
    np.testing.assert_array_equal(F.e4m3_decode(codes), np.array([known[int(c)] for c in codes]))
    assert np.isnan(F.e4m3_decode(np.array([0x7F, 0xFF], np.uint8))).all()
    pos = F.e4m3_decode(np.arange(0, 0x7F, dtype=np.uint8))
    assert (np.diff(pos) > 0).all()          # codes order like their values
    assert len(pos) == 127


def test_e4m3_roundtrip_every_code():
    codes = np.array([c for c in range(256) if (c & 0x7F) != 0x7F], dtype=np.uint8)
    vals = F.e4m3_decode(codes).astype(np.float32)
    back = F.e4m3_encode(vals)
    # -0 keeps its sign bit
    np.testing.assert_array_equal(back, codes)


def _brute_encode(v):
    """nearest finite e4m3 value by exhaustive search; ties to the even code; saturating."""
    grid = F.e4m3_decode(np.arange(0, 0x7F, dtype=np.uint8))
    out = np.empty(v.shape, np.uint8)
    for i, x in enumerate(v.astype(np.float64)):
        a = min(abs(x), 448.0)
        d = np.abs(grid - a)
        best = np.flatnonzero(d == d.min())
        c = int(best[0]) if len(best) == 1 else int([b for b in best if b % 2 == 0][0])
        out[i] = c | (0x80 if np.signbit(x) else 0)
    return out


def test_e4m3_encode_against_brute_force_and_ties():
    rng = np.random.default_rng(0)
    grid = F.e4m3_decode(np.arange(0, 0x7F, dtype=np.uint8))
    mids = (grid[:-1] + grid[1:]) / 2                      # every tie point is exactly representable in float32
    v = np.concatenate([mids, -mids, np.nextafter(mids.astype(np.float32), np.float32(0)), np.nextafter(mids.astype(np.float32), np.float32(1e9)),
                        rng.uniform(-500, 500, 4000), rng.standard_normal(4000) * 0.01, rng.standard_normal(4000),
                        [448.0, 464.0, 1e6, -1e6, 2.0 ** -10, 2.0 ** -11, 3 * 2.0 ** -11, 0.0]]).astype(np.float32)
    np.testing.assert_array_equal(F.e4m3_encode(v), _brute_encode(v))


def test_e4m3_encode_matches_torch_cast_in_range():
    rng = np.random.default_rng(1)
    v = np.concatenate([rng.uniform(-448, 448, 20000), rng.standard_normal(20000) * 2.0 ** rng.integers(-12, 8, 20000)]).astype(np.float32)
    v = v[np.abs(v) <= 448]
    t = torch.from_numpy(v).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    np.testing.assert_array_equal(F.e4m3_encode(v), t)


def test_quantize_tokens_bounds_and_degenerate_rows():
    rng = np.random.default_rng(2)
    x = rng.standard_normal((50, 512)).astype(np.float32) * rng.uniform(1e-3, 1e3, (50, 1)).astype(np.float32)
    x[7] = 0.0
    bits = W.f32_to_bf16_bits(x)
    xb = W.bf16_bits_to_f32(bits).astype(np.float64)
    codes, scale = F.quantize_tokens(bits)
    assert scale.dtype == np.float32 and codes.dtype == np.uint8
    amax = np.abs(xb).max(axis=1)
    assert scale[7] == 1.0 and (codes[7] == 0).all()
    nz = amax > 0
    np.testing.assert_allclose(scale[nz].astype(np.float64) * 448.0, amax[nz], rtol=2e-7)
    # the largest element of a row is coded +-448
    top = np.abs(F.e4m3_decode(codes)).max(axis=1)
    assert (top[nz] == 448.0).all()
    # error bound: half a spacing, i.e. |c - c~| <= 2^-4 |c| for normal codes, and <= s * 2^-10 below the normal range
    deq = F.e4m3_decode(codes) * scale[:, None].astype(np.float64)
    err = np.abs(deq - xb)
    bound = np.maximum(np.abs(xb) * 2.0 ** -4, scale[:, None].astype(np.float64) * 2.0 ** -10) * (1 + 1e-6)
    assert (err <= bound).all()


def test_append_indexing_by_hand():
    rng = np.random.default_rng(3)
    pool = np.full((5, F.PAGE_BYTES), 0xAB, np.uint8)
    lat = W.f32_to_bf16_bits(rng.standard_normal((70, 512)).astype(np.float32))
    rope = W.f32_to_bf16_bits(rng.standard_normal((70, 64)).astype(np.float32))
    pt = np.array([3, 0, 4], np.int32)
    F.append(pool, lat, rope, pt, start_pos=60)        # positions 60..129: pages 3 (slots 60-63), 0 (all), 4 (slots 0, 1)
    codes, scale = F.quantize_tokens(lat)
    # token 0 -> page 3 slot 60; token 4 -> page 0 slot 0; token 69 -> page 4 slot 1
    for tok, page, slot in [(0, 3, 60), (3, 3, 63), (4, 0, 0), (67, 0, 63), (68, 4, 0), (69, 4, 1)]:
        np.testing.assert_array_equal(pool[page, slot * 512:(slot + 1) * 512], codes[tok])
        np.testing.assert_array_equal(pool[page, 32768 + slot * 128:32768 + (slot + 1) * 128].view(np.uint16), rope[tok])
        assert pool[page, 40960 + slot * 4:40960 + slot * 4 + 4].view(np.float32)[0] == scale[tok]
    # untouched: pages 1, 2 entirely; page 3 slots < 60; page 4 slots >= 2
    assert (pool[1] == 0xAB).all() and (pool[2] == 0xAB).all()
    assert (pool[3, :60 * 512] == 0xAB).all() and (pool[4, 2 * 512:32768] == 0xAB).all()
    assert (pool[3, 40960:40960 + 60 * 4] == 0xAB).all() and (pool[4, 40960 + 8:] == 0xAB).all()


def _exact_case(seed, lens):
    """Latents that the fp8 cache holds exactly: e4m3 values times a per-token power of two, each token containing +-448 * 2^k."""
    rng = np.random.default_rng(seed)
    grid = F.e4m3_decode(np.arange(0, 0x7F, dtype=np.uint8))
    n_pages = [(L + 63) // 64 for L in lens]
    num_pages = sum(n_pages)
    perm = rng.permutation(num_pages).astype(np.int32)
    stride = max(n_pages)
    dpt = np.zeros((len(lens), stride), np.int32)
    pool16 = W.f32_to_bf16_bits(rng.standard_normal((num_pages, 64, 576)).astype(np.float32))   # stale slots: finite garbage
    pool8 = rng.integers(0, 127, (num_pages, F.PAGE_BYTES)).astype(np.uint8)
    off = 0
    for i, L in enumerate(lens):
        dpt[i, :n_pages[i]] = perm[off:off + n_pages[i]]
        off += n_pages[i]
        lat = grid[rng.integers(0, 127, (L, 512))] * rng.choice([-1.0, 1.0], (L, 512))
        lat[np.arange(L), rng.integers(0, 512, L)] = 448.0
        lat *= np.exp2(rng.integers(-9, -5, (L, 1)).astype(np.float64))
        rope = rng.standard_normal((L, 64)).astype(np.float32)
        lb, rb = W.f32_to_bf16_bits(lat.astype(np.float32)), W.f32_to_bf16_bits(rope)
        assert (W.bf16_bits_to_f32(lb).astype(np.float64) == lat).all()      # 4 significant bits: exact in bf16
        F.append(pool8, lb, rb, dpt[i], 0)
        O.append(pool16, lb, rb, dpt[i], 0)
    q = W.f32_to_bf16_bits(0.3 * rng.standard_normal((len(lens), 16, 576)).astype(np.float32))
    return pool8, pool16, dpt, np.asarray(lens, np.int32), q


def test_decode_equals_bf16_oracle_on_exactly_representable_cache():
    pool8, pool16, dpt, lens, q = _exact_case(4, [1, 63, 64, 65, 200, 333])
    out8, lse8 = F.decode(pool8, q, dpt, lens, W.SOFTMAX_SCALE)
    out16, _, lse16, _ = O.mixed_step(pool16, q, dpt, lens, 0, 0, np.zeros((0, 16, 576), np.uint16), np.zeros(1, np.int32), W.SOFTMAX_SCALE)
    np.testing.assert_allclose(out8, out16, rtol=0, atol=2e-6 * np.abs(out16).max() + 1e-9)
    np.testing.assert_allclose(lse8, lse16, rtol=0, atol=2e-5)
    # and the dequantised tokens are the originals bit for bit
    lat, rope = F.gather_tokens(pool8, dpt[4], 200)
    g16 = W.bf16_bits_to_f32(O.gather(pool16, dpt[4], 200)).astype(np.float64)
    np.testing.assert_array_equal(lat, g16[:, :512])
    np.testing.assert_array_equal(rope, g16[:, 512:])


def test_decode_closed_form_uniform_attention():
    """q = 0: every visible token weighs 1/L, out = mean of the dequantised latents, lse = ln L; stale slots have no say."""
    pool8, _, dpt, lens, q = _exact_case(5, [70, 130])
    q[:] = 0
    out, lse = F.decode(pool8, q, dpt, lens, W.SOFTMAX_SCALE)
    for i, L in enumerate(lens):
        lat, _ = F.gather_tokens(pool8, dpt[i], int(L))
        np.testing.assert_allclose(out[i], np.broadcast_to(lat.mean(axis=0), (16, 512)), rtol=1e-12, atol=1e-15)
        np.testing.assert_allclose(lse[i], np.log(float(L)), rtol=1e-12)
