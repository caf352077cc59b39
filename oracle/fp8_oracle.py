"""fp8 latent cache: codec, quantising append and decode attention -- TEST INFRASTRUCTURE, not the product.

Only tests/ and bench.py's cpu_baseline leg may import this.  The paper does not describe an fp8 cache (PAPER.md has no
such passage); SURVEY.md 8(f) row 4 lists "an fp8 latent-cache variant (halves the decode roofline)" as a next step, so the
format below IS the reading (G23).  Everything is plain numpy, the attention in float64; no code is shared with
csrc/fp8.cu.

G23  One cached token = 512 latent values as e4m3 codes (OCP 8-bit float: 1 sign, 4 exponent bits with bias 7, 3 mantissa
     bits, no infinities, 0x7f / 0xff = NaN, largest finite 448) + ONE float32 scale + its 64 RoPE key values kept in bf16.
     A page of 64 tokens is 41,216 bytes: codes [64][512] | RoPE bf16 [64][64] | scales float32 [64]  (644 B per token
     against 1,152 B in bf16).
     Quantisation of token t (all in float32, IEEE round-to-nearest-even; both sides take these decisions in this
     precision): amax = max_d |c_t[d]|;  s_t = amax / 448 (1 if amax = 0);  code_t[d] = e4m3_rne_satfinite(c_t[d] / s_t).
     The cached latent is c~_t[d] = s_t * value(code_t[d]) exactly (a real number, not rounded again); attention is the
     plain definition over c~ and the bf16 RoPE keys with the bf16 query:
       s[h,t] = sigma * (q_lat[h] . c~_t + q_rope[h] . kR_t),  p = softmax_t(s),  out[h,:] = sum_t p[h,t] c~_t.
"""
from __future__ import annotations

import numpy as np

PAGE = 64
LATENT = 512
ROPE = 64
HEADS = 16
PAGE_BYTES = PAGE * LATENT + PAGE * ROPE * 2 + PAGE * 4  # 41,216
OFF_ROPE = PAGE * LATENT                                  # 32,768
OFF_SCALE = OFF_ROPE + PAGE * ROPE * 2                    # 40,960
E4M3_MAX = 448.0


def _bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


# ---------------------------------------------------------------------------------------------- e4m3 codec
def e4m3_decode(code: np.ndarray) -> np.ndarray:
    """uint8 e4m3 codes -> float64 values (exact).  exponent field 0: subnormal m/8 * 2^-6; else (1 + m/8) * 2^(e-7)."""
    c = np.asarray(code, dtype=np.uint8).astype(np.int64)
    sign = np.where(c & 0x80, -1.0, 1.0)
    e = (c >> 3) & 0xF
    m = c & 0x7
    val = np.where(e == 0, m / 8.0 * 2.0 ** -6, (1.0 + m / 8.0) * np.exp2((e - 7).astype(np.float64)))
    val = np.where((c & 0x7F) == 0x7F, np.nan, val)
    return sign * val


def e4m3_encode(v: np.ndarray) -> np.ndarray:
    """float32 -> e4m3 code, round to nearest (ties to the even code), saturating at +-448.  Finite inputs only.

    Written from the format's definition: the representable magnitudes are k * 2^-9 for k = 0..7 (subnormal) and
    (8 + m) * 2^(E-3) for E = -6..8, m = 0..7 (without E = 8, m = 7, which is NaN); between 2^E and 2^(E+1) the spacing is
    2^(E-3).  Round |v| / spacing to the nearest integer, ties to even (numpy.rint), then clamp."""
    v = np.asarray(v, dtype=np.float32).astype(np.float64)  # float32 -> float64 is exact; everything below is exact in float64
    a = np.abs(v)
    E = np.floor(np.log2(np.maximum(a, 2.0 ** -20)))
    E = np.clip(E, -6, 8)                      # below 2^-6 the subnormal spacing 2^-9 applies
    # log2 of a float64 just below a power of two may round up: fix the exponent so that 2^E <= a < 2^(E+1) where a >= 2^-6
    E = np.where((a >= 2.0 ** -6) & (a < np.exp2(E)), E - 1, E)
    E = np.where((a >= 2.0 ** -6) & (a >= np.exp2(E + 1)), E + 1, E)
    E = np.clip(E, -6, 8)
    q = np.exp2(E - 3)                          # spacing
    k = np.rint(a / q)                          # nearest multiple, ties to even
    mag = np.minimum(k * q, E4M3_MAX)           # satfinite
    # magnitude -> (exponent field, mantissa)
    Em = np.floor(np.log2(np.maximum(mag, 2.0 ** -20)))
    Em = np.where(mag >= np.exp2(Em + 1), Em + 1, Em)
    Em = np.where(mag < np.exp2(Em), Em - 1, Em)
    normal = mag >= 2.0 ** -6
    ef = np.where(normal, Em + 7, 0).astype(np.int64)
    mf = np.where(normal, np.rint(mag / np.exp2(Em - 3)) - 8, np.rint(mag * 2.0 ** 9)).astype(np.int64)
    code = (ef << 3) | mf
    code = np.where(np.signbit(v), code | 0x80, code)
    return code.astype(np.uint8)


# ---------------------------------------------------------------------------------------------- quantising append
def quantize_tokens(latent_bits: np.ndarray):
    """latent bf16 bits uint16 [n,512] -> (codes uint8 [n,512], scales float32 [n]) by G23, in float32."""
    x = (np.ascontiguousarray(latent_bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)
    amax = np.max(np.abs(x), axis=1).astype(np.float32)
    scale = np.where(amax > 0, amax / np.float32(448.0), np.float32(1.0)).astype(np.float32)
    y = (x / scale[:, None]).astype(np.float32)           # float32 division, round to nearest
    return e4m3_encode(y), scale


def append(pool8: np.ndarray, latent_bits: np.ndarray, k_rope_bits: np.ndarray, page_table: np.ndarray, start_pos: int) -> None:
    """In place: token j of the request goes to position start_pos + j of its sequence, i.e. slot pos % 64 of page
    page_table[pos // 64] (the same indexing as the bf16 append).  pool8: uint8 [num_pages, 41216]."""
    assert pool8.dtype == np.uint8 and pool8.ndim == 2 and pool8.shape[1] == PAGE_BYTES
    codes, scale = quantize_tokens(latent_bits)
    rope = np.ascontiguousarray(k_rope_bits, dtype=np.uint16)
    for j in range(codes.shape[0]):
        pos = int(start_pos) + j
        page = pool8[int(page_table[pos // PAGE])]
        slot = pos % PAGE
        page[slot * LATENT:(slot + 1) * LATENT] = codes[j]
        page[OFF_ROPE + slot * ROPE * 2:OFF_ROPE + (slot + 1) * ROPE * 2] = rope[j].view(np.uint8)
        page[OFF_SCALE + slot * 4:OFF_SCALE + (slot + 1) * 4] = scale[j:j + 1].view(np.uint8)


def gather_tokens(pool8: np.ndarray, page_table: np.ndarray, n: int):
    """The first n cached tokens of a sequence, dequantised: (latent float64 [n,512], rope float64 [n,64])."""
    lat = np.empty((n, LATENT), np.float64)
    rope = np.empty((n, ROPE), np.float64)
    for g in range((n + PAGE - 1) // PAGE):
        page = pool8[int(page_table[g])]
        k = min(PAGE, n - g * PAGE)
        codes = page[:k * LATENT].reshape(k, LATENT)
        sc = page[OFF_SCALE:OFF_SCALE + k * 4].view(np.float32).astype(np.float64)
        lat[g * PAGE:g * PAGE + k] = e4m3_decode(codes) * sc[:, None]
        rope[g * PAGE:g * PAGE + k] = _bf16_bits_to_f64(page[OFF_ROPE:OFF_ROPE + k * ROPE * 2].view(np.uint16).reshape(k, ROPE))
    return lat, rope


# ---------------------------------------------------------------------------------------------- decode attention
def decode(pool8, q_dec_bits, dec_page_tables, dec_ctx_lens, sigma: float):
    """Decode attention over the fp8 cache (G23), float64.  Returns (out [B,16,512], lse [B,16]) as float64."""
    q = _bf16_bits_to_f64(q_dec_bits).reshape(-1, HEADS, LATENT + ROPE)
    B = q.shape[0]
    out = np.empty((B, HEADS, LATENT), np.float64)
    lse = np.empty((B, HEADS), np.float64)
    for i in range(B):
        n = int(dec_ctx_lens[i])
        lat, rope = gather_tokens(pool8, np.asarray(dec_page_tables)[i], n)
        s = sigma * (q[i, :, :LATENT] @ lat.T + q[i, :, LATENT:] @ rope.T)   # [16, n]
        m = s.max(axis=1, keepdims=True)
        e = np.exp(s - m)
        l = e.sum(axis=1, keepdims=True)
        out[i] = (e / l) @ lat
        lse[i] = (m + np.log(l))[:, 0]
    return out, lse
