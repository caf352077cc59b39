"""Seeded synthetic inputs for the mixed-step MLA attention path (numpy only).

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2607_02043_b200.kairos``).  It holds no attention arithmetic: it
draws contexts, page tables, the latent pool and the queries, and rounds fp32
draws to bf16 bit patterns (round-to-nearest-even, done exactly once, here --
SURVEY.md 8(c) G10) so both sides consume identical bits.

Recipe (BASELINE.json ``configs``), draw order from
``np.random.default_rng(seed)``:

1. decode contexts: fixed list, or lognormal ``clip(rint(exp(ln(median)+sigma*z)), lo, hi)``
   with ``z = rng.standard_normal(B)`` drawn first (G18);
2. ``perm = rng.permutation(num_pages)``; consecutive slices go to decode 0..B-1,
   then to the chunk's sequence ("page tables are a random permutation of pages", G6);
3. the whole pool ``[num_pages, 64, 576]`` = N(0,1) -> bf16, page-batch by page-batch
   (stale slots therefore hold finite garbage, G7);
4. the chunk's own latent ``[C,512]`` and RoPE key ``[C,64]`` = N(0,1) -> bf16; they are
   written into the cache by the append call at ``start_pos = P`` (G4);
5. ``q_dec [B,16,576]`` and ``q_chunk [C,16,576]`` = q_scale * N(0,1) -> bf16 (G9: 0.1 for all
   configs; 1.0 is the sharper-softmax stress variant).

The paper's production traces (section 3) are proprietary; the lognormal
contexts stand in for its heavy-tailed prompt lengths (P25/median/P90 = 2071/3569/10336,
PAPER.md:88).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np

NUM_HEADS = 16
LATENT_DIM = 512
ROPE_DIM = 64
HEAD_DIM = LATENT_DIM + ROPE_DIM  # 576
PAGE_SIZE = 64
SOFTMAX_SCALE = 1.0 / math.sqrt(192.0)

TOKEN_BYTES = HEAD_DIM * 2                      # 1152 B per cached token
Q_BYTES = NUM_HEADS * HEAD_DIM * 2              # 18432 B per query token
OUT_BYTES = NUM_HEADS * LATENT_DIM * 2          # 16384 B per query token (bf16 out)
FLOP_PER_PAIR = NUM_HEADS * 2 * (HEAD_DIM + LATENT_DIM)  # 34816


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit pattern (uint16), round-to-nearest-even. Finite inputs only."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    b = x.view(np.uint32)
    r = (b + np.uint32(0x7FFF) + ((b >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> fp32, exact."""
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def lognormal_contexts(rng: np.random.Generator, n: int, median: float, sigma: float,
                       lo: int, hi: int) -> np.ndarray:
    z = rng.standard_normal(n)
    return np.clip(np.rint(np.exp(math.log(median) + sigma * z)), lo, hi).astype(np.int32)


@dataclasses.dataclass
class MixedStepInputs:
    """One mixed step: B decodes + one prefill chunk over a paged latent cache."""
    name: str
    seed: int
    num_pages: int
    pool: np.ndarray               # uint16 [num_pages, 64, 576]  (bf16 bits), chunk slots NOT yet appended
    dec_ctx_lens: np.ndarray       # int32 [B]
    dec_page_tables: np.ndarray    # int32 [B, dec_table_stride]  (unused entries = 0)
    dec_table_stride: int
    q_dec: np.ndarray              # uint16 [B, 16, 576]
    chunk_len: int                 # C
    prefix_len: int                # P
    chunk_page_table: np.ndarray   # int32 [ceil((P+C)/64)]
    chunk_latent: np.ndarray       # uint16 [C, 512]
    chunk_k_rope: np.ndarray       # uint16 [C, 64]
    q_chunk: np.ndarray            # uint16 [C, 16, 576]
    softmax_scale: float = SOFTMAX_SCALE

    @property
    def n_dec(self) -> int:
        return int(self.dec_ctx_lens.shape[0])

    def algorithmic_bytes(self) -> int:
        """each cached token read once per request, q in, out (bf16)."""
        dec = int(self.dec_ctx_lens.astype(np.int64).sum()) * TOKEN_BYTES + self.n_dec * (Q_BYTES + OUT_BYTES)
        ch = 0
        if self.chunk_len > 0:
            ch = (self.prefix_len + self.chunk_len) * TOKEN_BYTES + self.chunk_len * (Q_BYTES + OUT_BYTES)
        return dec + ch

    def algorithmic_flops(self) -> int:
        C, P = self.chunk_len, self.prefix_len
        pairs = int(self.dec_ctx_lens.astype(np.int64).sum()) + C * P + C * (C + 1) // 2
        return pairs * FLOP_PER_PAIR


def make_inputs(name: str, seed: int, dec_ctx_lens: Optional[Sequence[int]], chunk_len: int,
                prefix_len: int, *, lognormal: Optional[dict] = None, n_dec: Optional[int] = None,
                q_scale: float = 0.1, extra_pages: int = 0, page_batch: int = 4096) -> MixedStepInputs:
    """Generate one mixed step following the module-level recipe.

    ``lognormal`` = dict(median, sigma, lo, hi) with ``n_dec`` requests, or a fixed
    ``dec_ctx_lens`` list.  ``extra_pages`` adds unowned pages to the pool (they are part of
    the permutation, so owned pages are scattered among them).
    """
    rng = np.random.default_rng(seed)
    if lognormal is not None:
        lens = lognormal_contexts(rng, int(n_dec), **lognormal)
    else:
        lens = np.asarray(list(dec_ctx_lens or []), dtype=np.int32)
    B = int(lens.shape[0])
    C, P = int(chunk_len), int(prefix_len)
    dec_pages = [(int(L) + PAGE_SIZE - 1) // PAGE_SIZE for L in lens]
    chunk_pages = (P + C + PAGE_SIZE - 1) // PAGE_SIZE if C > 0 else 0
    num_pages = int(sum(dec_pages) + chunk_pages + extra_pages)
    num_pages = max(num_pages, 1)
    perm = rng.permutation(num_pages).astype(np.int32)
    stride = max(max(dec_pages, default=0), 1)
    dec_pt = np.zeros((B, stride), dtype=np.int32)
    off = 0
    for i, n in enumerate(dec_pages):
        dec_pt[i, :n] = perm[off:off + n]
        off += n
    chunk_pt = perm[off:off + chunk_pages].copy()
    off += chunk_pages

    pool = np.empty((num_pages, PAGE_SIZE, HEAD_DIM), dtype=np.uint16)
    for p0 in range(0, num_pages, page_batch):
        p1 = min(num_pages, p0 + page_batch)
        draw = rng.standard_normal((p1 - p0, PAGE_SIZE, HEAD_DIM), dtype=np.float32)
        pool[p0:p1] = f32_to_bf16_bits(draw)

    chunk_latent = f32_to_bf16_bits(rng.standard_normal((C, LATENT_DIM), dtype=np.float32))
    chunk_k_rope = f32_to_bf16_bits(rng.standard_normal((C, ROPE_DIM), dtype=np.float32))
    q_dec = f32_to_bf16_bits(np.float32(q_scale) * rng.standard_normal((B, NUM_HEADS, HEAD_DIM), dtype=np.float32))
    q_chunk = f32_to_bf16_bits(np.float32(q_scale) * rng.standard_normal((C, NUM_HEADS, HEAD_DIM), dtype=np.float32))
    return MixedStepInputs(name=name, seed=seed, num_pages=num_pages, pool=pool,
                           dec_ctx_lens=lens, dec_page_tables=dec_pt, dec_table_stride=stride,
                           q_dec=q_dec, chunk_len=C, prefix_len=P, chunk_page_table=chunk_pt,
                           chunk_latent=chunk_latent, chunk_k_rope=chunk_k_rope, q_chunk=q_chunk)


# BASELINE.json `configs` (index = list position; SURVEY.md calls them configs 1..5).
CONFIG_NAMES = ["pr1_ref", "steady_state", "heavy_tail", "chunk_sweep", "long_context"]
SWEEP_CHUNKS = [0, 256, 512, 1024, 2048, 4096, 8192]


def make_config(index: int, *, chunk_len: Optional[int] = None, q_scale: float = 0.1) -> MixedStepInputs:
    """BASELINE.json configs[index]; ``chunk_len`` selects the sweep point of configs[3]."""
    if index == 0:
        return make_inputs("pr1_ref", 0, [64, 128, 200, 256], 64, 128, q_scale=q_scale)
    if index == 1:
        return make_inputs("steady_state", 1, None, 512, 0, n_dec=64, q_scale=q_scale,
                           lognormal=dict(median=1024, sigma=0.8, lo=64, hi=8192))
    if index == 2:
        return make_inputs("heavy_tail", 2, None, 2048, 6144, n_dec=128, q_scale=q_scale,
                           lognormal=dict(median=2048, sigma=1.0, lo=64, hi=16384))
    if index == 3:
        C = 512 if chunk_len is None else int(chunk_len)
        return make_inputs(f"chunk_sweep_C{C}", 3, [2048] * 256, C, 0, q_scale=q_scale)
    if index == 4:
        return make_inputs("long_context", 4, [32768] * 32, 4096, 28672, q_scale=q_scale)
    raise ValueError(f"no such config index {index}")


def make_arrivals(seed: int, n: int, rate: float, burst_every: float, burst_size: int, prompt_median: float = 3569.0,
                  prompt_sigma: float = 0.8, prompt_lo: int = 64, prompt_hi: int = 16384, out_median: float = 200.0,
                  out_sigma: float = 0.6, out_lo: int = 1, out_hi: int = 2000):
    """Synthetic bursty arrivals for the policy simulator: a Poisson stream of `rate` requests per time
    unit plus `burst_size` simultaneous-ish requests every `burst_every` time units (the paper's Bursty trace is proprietary,
    PAPER.md:86-90; its prompt lengths have median 3569, P25/P90 = 2071/10336, i.e. lognormal sigma ~ 0.8).
    Returns a list of (arrival, prompt_len, output_len) sorted by arrival.  No method arithmetic here."""
    rng = np.random.default_rng(seed)
    n_burst = 0
    t_end = n / max(rate, 1e-12)
    if burst_every > 0 and burst_size > 0:
        n_burst = min(n // 2, int(t_end / burst_every) * burst_size)
    base = np.cumsum(rng.exponential(1.0 / rate, n - n_burst))
    bursts = []
    for k in range(n_burst):
        bursts.append((k // burst_size + 1) * burst_every + 1e-3 * burst_every * rng.random())
    t = np.sort(np.concatenate([base, np.asarray(bursts, dtype=np.float64)]))
    prompts = np.clip(np.rint(np.exp(math.log(prompt_median) + prompt_sigma * rng.standard_normal(n))), prompt_lo, prompt_hi).astype(np.int64)
    outs = np.clip(np.rint(np.exp(math.log(out_median) + out_sigma * rng.standard_normal(n))), out_lo, out_hi).astype(np.int64)
    return [(float(t[i]), int(prompts[i]), int(outs[i])) for i in range(n)]
