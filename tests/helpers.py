"""Shared test plumbing: run one MixedStepInputs through the C-ABI on the GPU and through the oracle on the CPU.

The comparison rule (BASELINE.json north_star): GPU bf16 outputs are upcast exactly to fp32
and compared with the oracle's unrounded fp32: max-abs <= 2e-2 and relative L2 <= 5e-3 over decode + chunk
outputs concatenated.  Cache append / gather are compared bit for bit.
"""
from __future__ import annotations

import numpy as np

from oracle import oracle
from paper_2607_02043_b200 import workloads as W

MAX_ABS_TOL = 2e-2
REL_L2_TOL = 5e-3
LSE_TOL = 1e-3


def oracle_pool_after_append(inp: W.MixedStepInputs) -> np.ndarray:
    pool = inp.pool.copy()
    if inp.chunk_len:
        oracle.append(pool, inp.chunk_latent, inp.chunk_k_rope, inp.chunk_page_table, inp.prefix_len)
    return pool


class GpuRun:
    """Uploads the inputs, appends the chunk, runs kairos_mixed_step.  Keeps device tensors for reuse.

    `pairs` forces the launch order of the two grids through the test-only kairos_debug_set (None = the planner decides);
    `knobs` = further kairos_debug_set pairs, e.g. dict(graph=0, plan_cache=0).
    """

    def __init__(self, inp: W.MixedStepInputs, workspace_bytes=None, pairs=None, knobs=None):
        import torch
        from paper_2607_02043_b200 import kairos as K
        self.K, self.torch, self.inp = K, torch, inp
        self.pool = K.bf16_tensor(inp.pool)
        ws = K.workspace_bytes(max(inp.n_dec, 1), max(inp.chunk_len, 1)) if workspace_bytes is None else workspace_bytes
        self.ws = torch.empty(ws, dtype=torch.uint8, device="cuda")
        self.ctx = K.Kairos(self.pool, self.ws, inp.softmax_scale)
        if pairs is not None:
            self.ctx.debug_set("pairs", pairs)
        for k, v in (knobs or {}).items():
            self.ctx.debug_set(k, v)
        dev = "cuda"
        self.q_dec = K.bf16_tensor(inp.q_dec)
        self.q_chunk = K.bf16_tensor(inp.q_chunk)
        self.dec_pt = torch.from_numpy(inp.dec_page_tables).to(dev)
        self.chunk_pt = torch.from_numpy(inp.chunk_page_table).to(dev)
        self.latent = K.bf16_tensor(inp.chunk_latent)
        self.k_rope = K.bf16_tensor(inp.chunk_k_rope)
        self.out = None

    def append(self):
        if self.inp.chunk_len:
            self.ctx.append_latent(self.latent, self.k_rope, self.chunk_pt, self.inp.prefix_len)

    def step(self, reuse_outputs=False):
        """One kairos_mixed_step.  reuse_outputs: pass the previous call's output tensors again (same pointers: the
        plan's kernels are then replayed as a CUDA graph from the second such call on), poisoned first."""
        i = self.inp
        kw = {}
        if reuse_outputs and self.out is not None:
            for t in self.out:
                t.fill_(float("nan"))
            kw = dict(out_dec=self.out[0], out_chunk=self.out[1], lse_dec=self.out[2], lse_chunk=self.out[3])
        self.out = self.ctx.mixed_step(self.q_dec, self.dec_pt, i.dec_ctx_lens, self.q_chunk, self.chunk_pt,
                                       i.chunk_len, i.prefix_len, **kw)
        od, oc, ld, lc = self.out
        self.torch.cuda.synchronize()
        f = lambda t: W.bf16_bits_to_f32(self.K.bf16_bits(t))
        return f(od), f(oc), ld.cpu().numpy(), lc.cpu().numpy()

    def pool_bits(self) -> np.ndarray:
        return self.K.bf16_bits(self.pool)


def errors(gpu: np.ndarray, ref: np.ndarray):
    g = gpu.astype(np.float64).ravel()
    r = ref.astype(np.float64).ravel()
    if r.size == 0:
        return 0.0, 0.0
    return float(np.abs(g - r).max()), float(np.linalg.norm(g - r) / np.linalg.norm(r))


def assert_attention_close(gpu_parts, ref_parts, what=""):
    g = np.concatenate([p.ravel() for p in gpu_parts])
    r = np.concatenate([p.ravel() for p in ref_parts])
    assert np.all(np.isfinite(g)), f"{what}: non-finite GPU output"
    max_abs, rel = errors(g, r)
    assert max_abs <= MAX_ABS_TOL and rel <= REL_L2_TOL, f"{what}: max_abs={max_abs:.3e} rel_l2={rel:.3e}"
    return max_abs, rel


def sample_indices(n: int, k: int, rng, always=()):
    if n <= k:
        return np.arange(n, dtype=np.int32)
    s = set(int(x) for x in always if 0 <= x < n)
    while len(s) < k:
        s.add(int(rng.integers(0, n)))
    return np.array(sorted(s), dtype=np.int32)


def oracle_sampled(inp: W.MixedStepInputs, pool_np: np.ndarray, dec_idx: np.ndarray, chunk_idx: np.ndarray):
    """Oracle rows for a subset of decodes and chunk tokens (rows are independent, so parity on them is exact)."""
    out_d = lse_d = out_c = lse_c = None
    if len(dec_idx):
        out_d, lse_d = oracle.attend_rows(pool_np, inp.dec_page_tables, inp.dec_table_stride, dec_idx,
                                          inp.q_dec[dec_idx], inp.dec_ctx_lens[dec_idx], inp.softmax_scale)
    if len(chunk_idx):
        out_c, lse_c = oracle.attend_rows(pool_np, inp.chunk_page_table[None, :], inp.chunk_page_table.shape[0],
                                          np.zeros(len(chunk_idx), np.int32), inp.q_chunk[chunk_idx],
                                          (inp.prefix_len + chunk_idx + 1).astype(np.int32), inp.softmax_scale)
    return out_d, lse_d, out_c, lse_c
