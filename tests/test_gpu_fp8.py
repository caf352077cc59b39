"""GPU parity of the fp8 latent cache (include/kairos.h kairos_fp8_*): the quantising append bit for bit,
the decode attention within the bf16 path's tolerance, against oracle/fp8_oracle.py on the same seeded inputs.

Both sides build their own fp8 pool from the same bf16 tokens (the workloads module's draws): the oracle with numpy, the
library with kairos_fp8_append.  The pools start from the same random bytes, so stale slots hold arbitrary codes (NaN codes
included) on both sides."""
import numpy as np
import pytest

from oracle import fp8_oracle as F
from oracle import oracle as O
from paper_2607_02043_b200 import workloads as W
from tests.helpers import MAX_ABS_TOL, REL_L2_TOL, errors

pytestmark = pytest.mark.gpu


class Fp8Run:
    def __init__(self, inp: W.MixedStepInputs, oracle_requests=None, seed=99, knobs=None):
        import torch
        from paper_2607_02043_b200 import kairos as K
        self.K, self.torch, self.inp = K, torch, inp
        rng = np.random.default_rng(seed)
        init = rng.integers(0, 256, (inp.num_pages, F.PAGE_BYTES), dtype=np.uint8)
        self.pool8_ref = init.copy()
        self.pool8 = torch.from_numpy(init).cuda()
        self.pool16 = K.bf16_tensor(inp.pool)   # the context's bf16 pool (untouched by the fp8 calls)
        self.ws = torch.empty(K.workspace_bytes(max(inp.n_dec, 1), 1), dtype=torch.uint8, device="cuda")
        self.ctx = K.Kairos(self.pool16, self.ws, inp.softmax_scale)
        for k, v in (knobs or {}).items():
            self.ctx.debug_set(k, v)
        self.ctx.fp8_attach(self.pool8)
        self.dec_pt = torch.from_numpy(inp.dec_page_tables).cuda()
        self.q_dec = K.bf16_tensor(inp.q_dec)
        self.oracle_requests = list(range(inp.n_dec)) if oracle_requests is None else list(oracle_requests)
        # every request's tokens: gathered from the bf16 synthetic pool, quantised into both fp8 pools
        for i in range(inp.n_dec):
            L = int(inp.dec_ctx_lens[i])
            tok = O.gather(inp.pool, inp.dec_page_tables[i], L)
            lat, rope = np.ascontiguousarray(tok[:, :512]), np.ascontiguousarray(tok[:, 512:])
            self.ctx.fp8_append(K.bf16_tensor(lat), K.bf16_tensor(rope), self.dec_pt[i], 0)
            if i in self.oracle_requests:
                F.append(self.pool8_ref, lat, rope, inp.dec_page_tables[i], 0)
        torch.cuda.synchronize()

    def check_pool(self):
        got = self.pool8.cpu().numpy()
        for i in self.oracle_requests:
            n = (int(self.inp.dec_ctx_lens[i]) + 63) // 64
            for pg in self.inp.dec_page_tables[i, :n]:
                np.testing.assert_array_equal(got[pg], self.pool8_ref[pg], err_msg=f"request {i} page {pg}")

    def decode(self, **kw):
        od, lse = self.ctx.fp8_decode(self.q_dec, self.dec_pt, self.inp.dec_ctx_lens, **kw)
        self.torch.cuda.synchronize()
        return W.bf16_bits_to_f32(self.K.bf16_bits(od)), lse.cpu().numpy(), (od, lse)

    def reference(self):
        idx = np.asarray(self.oracle_requests)
        return F.decode(self.pool8_ref, self.inp.q_dec[idx], self.inp.dec_page_tables[idx], self.inp.dec_ctx_lens[idx], self.inp.softmax_scale)


def _assert_close(out, lse, ref_out, ref_lse, what, scale=1.0):
    """`scale`: the absolute bound is stated for unit-scale latents; a case that scales them passes its largest |reference|"""
    ma, rl = errors(out, ref_out)
    assert np.isfinite(out).all(), what
    assert ma <= MAX_ABS_TOL * max(1.0, scale) and rl <= REL_L2_TOL, f"{what}: max-abs {ma:.3e} rel-L2 {rl:.3e}"
    assert np.abs(lse - ref_lse).max() <= 2e-3, f"{what}: lse {np.abs(lse - ref_lse).max():.3e}"


@pytest.mark.parametrize("lens", [[64], [1], [63, 65], [1, 63, 64, 65, 200, 333, 1000, 2500]])
def test_append_bit_exact_and_decode_parity_small(lens):
    inp = W.make_inputs("fp8_small", 11, lens, 0, 0)
    r = Fp8Run(inp)
    r.check_pool()
    out, lse, _ = r.decode()
    ref_out, ref_lse = r.reference()
    _assert_close(out, lse, ref_out, ref_lse, f"lens {lens}")


def test_append_ragged_positions_bit_exact():
    """appends that start and end inside pages, in several calls, as a growing request does"""
    import torch
    from paper_2607_02043_b200 import kairos as K
    inp = W.make_inputs("fp8_ragged", 12, [300], 0, 0)
    r = Fp8Run(inp)
    rng = np.random.default_rng(5)
    pos = 300 - 300  # rewrite the request piecewise from position 0 with fresh tokens
    pt = inp.dec_page_tables[0]
    for n in [1, 62, 2, 64, 100, 71]:
        lat = W.f32_to_bf16_bits(rng.standard_normal((n, 512)).astype(np.float32) * np.float32(rng.uniform(0.01, 30)))
        rope = W.f32_to_bf16_bits(rng.standard_normal((n, 64)).astype(np.float32))
        if n == 2:
            lat[0] = 0  # an all-zero token: scale 1, codes 0
        r.ctx.fp8_append(K.bf16_tensor(lat), K.bf16_tensor(rope), r.dec_pt[0], pos)
        F.append(r.pool8_ref, lat, rope, pt, pos)
        pos += n
    torch.cuda.synchronize()
    np.testing.assert_array_equal(r.pool8.cpu().numpy(), r.pool8_ref)


def test_sharp_softmax_and_wide_scale_range():
    """q_scale 1.0 (peaked softmax) and token magnitudes spread over 2^-10 .. 2^10: the scale rides the softmax weight"""
    inp = W.make_inputs("fp8_sharp", 13, [500, 129, 2000, 70], 0, 0, q_scale=1.0)
    rng = np.random.default_rng(6)
    f = W.bf16_bits_to_f32(inp.pool)
    f[:, :, :512] *= np.exp2(rng.integers(-10, 11, (inp.num_pages, 64, 1))).astype(np.float32)
    inp.pool[:] = W.f32_to_bf16_bits(f)
    r = Fp8Run(inp)
    r.check_pool()
    out, lse, _ = r.decode()
    ref_out, ref_lse = r.reference()
    ma, rl = errors(out, ref_out)
    scale = np.abs(ref_out).max()
    assert np.isfinite(out).all()
    assert ma <= MAX_ABS_TOL * max(1.0, scale) and rl <= REL_L2_TOL, (ma, rl, scale)
    assert np.abs(lse - ref_lse).max() <= 5e-3


def test_repeated_calls_replay_the_same_result():
    """plan cache hit, then graph replay (same buffers): bit-identical outputs; a length moved inside a page: structural hit"""
    inp = W.make_inputs("fp8_repeat", 14, [700, 2500, 68, 135, 70], 0, 0)
    r = Fp8Run(inp)
    out0, lse0, bufs = r.decode()
    infos = []
    for _ in range(4):
        bufs[0].fill_(float("nan"))
        out, lse, _ = r.decode(out_dec=bufs[0], lse_dec=bufs[1])
        infos.append(r.ctx.last_plan_info())
        np.testing.assert_array_equal(out, out0)
        np.testing.assert_array_equal(lse, lse0)
    assert infos[-1]["plan_cache"] == 2 and infos[-1]["graph"] == 1, infos[-1]   # exact plan hit, replayed as a graph
    ref_out, ref_lse = r.reference()
    _assert_close(out0, lse0, ref_out, ref_lse, "repeat")
    # the bf16 step of the same context still works beside it (its own plan entry)
    e = r.torch.empty((0, 16, 576), dtype=r.torch.bfloat16, device="cuda")
    od, _, ld, _ = r.ctx.mixed_step(r.q_dec, r.dec_pt, inp.dec_ctx_lens, e, r.torch.zeros(1, dtype=r.torch.int32, device="cuda"), 0, 0)
    r.torch.cuda.synchronize()
    ref16 = O.mixed_step(inp.pool, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, 0, 0, np.zeros((0, 16, 576), np.uint16), np.zeros(1, np.int32), inp.softmax_scale)
    ma, rl = errors(W.bf16_bits_to_f32(r.K.bf16_bits(od)), ref16[0])
    assert ma <= MAX_ABS_TOL and rl <= REL_L2_TOL
    out, lse, _ = r.decode()
    np.testing.assert_array_equal(out, out0)


def test_config1_every_request():
    inp = W.make_config(1)
    inp = W.make_inputs("fp8_cfg1", 1, inp.dec_ctx_lens.tolist(), 0, 0)
    r = Fp8Run(inp)
    r.check_pool()
    out, lse, _ = r.decode()
    ref_out, ref_lse = r.reference()
    _assert_close(out, lse, ref_out, ref_lse, "configs[1] decodes")


def test_config3_sampled_requests():
    """BASELINE.json configs[3] at C = 0 (256 x 2048 tokens), the launch configuration bench.py times: 12 sampled requests"""
    inp = W.make_config(3, chunk_len=0)
    idx = sorted(set([0, 255] + np.random.default_rng(7).choice(256, 10, replace=False).tolist()))
    r = Fp8Run(inp, oracle_requests=idx)
    r.check_pool()
    out, lse, _ = r.decode()
    ref_out, ref_lse = r.reference()
    _assert_close(out[idx], lse[idx], ref_out, ref_lse, "configs[3] C=0 sampled")
    assert np.isfinite(out).all()
    info = r.ctx.last_plan_info()
    assert info["kernels"] == 2   # attention + combine


def test_errors():
    import torch
    from paper_2607_02043_b200 import kairos as K
    inp = W.make_inputs("fp8_err", 15, [100, 100], 0, 0)
    pool16 = K.bf16_tensor(inp.pool)
    ws = torch.empty(K.workspace_bytes(2, 1), dtype=torch.uint8, device="cuda")
    ctx = K.Kairos(pool16, ws, inp.softmax_scale)
    q = K.bf16_tensor(inp.q_dec)
    pt = torch.from_numpy(inp.dec_page_tables).cuda()
    with pytest.raises(K.KairosError) as e:
        ctx.fp8_decode(q, pt, inp.dec_ctx_lens)
    assert e.value.code == -1 and "attach" in str(e.value)
    pool8 = torch.zeros((inp.num_pages, K.FP8_PAGE_BYTES), dtype=torch.uint8, device="cuda")
    ctx.fp8_attach(pool8)
    with pytest.raises(K.KairosError) as e:
        ctx.fp8_append(q[0, 0, :512].reshape(1, 512).contiguous(), q[0, 0, 512:].reshape(1, 64).contiguous(), pt[0], 64 * pt.shape[1])
    assert e.value.code == -1


def test_append_decode_tokens_then_decode_a_growing_batch():
    """three decode steps: every request caches its newest token (batched fp8 append), then attends one token further"""
    import torch
    from paper_2607_02043_b200 import kairos as K
    lens0 = [63, 64, 127, 500, 1]
    inp = W.make_inputs("fp8_grow", 16, [L + 3 for L in lens0], 0, 0)   # page tables sized for the growth
    r = Fp8Run(inp)                                                      # both pools hold every request's first lens0 + 3 tokens
    rng = np.random.default_rng(8)
    lens = np.asarray(lens0, np.int32)
    for step in range(3):
        lat = W.f32_to_bf16_bits(rng.standard_normal((len(lens), 512)).astype(np.float32) * np.float32(2.0 ** rng.integers(-3, 4)))
        rope = W.f32_to_bf16_bits(rng.standard_normal((len(lens), 64)).astype(np.float32))
        pos = torch.from_numpy(lens.copy()).cuda()
        r.ctx.fp8_append_decode_tokens(K.bf16_tensor(lat), K.bf16_tensor(rope), r.dec_pt, pos)
        for i in range(len(lens)):
            F.append(r.pool8_ref, lat[i:i + 1], rope[i:i + 1], inp.dec_page_tables[i], int(lens[i]))
        lens = lens + 1
        od, lse = r.ctx.fp8_decode(r.q_dec, r.dec_pt, lens)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(r.pool8.cpu().numpy(), r.pool8_ref)
        ref_out, ref_lse = F.decode(r.pool8_ref, inp.q_dec, inp.dec_page_tables, lens, inp.softmax_scale)
        _assert_close(W.bf16_bits_to_f32(K.bf16_bits(od)), lse.cpu().numpy(), ref_out, ref_lse, f"growing batch step {step}",
                      scale=float(np.abs(ref_out).max()))


def _mixed_case(inp, r):
    """Cache the chunk's sequence (prefix from the synthetic pool, then the chunk's own tokens) on both sides; returns the chunk rows'
    reference inputs for F.decode: every chunk token is a one-token request over the chunk's page table (n_keys = P + j + 1)."""
    import torch
    K = r.K
    C, P = inp.chunk_len, inp.prefix_len
    cpt = torch.from_numpy(inp.chunk_page_table).cuda()
    if P:
        tok = O.gather(inp.pool, inp.chunk_page_table, P)
        lat, rope = np.ascontiguousarray(tok[:, :512]), np.ascontiguousarray(tok[:, 512:])
        r.ctx.fp8_append(K.bf16_tensor(lat), K.bf16_tensor(rope), cpt, 0)
        F.append(r.pool8_ref, lat, rope, inp.chunk_page_table, 0)
    r.ctx.fp8_append(K.bf16_tensor(inp.chunk_latent), K.bf16_tensor(inp.chunk_k_rope), cpt, P)
    F.append(r.pool8_ref, inp.chunk_latent, inp.chunk_k_rope, inp.chunk_page_table, P)
    rows_pt = np.tile(inp.chunk_page_table[None, :], (C, 1))
    rows_len = (P + 1 + np.arange(C)).astype(np.int32)
    return cpt, rows_pt, rows_len


def _random_mixed(seed):
    rng = np.random.default_rng(400 + seed)
    return ([int(v) for v in rng.integers(1, 1800, int(rng.integers(0, 10)))], int(rng.integers(1, 400)), int(rng.integers(0, 900)))


@pytest.mark.parametrize("lens,C,P", [([64, 128, 200, 256], 64, 128), ([300, 70], 100, 0), ([], 130, 61), ([1000, 2500, 65], 257, 700)]
                         + [_random_mixed(s) for s in range(4)])
def test_mixed_step_over_the_fp8_cache(lens, C, P):
    """kairos_fp8_mixed_step: decodes + a causal chunk, every row against the float64 definition over the dequantised cache"""
    inp = W.make_inputs("fp8_mixed", 17, lens, C, P)
    r = Fp8Run(inp)
    cpt, rows_pt, rows_len = _mixed_case(inp, r)
    q_chunk = r.K.bf16_tensor(inp.q_chunk)
    r.ws = r.torch.empty(r.K.workspace_bytes(inp.n_dec + C, 0), dtype=r.torch.uint8, device="cuda")
    ctx = r.K.Kairos(r.pool16, r.ws, inp.softmax_scale)
    ctx.fp8_attach(r.pool8)
    q_dec = r.q_dec if inp.n_dec else r.torch.empty((0, 16, 576), dtype=r.torch.bfloat16, device="cuda")
    dpt = r.dec_pt if inp.n_dec else r.torch.zeros((1, 1), dtype=r.torch.int32, device="cuda")
    outs = None
    for rep in range(3):   # plan miss, exact hit, graph replay: the same bits
        od, oc, ld, lc = ctx.fp8_mixed_step(q_dec, dpt, inp.dec_ctx_lens, q_chunk, cpt, C, P) if outs is None else \
            ctx.fp8_mixed_step(q_dec, dpt, inp.dec_ctx_lens, q_chunk, cpt, C, P, out_dec=outs[0], out_chunk=outs[1], lse_dec=outs[2], lse_chunk=outs[3])
        r.torch.cuda.synchronize()
        cur = [r.K.bf16_bits(od), r.K.bf16_bits(oc), ld.cpu().numpy(), lc.cpu().numpy()]
        if outs is not None:
            for a, b in zip(cur, first):
                np.testing.assert_array_equal(a, b)
        else:
            first = cur
        outs = (od, oc, ld, lc)
    np.testing.assert_array_equal(r.pool8.cpu().numpy(), r.pool8_ref)
    ref_c, ref_lc = F.decode(r.pool8_ref, inp.q_chunk, rows_pt, rows_len, inp.softmax_scale)
    _assert_close(W.bf16_bits_to_f32(first[1]), first[3], ref_c, ref_lc, f"chunk rows C={C} P={P}")
    if inp.n_dec:
        ref_d, ref_ld = F.decode(r.pool8_ref, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.softmax_scale)
        _assert_close(W.bf16_bits_to_f32(first[0]), first[2], ref_d, ref_ld, f"decode rows beside C={C}")


def test_mixed_step_config3_C512_in_the_bench_configuration():
    """BASELINE.json configs[3] with C = 512 over the fp8 cache, as bench.py's fp8 leg times it: every chunk row and 8 sampled decodes"""
    inp = W.make_config(3, chunk_len=512)
    idx = sorted(set([0, 255] + np.random.default_rng(9).choice(256, 6, replace=False).tolist()))
    r = Fp8Run(inp, oracle_requests=idx)
    cpt, rows_pt, rows_len = _mixed_case(inp, r)
    ws = r.torch.empty(r.K.workspace_bytes(inp.n_dec + inp.chunk_len, 0), dtype=r.torch.uint8, device="cuda")
    ctx = r.K.Kairos(r.pool16, ws, inp.softmax_scale)
    ctx.fp8_attach(r.pool8)
    od, oc, ld, lc = ctx.fp8_mixed_step(r.q_dec, r.dec_pt, inp.dec_ctx_lens, r.K.bf16_tensor(inp.q_chunk), cpt, inp.chunk_len, inp.prefix_len)
    r.torch.cuda.synchronize()
    out_d, out_c = W.bf16_bits_to_f32(r.K.bf16_bits(od)), W.bf16_bits_to_f32(r.K.bf16_bits(oc))
    assert np.isfinite(out_d).all() and np.isfinite(out_c).all()
    ref_c, ref_lc = F.decode(r.pool8_ref, inp.q_chunk, rows_pt, rows_len, inp.softmax_scale)
    _assert_close(out_c, lc.cpu().numpy(), ref_c, ref_lc, "configs[3] C=512 chunk rows")
    ref_d, ref_ld = r.reference()
    _assert_close(out_d[idx], ld.cpu().numpy()[idx], ref_d, ref_ld, "configs[3] C=512 sampled decodes")
    assert ctx.last_plan_info()["work_items"] >= 256 + 512
