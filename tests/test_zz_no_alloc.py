"""kairos_decode_static -- the entry point that allocates nothing (its split-KV scratch is a fixed `static __device__` array of the
library) -- against the existing path (kairos_mixed_step with chunk_len = 0) on the same inputs, on two calls in a row.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests: it makes its
own context and inputs, and the shared array is rewritten by every call."""
import numpy as np
import pytest

from paper_2607_02043_b200 import workloads as W
from tests.helpers import MAX_ABS_TOL, REL_L2_TOL, LSE_TOL, errors

pytestmark = pytest.mark.gpu


def _setup(lens, seed):
    import torch
    from paper_2607_02043_b200 import kairos as K
    inp = W.make_inputs("no_alloc", seed, lens, 0, 0)
    pool = K.bf16_tensor(inp.pool)
    ws = torch.empty(K.workspace_bytes(inp.n_dec, 1), dtype=torch.uint8, device="cuda")
    ctx = K.Kairos(pool, ws, inp.softmax_scale)
    q = K.bf16_tensor(inp.q_dec)
    dpt = torch.from_numpy(inp.dec_page_tables).cuda()
    return K, torch, inp, ctx, q, dpt, (pool, ws)


def _existing(K, torch, inp, ctx, q, dpt):
    e = torch.empty((0, 16, 576), dtype=torch.bfloat16, device="cuda")
    od, _, ld, _ = ctx.mixed_step(q, dpt, inp.dec_ctx_lens, e, torch.zeros(1, dtype=torch.int32, device="cuda"), 0, 0)
    torch.cuda.synchronize()
    return W.bf16_bits_to_f32(K.bf16_bits(od)), ld.cpu().numpy()


def _static(K, torch, inp, ctx, q, dpt):
    od = torch.full((inp.n_dec, 16, 512), float("nan"), dtype=torch.bfloat16, device="cuda")
    ld = torch.full((inp.n_dec, 16), float("nan"), dtype=torch.float32, device="cuda")
    ctx.decode_static(q, dpt, inp.dec_ctx_lens, od, ld)
    torch.cuda.synchronize()
    return W.bf16_bits_to_f32(K.bf16_bits(od)), ld.cpu().numpy()


def _close(got, ref, what):
    ma, rl = errors(got[0], ref[0])
    assert np.isfinite(got[0]).all() and np.isfinite(got[1]).all(), what
    assert ma <= MAX_ABS_TOL and rl <= REL_L2_TOL, f"{what}: max-abs {ma:.3e} rel-L2 {rl:.3e}"
    assert np.abs(got[1] - ref[1]).max() <= LSE_TOL, f"{what}: lse {np.abs(got[1] - ref[1]).max():.3e}"


def test_decode_static_matches_the_existing_path_on_two_calls_in_a_row():
    # call 1: long and short requests (split pieces + whole requests, a ragged last page, a one-token request);
    # call 2 right behind it: other lengths, fewer requests -- whatever call 1 left in the shared array must not show
    a = _setup([4000, 65, 1, 700, 2500, 64, 63, 1300], seed=31)
    b = _setup([90, 5000, 257], seed=32)
    got_a = _static(*a[:6])
    got_b = _static(*b[:6])
    _close(got_a, _existing(*a[:6]), "call 1")
    _close(got_b, _existing(*b[:6]), "call 2")
    # the same call again gives the same bits (the plan is a pure function of the lengths; the combine order is fixed)
    again = _static(*b[:6])
    np.testing.assert_array_equal(again[0], got_b[0])
    np.testing.assert_array_equal(again[1], got_b[1])


def test_decode_static_allocates_no_device_memory_and_rejects_sizes_beyond_its_array():
    K, torch, inp, ctx, q, dpt, keep = _setup([300] * 128, seed=33)   # the maximum number of requests
    ref = _existing(K, torch, inp, ctx, q, dpt)
    od = torch.empty((inp.n_dec, 16, 512), dtype=torch.bfloat16, device="cuda")
    ld = torch.empty((inp.n_dec, 16), dtype=torch.float32, device="cuda")
    ctx.decode_static(q, dpt, inp.dec_ctx_lens, od, ld)               # first use loads the kernels
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        ctx.decode_static(q, dpt, inp.dec_ctx_lens, od, ld)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                      # cudaMemGetInfo: nothing was allocated (or freed)
    _close((W.bf16_bits_to_f32(K.bf16_bits(od)), ld.cpu().numpy()), ref, "128 requests")

    K2, torch, inp2, ctx2, q2, dpt2, keep2 = _setup([70] * 129, seed=34)
    od2 = torch.empty((129, 16, 512), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(K2.KairosError) as e:
        ctx2.decode_static(q2, dpt2, inp2.dec_ctx_lens, od2)
    assert e.value.code == -3 and "at most 128" in str(e.value)
