"""-m gpu: kairos_run_schedule against the oracle, every row.

The prompt's outputs must equal the ONE-SHOT oracle prefill row for row (chunk invariance); every decode
output of every step must equal the oracle's decode over the context as it stands at that step (the decodes cache one
token per step, and "a decode equals the last row of the corresponding prefill"); the pool afterwards is
bit-identical to the oracle's appends; the CUDA-graph replay, the step-by-step timed mode and m separate
kairos_append_* / kairos_mixed_step calls give identical bits.
"""
import numpy as np
import pytest

from paper_2607_02043_b200 import workloads as W
from tests import helpers as Hp

pytestmark = pytest.mark.gpu


def _setup(seed, lens, prompt_len, prefix, m_steps, grow):
    """Pool + page tables sized for the decodes' growth and the whole prompt; per-step decode queries and new tokens."""
    rng = np.random.default_rng(seed)
    B = len(lens)
    final = [L + (m_steps if grow else 0) for L in lens]
    inp = W.make_inputs("sched", seed, final, prompt_len, prefix, q_scale=0.5, extra_pages=3)
    x = dict(inp=inp, lens=np.asarray(lens, np.int32))
    x["q_dec"] = W.f32_to_bf16_bits(np.float32(0.5) * rng.standard_normal((m_steps, B, 16, 576), dtype=np.float32))
    x["dec_lat"] = W.f32_to_bf16_bits(rng.standard_normal((m_steps, B, 512), dtype=np.float32))
    x["dec_rope"] = W.f32_to_bf16_bits(rng.standard_normal((m_steps, B, 64), dtype=np.float32))
    return x


def _oracle_schedule(x, chunks, prefix, grow):
    from oracle import oracle
    inp = x["inp"]
    pool = inp.pool.copy()
    B, m = len(x["lens"]), len(chunks)
    out_dec = np.zeros((m, B, 16, 512), np.float32)
    lse_dec = np.zeros((m, B, 16), np.float32)
    done = 0
    for i, C in enumerate(chunks):
        lens = x["lens"] + (i + 1 if grow else 0)
        if grow:
            for j in range(B):
                oracle.append(pool, x["dec_lat"][i, j:j + 1], x["dec_rope"][i, j:j + 1], inp.dec_page_tables[j], int(x["lens"][j]) + i)
        oracle.append(pool, inp.chunk_latent[done:done + C], inp.chunk_k_rope[done:done + C], inp.chunk_page_table, prefix + done)
        if B:
            out_dec[i], lse_dec[i] = oracle.attend_rows(pool, inp.dec_page_tables, inp.dec_table_stride, np.arange(B, dtype=np.int32),
                                                        x["q_dec"][i], lens.astype(np.int32), inp.softmax_scale)
        done += C
    # the prompt in ONE shot over the finished cache: row t sees prefix + t + 1 keys
    L = inp.chunk_len
    out_p, lse_p = oracle.attend_rows(pool, inp.chunk_page_table[None, :], inp.chunk_page_table.shape[0], np.zeros(L, np.int32),
                                      inp.q_chunk, (prefix + np.arange(L) + 1).astype(np.int32), inp.softmax_scale)
    return pool, out_dec, lse_dec, out_p, lse_p


CASES = [
    ("five_chunks_growing_decodes", dict(lens=[64, 200, 700, 1500], prompt_len=400, prefix=0, chunks=[128, 100, 1, 71, 100], grow=True)),
    ("prefix_and_fixed_decodes", dict(lens=[130, 2500], prompt_len=300, prefix=91, chunks=[150, 100, 50], grow=False)),
    ("no_decodes_long_prompt", dict(lens=[], prompt_len=1500, prefix=0, chunks=[512, 512, 476], grow=False)),
    ("single_step", dict(lens=[63], prompt_len=37, prefix=5, chunks=[37], grow=True)),
]


def _random_case(seed):
    """A seeded random schedule off the hand-picked ones: 2-6 chunks of 1-600 tokens, 0-11 decodes, any prefix."""
    rng = np.random.default_rng(300 + seed)
    B = int(rng.integers(0, 12))
    lens = [int(v) for v in rng.integers(1, 2000, B)]
    chunks = [int(v) for v in rng.integers(1, 600, int(rng.integers(2, 7)))]
    return (f"random{seed}", dict(lens=lens, prompt_len=sum(chunks), prefix=int(rng.integers(0, 700)), chunks=chunks,
                                  grow=bool(rng.integers(0, 2)) and B > 0))


CASES += [_random_case(s) for s in range(4)]


@pytest.mark.parametrize("name,kw", CASES, ids=[c[0] for c in CASES])
@pytest.mark.parametrize("pairs", [None, 0, 2])
def test_run_schedule_every_row(name, kw, pairs):
    import torch
    from paper_2607_02043_b200 import kairos as K
    chunks, prefix, grow = kw["chunks"], kw["prefix"], kw["grow"]
    x = _setup(200 + len(name), kw["lens"], kw["prompt_len"], prefix, len(chunks), grow)
    inp = x["inp"]
    pool_ref, rd, rld, rp, rlp = _oracle_schedule(x, chunks, prefix, grow)
    f = lambda t: W.bf16_bits_to_f32(K.bf16_bits(t))

    def fresh():
        run = Hp.GpuRun(inp, pairs=pairs)
        args = (K.bf16_tensor(x["q_dec"]), run.dec_pt, x["lens"], K.bf16_tensor(x["dec_lat"]) if grow else None,
                K.bf16_tensor(x["dec_rope"]) if grow else None, chunks, run.q_chunk, run.latent, run.k_rope, run.chunk_pt)
        return run, args

    # 1. the captured graph (twice: capture, then replay)
    run, args = fresh()
    od, op, ld, lp, ttft, _ = run.ctx.run_schedule(*args, prefix_len=prefix)
    assert run.ctx.last_plan_info()["graph"] == 1 and ttft > 0
    assert np.array_equal(run.pool_bits(), pool_ref), "pool after the schedule differs from the oracle's appends"
    got = (f(od), f(op), ld.cpu().numpy(), lp.cpu().numpy())
    Hp.assert_attention_close([got[0], got[1]], [rd, rp], f"{name}: schedule vs one-shot oracle prefill + per-step decodes")
    assert np.abs(got[3] - rlp).max() <= Hp.LSE_TOL
    if len(kw["lens"]):
        assert np.abs(got[2] - rld).max() <= Hp.LSE_TOL
    if not grow:  # replay on the same buffers (growing decodes would append at the same slots again: same bytes, also fine)
        od.fill_(float("nan")); op.fill_(float("nan"))
    od2, op2, ld2, lp2, ttft2, _ = run.ctx.run_schedule(*args, prefix_len=prefix, out_dec=od, out_prompt=op, lse_dec=ld, lse_prompt=lp)
    for a, b in zip(got, (f(od2), f(op2), ld2.cpu().numpy(), lp2.cpu().numpy())):
        assert np.array_equal(a, b)
    # 2. step-by-step timed mode on a fresh context
    run2, args2 = fresh()
    od3, op3, ld3, lp3, ttft3, steps = run2.ctx.run_schedule(*args2, prefix_len=prefix, time_steps=True)
    assert run2.ctx.last_plan_info()["graph"] == 0 and len(steps) == len(chunks) and np.all(steps > 0)
    assert steps.sum() <= ttft3 * 1.001
    for a, b in zip(got, (f(od3), f(op3), ld3.cpu().numpy(), lp3.cpu().numpy())):
        assert np.array_equal(a, b)
    # 3. m separate public calls
    run3, args3 = fresh()
    done, B = 0, len(kw["lens"])
    for i, C in enumerate(chunks):
        lens_i = x["lens"] + (i + 1 if grow else 0)
        if grow and B:
            pos = torch.from_numpy((x["lens"] + i).astype(np.int32)).cuda()
            run3.ctx.append_decode_tokens(args3[3][i], args3[4][i], run3.dec_pt, pos)
        run3.ctx.append_latent(run3.latent[done:done + C], run3.k_rope[done:done + C], run3.chunk_pt, prefix + done)
        o_d, o_c, l_d, l_c = run3.ctx.mixed_step(args3[0][i], run3.dec_pt, lens_i, run3.q_chunk[done:done + C], run3.chunk_pt, C, prefix + done)
        assert np.array_equal(f(o_c), got[1][done:done + C]) and np.array_equal(l_c.cpu().numpy(), got[3][done:done + C])
        if B:
            assert np.array_equal(f(o_d), got[0][i])
        done += C


def test_run_schedule_argument_errors():
    from paper_2607_02043_b200 import kairos as K
    x = _setup(9, [100], 64, 0, 2, True)
    run = Hp.GpuRun(x["inp"])
    args = lambda chunks: (K.bf16_tensor(x["q_dec"]), run.dec_pt, x["lens"], K.bf16_tensor(x["dec_lat"]), K.bf16_tensor(x["dec_rope"]),
                           chunks, run.q_chunk, run.latent, run.k_rope, run.chunk_pt)
    with pytest.raises(K.KairosError) as ei:   # a chunk of 0 tokens
        run.ctx.run_schedule(*args([64, 0]))
    assert ei.value.code == -1
    with pytest.raises(K.KairosError) as ei:   # prefix pushes the prompt beyond its page table
        run.ctx.run_schedule(*args([32, 32]), prefix_len=64)
    assert ei.value.code == -1
