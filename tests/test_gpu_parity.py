"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): cache append and page indexing bit-exact; attention max-abs <= 2e-2 and
relative L2 <= 5e-3 (bf16 in, fp32 accumulation).  Every test compares EVERY row: the small and edge cases, and BASELINE.json configs[1]-[4] at
full size in the launch configuration bench.py times ("Parity for configs 1-4 is always over all rows").
"""
import numpy as np
import pytest

from paper_2607_02043_b200 import workloads as W
from tests import helpers as Hp

pytestmark = pytest.mark.gpu

def _full_compare(inp, check_append=True, pairs=None, knobs=None):
    from oracle import oracle
    run = Hp.GpuRun(inp, pairs=pairs, knobs=knobs)
    run.append()
    pool_np = Hp.oracle_pool_after_append(inp)
    if check_append:
        assert np.array_equal(run.pool_bits(), pool_np), "append: pool bytes differ"
    od, oc, ld, lc = run.step()
    rd, rc, rld, rlc = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len,
                                         inp.prefix_len, inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
    e = Hp.assert_attention_close([od, oc], [rd, rc], f"{inp.name}/pairs={pairs}")
    if od.size:
        assert np.abs(ld - rld).max() <= Hp.LSE_TOL
    if oc.size:
        assert np.abs(lc - rlc).max() <= Hp.LSE_TOL
    return run, (od, oc, ld, lc), e


# ------------------------------------------------------------------ append / gather: bit-exact
def test_append_and_gather_bit_exact():
    import torch
    from oracle import oracle
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(0)
    num_pages = 40
    pool_np = np.full((num_pages, 64, 576), 0xABCD, np.uint16)
    pt = rng.permutation(num_pages).astype(np.int32)[:30]
    pool = K.bf16_tensor(pool_np)
    ws = torch.empty(K.workspace_bytes(1, 1), dtype=torch.uint8, device="cuda")
    ctx = K.Kairos(pool, ws)
    pt_d = torch.from_numpy(pt).cuda()
    for n, start in [(1, 0), (100, 37), (64, 64), (1, 1919), (700, 900)]:
        lat = rng.integers(0, 2 ** 16, (n, 512), dtype=np.uint16)
        rope = rng.integers(0, 2 ** 16, (n, 64), dtype=np.uint16)
        ctx.append_latent(K.bf16_tensor(lat), K.bf16_tensor(rope), pt_d, start)
        oracle.append(pool_np, lat, rope, pt, start)
        torch.cuda.synchronize()
        assert np.array_equal(K.bf16_bits(pool), pool_np), (n, start)
    g = ctx.gather_latent(pt_d, 1777)
    assert np.array_equal(K.bf16_bits(g), oracle.gather(pool_np, pt, 1777))
    # batched one-token-per-request append; request i owns its own 4 pages, so the target slots are distinct by construction
    n = 7
    pts = rng.permutation(num_pages).astype(np.int32)[:4 * n].reshape(n, 4)
    pos = rng.integers(0, 256, n).astype(np.int32)
    lat = rng.integers(0, 2 ** 16, (n, 512), dtype=np.uint16)
    rope = rng.integers(0, 2 ** 16, (n, 64), dtype=np.uint16)
    ctx.append_decode_tokens(K.bf16_tensor(lat), K.bf16_tensor(rope), torch.from_numpy(pts).cuda(),
                             torch.from_numpy(pos).cuda())
    torch.cuda.synchronize()
    for i in range(n):
        oracle.append(pool_np, lat[i:i + 1], rope[i:i + 1], pts[i], int(pos[i]))
    assert np.array_equal(K.bf16_bits(pool), pool_np)
    # error paths: detected on the host, nothing enqueued
    with pytest.raises(K.KairosError) as ei:
        ctx.append_latent(K.bf16_tensor(lat), K.bf16_tensor(rope), pt_d, 30 * 64 - 3)
    assert ei.value.code == -1


# ------------------------------------------------------------------ BASELINE.json configs[0]: every row
def test_config0_pr1_ref():
    _full_compare(W.make_config(0))


def test_config0_unscaled_q():
    """G9: sharper softmax (score std ~1.7) exercises the running-max / rescale path."""
    _full_compare(W.make_config(0, q_scale=1.0))


# ------------------------------------------------------------------ edge cases (every row)
EDGE = [
    ("decode_only", dict(dec_ctx_lens=[1, 2, 63, 64, 65, 700], chunk_len=0, prefix_len=0)),
    ("chunk_only_ragged", dict(dec_ctx_lens=[], chunk_len=37, prefix_len=91)),
    ("chunk_one_token_no_prefix", dict(dec_ctx_lens=[5], chunk_len=1, prefix_len=0)),
    ("chunk_crosses_pages", dict(dec_ctx_lens=[130], chunk_len=130, prefix_len=63)),
    ("long_decode_split", dict(dec_ctx_lens=[9000, 64, 4097], chunk_len=6, prefix_len=300)),
    ("few_tiles_long_prefix", dict(dec_ctx_lens=[], chunk_len=10, prefix_len=5000)),
]


@pytest.mark.parametrize("name,kw", EDGE, ids=[e[0] for e in EDGE])
def test_edge_cases(name, kw):
    inp = W.make_inputs(name, 100 + len(name), q_scale=0.5, extra_pages=3, **kw)
    _full_compare(inp)


# ------------------------------------------------------------------ the chunk on 2-CTA clusters (attn_pair.cu), forced
# The planner only moves the chunk to the pair kernel for large chunks (configs[2], [3] at C >= 2048, [4]); here it is
# forced so that every row of the small cases -- ragged tiles, prefixes that end inside a page, one tile on one pair,
# more tiles than pairs, the thresholded rescale path with unscaled q -- is compared with the oracle.
@pytest.mark.parametrize("pairs", [1, 3])
@pytest.mark.parametrize("q_scale", [0.1, 1.0])
def test_config0_on_pair_kernel(pairs, q_scale):
    run, _, _ = _full_compare(W.make_config(0, q_scale=q_scale), pairs=pairs)
    assert run.ctx.last_plan_info()["kernels"] == 2  # pair grid + decode grid, no combine at this size


@pytest.mark.parametrize("name,kw", [e for e in EDGE if e[1]["chunk_len"] > 0], ids=[e[0] for e in EDGE if e[1]["chunk_len"] > 0])
def test_edge_cases_on_pair_kernel(name, kw):
    inp = W.make_inputs(name, 100 + len(name), q_scale=0.5, extra_pages=3, **kw)
    _full_compare(inp, pairs=2)


def test_pair_kernel_rescale_path_and_long_tiles():
    """Scores with a steep positional trend force running-max updates page after page (the O-CTA's rescale path)."""
    inp = W.make_inputs("pair_rescale", 77, [300], 40, 1500, q_scale=2.0)
    _full_compare(inp, pairs=2)


def test_empty_step_is_noop_and_errors_are_host_side():
    import torch
    from paper_2607_02043_b200 import kairos as K
    inp = W.make_inputs("t", 1, [70], 8, 8)
    run = Hp.GpuRun(inp)
    e = torch.empty((0, 16, 576), dtype=torch.bfloat16, device="cuda")
    run.ctx.mixed_step(e, torch.empty((0, 1), dtype=torch.int32, device="cuda"), [], e,
                       torch.empty(0, dtype=torch.int32, device="cuda"), 0, 0)
    with pytest.raises(K.KairosError) as ei:   # ctx_len 0
        run.ctx.mixed_step(run.q_dec, run.dec_pt, [0], run.q_chunk, run.chunk_pt, inp.chunk_len, inp.prefix_len)
    assert ei.value.code == -1
    with pytest.raises(K.KairosError) as ei:   # ctx_len beyond its table
        run.ctx.mixed_step(run.q_dec, run.dec_pt, [64 * run.dec_pt.shape[1] + 1], run.q_chunk, run.chunk_pt,
                           inp.chunk_len, inp.prefix_len)
    assert ei.value.code == -1
    with pytest.raises(K.KairosError) as ei:   # chunk table too short
        run.ctx.mixed_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, inp.chunk_len, 64)
    assert ei.value.code == -1


# ------------------------------------------------------------------ invariants on the GPU
def test_page_permutation_and_stale_slots_bit_identical():
    """G13 / G7: the planner depends only on lengths, so permuting physical pages -- or poisoning every slot
    that is not visible with +-1e4 -- must leave the GPU output bit-identical."""
    inp = W.make_inputs("perm", 21, [64, 130, 700, 2500], 70, 90, q_scale=0.5, extra_pages=5)
    run = Hp.GpuRun(inp)
    run.append()
    a = run.step()
    rng = np.random.default_rng(5)
    pool_np = Hp.oracle_pool_after_append(inp)
    sig = rng.permutation(inp.num_pages)
    pool2 = np.empty_like(pool_np)
    pool2[sig] = pool_np
    used = np.zeros((inp.num_pages, 64), bool)
    for i, L in enumerate(inp.dec_ctx_lens):
        t = np.arange(L)
        used[sig[inp.dec_page_tables[i][t // 64]], t % 64] = True
    t = np.arange(inp.prefix_len + inp.chunk_len)
    used[sig[inp.chunk_page_table[t // 64]], t % 64] = True
    pool2[~used] = W.f32_to_bf16_bits(np.float32(1e4))
    inp2 = W.MixedStepInputs(**{**inp.__dict__, "pool": pool2,
                                "dec_page_tables": sig[inp.dec_page_tables].astype(np.int32),
                                "chunk_page_table": sig[inp.chunk_page_table].astype(np.int32), "chunk_len": inp.chunk_len})
    run2 = Hp.GpuRun(inp2)   # chunk already in pool2: no append
    b = run2.step()
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_decode_equals_last_prefill_row_and_chunk_invariance_gpu():
    """PAPER.md:66 / :23 on the GPU: a prompt run as successive (append, step) chunks matches the one-shot
    oracle prefill row for row, and a decode over the finished cache matches the last row (within tolerance)."""
    from oracle import oracle
    import torch
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(3)
    L = 400
    inp = W.make_inputs("sched", 31, [], L, 0, q_scale=0.5, extra_pages=2)
    pool_np = inp.pool.copy()
    oracle.append(pool_np, inp.chunk_latent, inp.chunk_k_rope, inp.chunk_page_table, 0)
    _, ref, _, _ = oracle.mixed_step(pool_np, np.zeros((0, 16, 576), np.uint16), np.zeros((0, 1), np.int32),
                                     np.zeros(0, np.int32), L, 0, inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
    run = Hp.GpuRun(inp)
    outs, pos = [], 0
    e = torch.empty((0, 16, 576), dtype=torch.bfloat16, device="cuda")
    ept = torch.empty((0, 1), dtype=torch.int32, device="cuda")
    for c in [128, 100, 1, 71, 100]:
        run.ctx.append_latent(run.latent[pos:pos + c], run.k_rope[pos:pos + c], run.chunk_pt, pos)
        _, oc, _, _ = run.ctx.mixed_step(e, ept, [], run.q_chunk[pos:pos + c].contiguous(), run.chunk_pt, c, pos)
        outs.append(W.bf16_bits_to_f32(K.bf16_bits(oc)))
        pos += c
    got = np.concatenate(outs)
    assert np.array_equal(run.pool_bits(), pool_np)
    Hp.assert_attention_close([got], [ref], "chunk schedule")
    od, _, _, _ = run.ctx.mixed_step(run.q_chunk[L - 1:L].contiguous(), run.chunk_pt[None, :].contiguous(), [L], e,
                                     run.chunk_pt, 0, 0)
    torch.cuda.synchronize()
    Hp.assert_attention_close([W.bf16_bits_to_f32(K.bf16_bits(od))[0]], [ref[L - 1]], "decode = last row")


# ------------------------------------------------------------------ BASELINE.json configs at full size, every row
def test_config1_steady_state_every_row():
    _full_compare(W.make_config(1))


def test_config1_unscaled_q_every_row():
    _full_compare(W.make_config(1, q_scale=1.0))


# The three orders in which the decode grid and the chunk clusters share the SMs, and the chunk as gen-1
# tiles of the decode queue, each on every row of configs[1]: pairs n > 0 = decode grid first (as 2-CTA clusters)
# beside n chunk clusters, -(n + 1) = n chunk clusters first with the full decode grid behind them, 0 = one queue.
@pytest.mark.parametrize("pairs", [0, 20, -17, 74])
def test_config1_every_row_in_every_launch_order(pairs):
    run, _, _ = _full_compare(W.make_config(1), pairs=pairs)
    info = run.ctx.last_plan_info()
    assert (info["chunk_pairs"] == 0) == (pairs == 0)


@pytest.mark.parametrize("name,kw", [e for e in EDGE if e[1]["chunk_len"] > 0 and len(e[1]["dec_ctx_lens"]) > 0],
                         ids=[e[0] for e in EDGE if e[1]["chunk_len"] > 0 and len(e[1]["dec_ctx_lens"]) > 0])
def test_edge_cases_clusters_first(name, kw):
    inp = W.make_inputs(name, 100 + len(name), q_scale=0.5, extra_pages=3, **kw)
    _full_compare(inp, pairs=-3)


def test_config2_heavy_tail_every_row():
    _full_compare(W.make_config(2))


@pytest.mark.parametrize("C", W.SWEEP_CHUNKS)
def test_config3_chunk_sweep_every_row(C):
    """All seven points of the latency-table sweep (BASELINE.json configs[3]), each in the launch order the planner picks."""
    _full_compare(W.make_config(3, chunk_len=C))


def test_config4_long_context_every_row():
    _full_compare(W.make_config(4))


# ------------------------------------------------------------------ plan cache, CUDA-graph replay, staging
def test_plan_cache_and_graph_replay_match_direct_launch():
    """The same step issued repeatedly with the same buffers: first planned and launched directly, then an exact cache
    hit, then replayed as a CUDA graph.  Every repetition is compared with the oracle on every row and must be
    bit-identical to the first; a context with the cache and graphs switched off gives the same bits."""
    from oracle import oracle
    for cfg, pairs in [(0, None), (1, None), (1, 0), (1, 20)]:
        inp = W.make_config(cfg)
        run = Hp.GpuRun(inp, pairs=pairs)
        run.append()
        pool_np = Hp.oracle_pool_after_append(inp)
        ref = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                                inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
        first, states = None, []
        for rep in range(5):
            got = run.step(reuse_outputs=True)
            info = run.ctx.last_plan_info()
            states.append((info["plan_cache"], info["graph"]))
            Hp.assert_attention_close(got[:2], ref[:2], f"configs[{cfg}] rep {rep}")
            if first is None:
                first = got
            for x, y in zip(first, got):
                assert np.array_equal(x, y), (cfg, pairs, rep)
        assert states[0] == (0, 0) and states[1][0] == 2 and states[-1] == (2, 1), states
        # the pre-marshalled form of the same calls (Kairos.bind_step) gives the same bits
        import torch
        od, oc, ld, lc = (torch.full_like(t, float("nan")) for t in run.out)
        bound = run.ctx.bind_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, inp.chunk_len, inp.prefix_len,
                                  od, oc, ld, lc, run.latent, run.k_rope)
        for _ in range(3):
            bound.run()
        torch.cuda.synchronize()
        f = lambda t: W.bf16_bits_to_f32(run.K.bf16_bits(t))
        for x, y in zip(first, (f(od), f(oc), ld.cpu().numpy(), lc.cpu().numpy())):
            assert np.array_equal(x, y)
        plain = Hp.GpuRun(inp, pairs=pairs, knobs=dict(graph=0, plan_cache=0, copy_stream=0))
        plain.append()
        got = plain.step()
        assert plain.ctx.last_plan_info()["plan_cache"] == 0
        for x, y in zip(first, got):
            assert np.array_equal(x, y)


def test_structural_plan_hit_lengths_move_inside_last_pages():
    """Decode lengths that grow without crossing a page boundary re-use the cached plan's structure (only n_keys is
    patched); each step is compared with the oracle on every row."""
    from oracle import oracle
    import torch
    lens0 = np.array([70, 135, 700, 2500, 68], np.int32)
    inp = W.make_inputs("structural", 41, lens0.tolist(), 24, 40, q_scale=0.5, extra_pages=2)
    run = Hp.GpuRun(inp)
    run.append()
    pool_np = Hp.oracle_pool_after_append(inp)
    seen = []
    for grow in [0, 1, 2, 3, 40]:
        lens = (lens0 - grow).astype(np.int32)  # the pool already holds every position < lens0
        od, oc, ld, lc = run.ctx.mixed_step(run.q_dec, run.dec_pt, lens, run.q_chunk, run.chunk_pt, inp.chunk_len,
                                            inp.prefix_len, out_dec=None if run.out is None else run.out[0],
                                            out_chunk=None if run.out is None else run.out[1])
        run.out = (od, oc, ld, lc)
        torch.cuda.synchronize()
        seen.append(run.ctx.last_plan_info()["plan_cache"])
        rd, rc, rld, rlc = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, lens, inp.chunk_len, inp.prefix_len,
                                             inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
        f = lambda t: W.bf16_bits_to_f32(run.K.bf16_bits(t))
        Hp.assert_attention_close([f(od), f(oc)], [rd, rc], f"structural grow={grow}")
        assert np.abs(ld.cpu().numpy() - rld).max() <= Hp.LSE_TOL
    assert seen == [0, 1, 1, 1, 0], seen  # -40 moves 68 -> 28 and 70 -> 30 (page counts change): planned again


@pytest.mark.parametrize("pairs", [None, 0, 3])
def test_soak_many_steps_rotating_pages(pairs):
    """60 back-to-back (append, step) pairs on ONE context, no host synchronisation in between, with the chunk's pages
    handed from step to step (each step overwrites pages the previous step was still reading: the programmatic-launch
    ordering and the plan buffers' re-use are what is under test).  Every step's outputs are kept on the device and each
    is compared with the oracle on every row afterwards."""
    import torch
    from oracle import oracle
    from paper_2607_02043_b200 import kairos as K
    rng = np.random.default_rng(17)
    lens = np.array([64, 200, 700, 1500], np.int32)
    inp = W.make_inputs("soak", 53, lens.tolist(), 48, 30, q_scale=0.5, extra_pages=4)
    run = Hp.GpuRun(inp, pairs=pairs)
    n_steps = 60
    lat = rng.integers(0, 2 ** 16, (n_steps, inp.chunk_len, 512), dtype=np.uint16) & np.uint16(0xBF7F)  # finite bf16, |x| < 2
    rope = rng.integers(0, 2 ** 16, (n_steps, inp.chunk_len, 64), dtype=np.uint16) & np.uint16(0xBF7F)
    lat_d, rope_d = K.bf16_tensor(lat), K.bf16_tensor(rope)
    shapes = [(24, 30), (48, 30), (48, 30), (7, 71)]  # (C, P) cycle: three plans alternate, one repeats back to back
    outs = []
    for s in range(n_steps):
        C, P = shapes[s % len(shapes)]
        run.ctx.append_latent(lat_d[s, :C], rope_d[s, :C], run.chunk_pt, P)
        outs.append(run.ctx.mixed_step(run.q_dec, run.dec_pt, lens, run.q_chunk[:C], run.chunk_pt, C, P))
    torch.cuda.synchronize()
    pool_np = inp.pool.copy()
    f = lambda t: W.bf16_bits_to_f32(K.bf16_bits(t))
    for s in range(n_steps):
        C, P = shapes[s % len(shapes)]
        oracle.append(pool_np, lat[s, :C], rope[s, :C], inp.chunk_page_table, P)
        rd, rc, rld, rlc = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, lens, C, P, inp.q_chunk[:C],
                                             inp.chunk_page_table, inp.softmax_scale)
        od, oc, ld, lc = outs[s]
        Hp.assert_attention_close([f(od), f(oc)], [rd, rc], f"soak step {s}")
        assert np.abs(lc.cpu().numpy() - rlc).max() <= Hp.LSE_TOL
    assert np.array_equal(run.pool_bits(), pool_np)


def test_nonfinite_stale_slots_do_not_reach_outputs():
    """include/kairos.h precondition: slots at positions >= the attended length may hold ANY bit pattern, NaN and Inf
    included (an allocator's leftovers).  Decode path, gen-1 chunk tiles and the cluster kernel, ragged last pages."""
    inp = W.make_inputs("poison", 61, [1, 63, 65, 130, 700], 37, 91, q_scale=0.5, extra_pages=3)
    pool_np = Hp.oracle_pool_after_append(inp)
    used = np.zeros((inp.num_pages, 64), bool)
    for i, L in enumerate(inp.dec_ctx_lens):
        t = np.arange(L)
        used[inp.dec_page_tables[i][t // 64], t % 64] = True
    t = np.arange(inp.prefix_len + inp.chunk_len)
    used[inp.chunk_page_table[t // 64], t % 64] = True
    poison = pool_np.copy()
    pat = np.array([0x7FC0, 0xFFC0, 0x7F80, 0xFF80], np.uint16)  # +-NaN, +-Inf
    poison[~used] = pat[np.arange(576) % 4]
    for pairs in [0, 2, -3]:
        clean = Hp.GpuRun(W.MixedStepInputs(**{**inp.__dict__, "pool": pool_np}), pairs=pairs).step()
        dirty = Hp.GpuRun(W.MixedStepInputs(**{**inp.__dict__, "pool": poison}), pairs=pairs).step()
        for x, y in zip(clean, dirty):
            assert np.all(np.isfinite(y))
            assert np.array_equal(x, y), pairs


def test_workspace_too_small_and_misaligned_pointers_are_host_side_errors():
    import torch
    from paper_2607_02043_b200 import kairos as K
    inp = W.make_inputs("ws", 3, [9000, 9000, 9000], 0, 0)
    run = Hp.GpuRun(inp, workspace_bytes=256 + 32896)  # counters + ONE partial slot: the long decodes need several
    with pytest.raises(K.KairosError) as ei:
        run.step()
    assert ei.value.code == -3
    ok = Hp.GpuRun(inp)
    qd = torch.empty(inp.q_dec.size + 8, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(K.KairosError) as ei:   # q_dec 4 bytes off a 16-byte boundary
        ok.ctx.mixed_step(qd[2:2 + inp.q_dec.size].view(3, 16, 576), ok.dec_pt, inp.dec_ctx_lens, ok.q_chunk, ok.chunk_pt, 0, 0)
    assert ei.value.code == -1
    with pytest.raises(K.KairosError) as ei:
        ok.ctx.debug_set("no_such_knob", 1)
    assert ei.value.code == -1


# ------------------------------------------------------------------ a11
def test_latency_table_shape_and_monotone():
    """a11: the table is produced, positive, and roughly monotone in C at the large end."""
    inp = W.make_inputs("lt", 7, [2048] * 64, 0, 0, extra_pages=140)
    run = Hp.GpuRun(inp)
    med, mn = run.ctx.step_latency_table([0, 64], [2048], [0, 256, 4096], warmup=2, reps=5)
    assert med.shape == (2, 1, 3) and med[0, 0, 0] == 0.0
    assert np.all(med.ravel()[1:] > 0) and np.all(mn <= med + 1e-9)
    assert med[1, 0, 2] > med[1, 0, 0] and med[0, 0, 2] > med[0, 0, 1]


def test_latency_table_matches_independently_timed_steps():
    """an entry of the table produced through kairos_step_latency_table must agree with the same point
    timed independently (CUDA events around back-to-back kairos_mixed_step calls on BASELINE.json configs[3] inputs), and
    the table must grow with C, with K and with B within noise."""
    import torch
    from paper_2607_02043_b200 import kairos as K
    from paper_2607_02043_b200 import latency_table as LT
    ctx = LT.make_context(LT.pages_needed([256], [2048], [2048]), 256, 2048)
    Cs = [0, 512, 2048]
    med, mn = ctx.step_latency_table([256], [2048], Cs, warmup=5, reps=20, flush_l2=False)
    for iC, C in enumerate(Cs):
        inp = W.make_config(3, chunk_len=C)
        run = Hp.GpuRun(inp)
        run.append()
        out = run.ctx.mixed_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, C, 0)
        bound = run.ctx.bind_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, C, 0, *out)
        for _ in range(5):
            bound.run()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(20):
            bound.run()
        e1.record()
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / 20
        assert abs(med[0, 0, iC] - us) <= 0.10 * us + 3.0, (C, med[0, 0, iC], us)
    assert med[0, 0, 0] < med[0, 0, 1] < med[0, 0, 2]
    grid, _ = ctx.step_latency_table([64, 256], [512, 2048], [0, 1024], warmup=3, reps=10, flush_l2=False)
    assert np.all(grid[1] > grid[0] * 0.98) and np.all(grid[:, 1] > grid[:, 0] * 0.98) and np.all(grid[:, :, 1] > grid[:, :, 0])


@pytest.mark.parametrize("cfg", [0, 1])
def test_host_buffer_step_matches_oracle_every_row(cfg):
    """kairos_mixed_step_host (the end-to-end leg bench.py times): HOST buffers in, HOST buffers out, the chunk appended by
    the call itself.  Every row against the oracle, the pool bit-exact, and the byte counts it reports."""
    from oracle import oracle
    inp = W.make_config(cfg)
    run = Hp.GpuRun(inp)
    od = np.zeros((inp.n_dec, 16, 512), np.uint16)
    oc = np.zeros((inp.chunk_len, 16, 512), np.uint16)
    for _ in range(2):  # the second call re-uses the context's device staging
        h2d, d2h = run.ctx.mixed_step_host(inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.q_chunk, inp.chunk_latent,
                                           inp.chunk_k_rope, inp.chunk_page_table, inp.chunk_len, inp.prefix_len, od, oc)
    pool_np = Hp.oracle_pool_after_append(inp)
    assert np.array_equal(run.pool_bits(), pool_np)
    rd, rc, _, _ = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                                     inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
    Hp.assert_attention_close([W.bf16_bits_to_f32(od), W.bf16_bits_to_f32(oc)], [rd, rc], f"configs[{cfg}] through host buffers")
    assert h2d == inp.q_dec.nbytes + inp.q_chunk.nbytes + inp.dec_page_tables.nbytes + inp.chunk_page_table.nbytes + inp.chunk_latent.nbytes + inp.chunk_k_rope.nbytes
    assert d2h == od.nbytes + oc.nbytes


@pytest.mark.parametrize("cfg,slice_tokens,pinned", [(1, 136, True), (1, 8, True), (1, 200, False), (2, 0, True)])
def test_host_buffer_step_in_slices_matches_oracle_every_row(cfg, slice_tokens, pinned):
    """kairos_mixed_step_host cuts a large chunk into slices that run as successive steps over a growing prefix while the
    copies of the neighbouring slices run beside them (three streams).  configs[1] with forced slices (ragged last slice;
    8-token slices = 64 steps, more than the plan cache holds; pageable host buffers) and configs[2] under the call's own
    rule (4 slices of whole rounds of the cluster grid): every row against the oracle, the pool bit-exact, the byte counts,
    twice in a row."""
    import torch
    from oracle import oracle
    inp = W.make_config(cfg)
    run = Hp.GpuRun(inp)
    if slice_tokens:
        run.ctx.debug_set("host_slice_tokens", slice_tokens)
    if pinned:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        od = torch.zeros((inp.n_dec, 16, 512), dtype=torch.int16).pin_memory().numpy().view(np.uint16)
        oc = torch.zeros((inp.chunk_len, 16, 512), dtype=torch.int16).pin_memory().numpy().view(np.uint16)
    else:  # pageable host memory: the copies lose their overlap, the results must not change
        pin = np.ascontiguousarray
        od = np.zeros((inp.n_dec, 16, 512), np.uint16)
        oc = np.zeros((inp.chunk_len, 16, 512), np.uint16)
    q_dec, q_chunk, lat, rope = pin(inp.q_dec), pin(inp.q_chunk), pin(inp.chunk_latent), pin(inp.chunk_k_rope)
    pool_np = Hp.oracle_pool_after_append(inp)
    rd, rc, rld, rlc = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                                         inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
    ld = np.zeros((inp.n_dec, 16), np.float32)
    lc = np.zeros((inp.chunk_len, 16), np.float32)
    for rep in range(2):
        od[:] = 0
        oc[:] = 0
        ld[:] = 0
        lc[:] = 0
        h2d, d2h = run.ctx.mixed_step_host(q_dec, inp.dec_page_tables, inp.dec_ctx_lens, q_chunk, lat, rope,
                                           inp.chunk_page_table, inp.chunk_len, inp.prefix_len, od, oc, lse_dec=ld, lse_chunk=lc)
        assert np.array_equal(run.pool_bits(), pool_np)
        Hp.assert_attention_close([W.bf16_bits_to_f32(od), W.bf16_bits_to_f32(oc)], [rd, rc],
                                  f"configs[{cfg}] through host buffers in slices of {slice_tokens or 'auto'} (call {rep})")
        assert np.abs(ld - rld).max() <= Hp.LSE_TOL and np.abs(lc - rlc).max() <= Hp.LSE_TOL  # every slice's lse lands at its own rows
        assert h2d == inp.q_dec.nbytes + inp.q_chunk.nbytes + inp.dec_page_tables.nbytes + inp.chunk_page_table.nbytes + inp.chunk_latent.nbytes + inp.chunk_k_rope.nbytes
        assert d2h == od.nbytes + oc.nbytes + ld.nbytes + lc.nbytes


def test_tuned_launch_order_keeps_parity_and_is_used():
    """kairos_tune_step pins a measured launch order for a shape; later steps of that shape use it (also through
    kairos_run_schedule / Kairos.bind_step) and still match the oracle on every row."""
    import torch
    from oracle import oracle
    inp = W.make_config(1)
    run = Hp.GpuRun(inp)
    run.append()
    od, oc, ld, lc = run.ctx.mixed_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, inp.chunk_len, inp.prefix_len)
    before = run.ctx.last_plan_info()
    mode, us, dus = run.ctx.tune_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, inp.chunk_len, inp.prefix_len, od, oc, reps=3)
    assert us > 0 and dus > 0 and us <= dus
    pool_np = Hp.oracle_pool_after_append(inp)
    rd, rc, rld, rlc = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                                         inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
    f = lambda t: W.bf16_bits_to_f32(run.K.bf16_bits(t))
    for _ in range(3):
        got = run.step(reuse_outputs=True)
        Hp.assert_attention_close(got[:2], [rd, rc], "after tuning")
    after = run.ctx.last_plan_info()
    if mode != -1:  # a different order was pinned: the plan reflects it
        assert (after["chunk_pairs"], after["dec_ctas_first"]) != (before["chunk_pairs"], before["dec_ctas_first"]) or mode == 0
    bound = run.ctx.bind_step(run.q_dec, run.dec_pt, inp.dec_ctx_lens, run.q_chunk, run.chunk_pt, inp.chunk_len, inp.prefix_len,
                              *run.out, run.latent, run.k_rope)
    for _ in range(3):
        bound.run()
    torch.cuda.synchronize()
    Hp.assert_attention_close([f(run.out[0]), f(run.out[1])], [rd, rc], "bound step after tuning")
    info = run.ctx.last_plan_info()
    assert (info["chunk_pairs"], info["dec_ctas_first"]) == (after["chunk_pairs"], after["dec_ctas_first"])
