"""-m gpu: seeded random step shapes through the C ABI against the CPU oracle, every row.

The BASELINE configs and the hand-picked edge cases fix the shapes the planner's rules were fitted on; these cases walk
off them: random decode batches (log-normal and uniform lengths, ragged last pages), random chunk and prefix lengths
(not multiples of the tile or the page), under the planner's own launch order and under a random forced order of the
two grids (kairos_debug_set("pairs", ...): every order must give the same rows).  Sizes are kept to what the oracle does
in about a second per case.
"""
import numpy as np
import pytest

from paper_2607_02043_b200 import workloads as W
from tests import helpers as Hp

pytestmark = pytest.mark.gpu


def _random_case(seed: int):
    rng = np.random.default_rng(1000 + seed)
    kind = seed % 4
    if kind == 0:      # many short decodes, a mid-size chunk over a short prefix
        n_dec, lens = int(rng.integers(20, 97)), None
        lognormal = dict(median=float(rng.integers(100, 700)), sigma=0.7, lo=1, hi=4096)
        C, P = int(rng.integers(1200, 2600)), int(rng.integers(0, 300))
    elif kind == 1:    # a few long decodes, a small chunk over a long prefix
        n_dec, lognormal = int(rng.integers(1, 9)), None
        lens = [int(x) for x in rng.integers(2000, 12000, n_dec)]
        C, P = int(rng.integers(1, 200)), int(rng.integers(1000, 5000))
    elif kind == 2:    # chunk only / decodes only, odd sizes
        if rng.integers(0, 2):
            n_dec, lens, lognormal = 0, [], None
            C, P = int(rng.integers(1, 1500)), int(rng.integers(0, 3000))
        else:
            n_dec, lognormal = int(rng.integers(1, 200)), None
            lens = [int(x) for x in rng.integers(1, 1500, n_dec)]
            C, P = 0, 0
    else:              # mid batch, chunk of more than 148 tiles over a mid prefix (the decode-first orders)
        n_dec, lens = int(rng.integers(32, 129)), None
        lognormal = dict(median=float(rng.integers(300, 1500)), sigma=0.5, lo=16, hi=6000)
        C, P = int(rng.integers(1190, 2200)), int(rng.integers(0, 2500))
    inp = W.make_inputs(f"fuzz{seed}", 5000 + seed, lens, C, P, lognormal=lognormal, n_dec=n_dec if lognormal else None,
                        q_scale=float(rng.choice([0.1, 0.3])), extra_pages=int(rng.integers(0, 40)))
    tiles = (C + 7) // 8
    forced = None
    if C > 0 and seed % 3 != 0:  # a random forced order: n clusters first (-(n + 1)), or the decode grid first beside n clusters
        n = int(rng.integers(1, max(2, min(tiles, 60))))
        forced = -(n + 1) if rng.integers(0, 2) else n
    return inp, forced


@pytest.mark.parametrize("seed", list(range(32)))
def test_random_shapes_every_row(seed):
    from oracle import oracle
    inp, forced = _random_case(seed)
    run = Hp.GpuRun(inp, pairs=forced)
    run.append()
    pool_np = Hp.oracle_pool_after_append(inp)
    assert np.array_equal(run.pool_bits(), pool_np), "append: pool bytes differ"
    od, oc, ld, lc = run.step()
    rd, rc, rld, rlc = oracle.mixed_step(pool_np, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                                         inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
    Hp.assert_attention_close([od, oc], [rd, rc], f"fuzz seed {seed}: B={inp.n_dec} C={inp.chunk_len} P={inp.prefix_len} pairs={forced}")
    if od.size:
        assert np.abs(ld - rld).max() <= Hp.LSE_TOL
    if oc.size:
        assert np.abs(lc - rlc).max() <= Hp.LSE_TOL
    od2, oc2, _, _ = run.step()  # the cached plan (and its graph): the same bits
    assert np.array_equal(od, od2) and np.array_equal(oc, oc2)


@pytest.mark.parametrize("seed", list(range(8)))
def test_random_decode_batches_over_the_fp8_cache(seed):
    """The fp8 latent cache (kairos_fp8_append / kairos_fp8_decode) on random decode batches: the quantising append bit for
    bit and every request's attention against oracle/fp8_oracle.py, twice (the second call replays the cached plan)."""
    from tests.test_gpu_fp8 import Fp8Run, _assert_close
    rng = np.random.default_rng(2000 + seed)
    n_dec = int(rng.integers(1, 40))
    if seed % 2:
        lens = [int(x) for x in rng.integers(1, 3000, n_dec)]
    else:
        lens = [int(x) for x in W.lognormal_contexts(rng, n_dec, median=float(rng.integers(64, 900)), sigma=0.9, lo=1, hi=5000)]
    inp = W.make_inputs(f"fp8_fuzz{seed}", 6000 + seed, lens, 0, 0, q_scale=float(rng.choice([0.1, 0.3])), extra_pages=int(rng.integers(0, 20)))
    r = Fp8Run(inp)
    r.check_pool()
    ref_out, ref_lse = r.reference()
    out, lse, _ = r.decode()
    _assert_close(out, lse, ref_out, ref_lse, f"fp8 fuzz seed {seed}: lens {lens}")
    out2, lse2, _ = r.decode()
    assert np.array_equal(out, out2) and np.array_equal(lse, lse2)


EXTREMES = [
    ("one_decode_262144_tokens", dict(lens=[262144], C=0, P=0)),                       # 4096 pages in one request: ~150 splits
    ("2000_tiny_decodes", dict(lens=[64 + (i * 37) % 70 for i in range(2000)], C=0, P=0)),
    ("chunk_12345_tokens_alone", dict(lens=[], C=12345, P=0)),                         # 1544 tiles, ragged last tile and page
    ("chunk_of_9_over_150000_prefix", dict(lens=[100], C=9, P=150000)),                # two tiles of 2344 pages each
    ("2000_decodes_beside_a_3000_token_chunk", dict(lens=[70 + (i * 13) % 500 for i in range(2000)], C=3000, P=777)),
]


@pytest.mark.parametrize("name,kw", EXTREMES, ids=[e[0] for e in EXTREMES])
def test_extreme_sizes(name, kw):
    """The sizes the API does not bound (any lengths the page tables cover): a very long request, thousands of requests, a
    chunk of a thousand tiles, a tiny chunk over a very long prefix.  Append bit-exact; every decode row and an evenly
    spaced sample of the chunk rows that always holds the first, the last and the rows either side of every 1000th (the
    oracle does a row at a time: rows are independent, so parity on them is exact); everything finite."""
    inp = W.make_inputs(name, 7000 + len(name), kw["lens"], kw["C"], kw["P"], q_scale=0.1)
    run = Hp.GpuRun(inp)
    run.append()
    pool_np = Hp.oracle_pool_after_append(inp)
    assert np.array_equal(run.pool_bits(), pool_np), "append: pool bytes differ"
    od, oc, ld, lc = run.step()
    assert np.isfinite(od).all() and np.isfinite(oc).all()
    C = inp.chunk_len
    dec_idx = np.arange(inp.n_dec, dtype=np.int32) if inp.n_dec <= 64 else np.arange(0, inp.n_dec, 31, dtype=np.int32)
    step = max(1, C // 160)
    chunk_idx = np.unique(np.concatenate([np.arange(0, C, step), np.array([0, C - 1] if C else [], dtype=np.int64),
                                          np.array([r + d for r in range(1000, C, 1000) for d in (-1, 0)], dtype=np.int64)])).astype(np.int32)
    rd, rld, rc, rlc = Hp.oracle_sampled(inp, pool_np, dec_idx, chunk_idx)
    parts_g, parts_r = [], []
    if len(dec_idx):
        parts_g.append(od[dec_idx]); parts_r.append(rd)
        assert np.abs(ld[dec_idx] - rld).max() <= Hp.LSE_TOL
    if len(chunk_idx):
        parts_g.append(oc[chunk_idx]); parts_r.append(rc)
        assert np.abs(lc[chunk_idx] - rlc).max() <= Hp.LSE_TOL
    Hp.assert_attention_close(parts_g, parts_r, name)
