"""Host planner through the C ABI, no GPU: kairos_plan_dump.

Properties that hold for every plan: each (decode request, logical page) is covered by exactly one decode split;
each chunk token belongs to exactly one query tile whose KV splits cover pages [0, ceil((P + last token + 1)/64))
exactly once; split items own distinct partial slots that stay inside the kairos_workspace_bytes bound; the plan
depends only on lengths (G13); chunk tiles see the causal key count P + q_index + 1 (G3)."""
import numpy as np
import pytest

from paper_2607_02043_b200 import kairos as K
from paper_2607_02043_b200 import workloads as W

PAGE = 64
SLOT_BYTES = 16 * 512 * 4 + 16 * 2 * 4
KIND, QI, PB, PE, NKEYS, NQ, SLOT, COST = range(8)


def _check_plan(lens, C, P, n_ctas=148, pair_mode=0):
    lens = np.asarray(lens, dtype=np.int32)
    items, n_slots, n_pairs = K.plan_dump(lens, C, P, n_ctas, pair_mode=pair_mode, with_pairs=True)
    dec = items[items[:, KIND] == 0]
    chk = items[items[:, KIND] >= 1]
    if n_pairs > 0:  # the chunk runs on the cluster kernel: whole 8-token tiles, no KV split, clusters fit beside the decode grid
        assert (chk[:, KIND] == 2).all() and (chk[:, SLOT] == -1).all() and (chk[:, PB] == 0).all()
        assert 1 <= n_pairs <= min(len(chk), n_ctas // 2) and 2 * n_pairs <= n_ctas
        assert (np.diff(chk[:, COST]) <= 0).all()
    else:
        assert (chk[:, KIND] == 1).all()
    # ---- decode coverage
    for i, L in enumerate(lens):
        pages = (int(L) + PAGE - 1) // PAGE
        cover = np.zeros(pages, dtype=np.int32)
        mine = dec[dec[:, QI] == i]
        assert len(mine) >= 1
        for it in mine:
            assert 0 <= it[PB] < it[PE] <= pages
            cover[it[PB]:it[PE]] += 1
            assert it[NKEYS] == L and it[NQ] == 1
        assert (cover == 1).all(), f"request {i}: pages not covered exactly once"
        if len(mine) == 1:
            assert mine[0][SLOT] == -1
        else:
            assert (mine[:, SLOT] >= 0).all()
    # ---- chunk coverage
    if C > 0:
        tiles = {}
        for it in chk:
            tiles.setdefault(int(it[QI]), []).append(it)
        tok_cover = np.zeros(C, dtype=np.int32)
        for q0, its in tiles.items():
            nq = int(its[0][NQ])
            assert 1 <= nq and q0 + nq <= C
            tok_cover[q0:q0 + nq] += 1
            pages = (P + q0 + nq + PAGE - 1) // PAGE
            cover = np.zeros(pages, dtype=np.int32)
            for it in its:
                assert it[NQ] == nq and it[NKEYS] == P + q0 + 1
                assert 0 <= it[PB] < it[PE] <= pages
                cover[it[PB]:it[PE]] += 1
            assert (cover == 1).all(), f"tile {q0}: pages not covered exactly once"
            if len(its) == 1:
                assert its[0][SLOT] == -1
        assert (tok_cover == 1).all()
    else:
        assert len(chk) == 0
    # ---- partial slots: distinct, inside the workspace bound
    used = []
    for it in items:
        if it[SLOT] >= 0:
            n = 1 if it[KIND] == 0 else int(it[NQ])  # chunk splits own one slot per query token of the tile
            used.extend(range(int(it[SLOT]), int(it[SLOT]) + n))
    assert len(used) == len(set(used)), "partial slots overlap"
    if used:
        assert max(used) < n_slots
    assert 256 + n_slots * SLOT_BYTES <= K.workspace_bytes(max(len(lens), 1), max(C, 1))
    return items


@pytest.mark.parametrize("index,chunk", [(0, None), (1, None), (2, None), (3, 0), (3, 512), (3, 8192), (4, None)])
def test_plan_covers_baseline_configs(index, chunk):
    rng = np.random.default_rng({0: 0, 1: 1, 2: 2, 3: 3, 4: 4}[index])
    spec = {0: ([64, 128, 200, 256], 64, 128),
            1: (W.lognormal_contexts(rng, 64, 1024, 0.8, 64, 8192), 512, 0),
            2: (W.lognormal_contexts(rng, 128, 2048, 1.0, 64, 16384), 2048, 6144),
            3: ([2048] * 256, 512 if chunk is None else chunk, 0),
            4: ([32768] * 32, 4096, 28672)}[index]
    _check_plan(*spec)


@pytest.mark.parametrize("lens,C,P", [([], 1, 0), ([1], 0, 0), ([63, 64, 65], 3, 61), ([100000], 0, 0),
                                      ([5] * 1000, 7, 1), ([], 8192, 0), ([4096] * 148, 0, 0), ([300] * 7, 129, 4000)])
def test_plan_edge_shapes(lens, C, P):
    _check_plan(lens, C, P)
    _check_plan(lens, C, P, n_ctas=1)
    _check_plan(lens, C, P, n_ctas=7)


@pytest.mark.parametrize("pair_mode", [-1, 1, 5, 74])
@pytest.mark.parametrize("lens,C,P", [([], 8, 0), ([100], 13, 61), ([2048] * 256, 2048, 0), ([2048] * 256, 8192, 0),
                                      ([32768] * 32, 4096, 28672), ([], 8192, 0), ([64] * 4, 64, 128), ([300] * 7, 129, 4000)])
def test_plan_with_pair_kernel(lens, C, P, pair_mode):
    _check_plan(lens, C, P, pair_mode=pair_mode)
    _check_plan(lens, C, P, n_ctas=7, pair_mode=pair_mode)


def test_planner_policy_for_the_pair_kernel():
    n = lambda lens, C, P: K.plan_dump(lens, C, P, 148, pair_mode=-1, with_pairs=True)[2]
    assert n([64, 128, 200, 256], 64, 128) == 0          # configs[0]
    assert 8 <= n([2048] * 256, 512, 0) <= 32            # small chunk beside many decodes: a few clusters first, decode grid behind
    assert n([3569] * 32, 96, 0) >= 8 and n([842] * 4, 124, 0) == 0   # gen-1 tiles only for a tiny chunk beside little decode work
    assert n([2048] * 256, 8192, 0) > 40                 # tensor-bound: most SM pairs go to the chunk
    assert n([32768] * 32, 4096, 28672) > 40             # configs[4]
    assert n([], 8192, 0) == 74


def test_plan_depends_only_on_lengths_and_is_deterministic():
    a, sa = K.plan_dump([500, 9000, 64], 300, 100)
    b, sb = K.plan_dump([500, 9000, 64], 300, 100)
    assert np.array_equal(a, b) and sa == sb


def test_plan_tail_is_fine_grained():
    """The dynamic queue ends with small items, so the finishing imbalance is a few pages."""
    items = _check_plan([2048] * 256, 0, 0)
    sizes = items[:, PE] - items[:, PB]
    assert (np.diff(items[:, COST]) <= 0).all(), "queue is not longest-first"
    assert sizes[-148:].max() <= 4
    assert sizes.sum() == 256 * 32
