"""Host-side checks of the seeded generators against the figures SURVEY.md 8(d) / BASELINE.md print."""
import numpy as np

from paper_2607_02043_b200 import workloads as W


def test_bf16_rne_round_trip_and_ties():
    x = np.array([1.0, 1.00390625, 1.01171875, -2.5, 0.1, 3.3895314e38], np.float32)
    b = W.f32_to_bf16_bits(x)
    back = W.bf16_bits_to_f32(b)
    assert back[0] == 1.0 and back[3] == -2.5
    assert back[1] == 1.0            # 1 + 2^-8 is a tie -> even mantissa (1.0)
    assert back[2] == 1.015625       # 1 + 3*2^-8 is a tie -> even mantissa (1 + 2^-6)
    assert abs(back[4] - 0.1) < 0.1 * 2 ** -8
    assert np.array_equal(W.f32_to_bf16_bits(back), b)


def test_config_figures_match_baseline_md():
    c1 = W.make_config(1)
    L = c1.dec_ctx_lens
    assert (int(L.sum()), int(L.min()), int(L.max())) == (77755, 117, 5573)
    assert c1.chunk_len == 512 and c1.prefix_len == 0
    assert round(c1.algorithmic_bytes() / 1e6, 2) == 110.22
    assert round(c1.algorithmic_flops() / 1e9, 2) == 7.28
    c0 = W.make_config(0)
    assert round(c0.algorithmic_bytes() / 1e6, 2) == 3.34 and round(c0.algorithmic_flops() / 1e9, 2) == 0.38


def test_page_tables_are_disjoint_permutation_slices():
    inp = W.make_inputs("t", 5, [64, 65, 1, 300], 100, 30, extra_pages=4)
    owned = []
    for i, Lc in enumerate(inp.dec_ctx_lens):
        owned += list(inp.dec_page_tables[i][: (Lc + 63) // 64])
    owned += list(inp.chunk_page_table)
    assert len(owned) == len(set(owned)) == 1 + 2 + 1 + 5 + 3
    assert max(owned) < inp.num_pages == 12 + 4
    assert inp.pool.shape == (16, 64, 576) and inp.pool.dtype == np.uint16
