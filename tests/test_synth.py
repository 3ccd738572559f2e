"""The seeded generator reproduces the length draws recorded in SURVEY.md 8(d) and a sane layout."""
import numpy as np

import synth


def test_length_draws_match_recorded_check_values():
    exp = {
        "C1": ([57, 1, 1, 1], [0, 17, 100, 255], 372, 29),
        "C2": (None, [1239, 1298, 1672, 1972, 565, 733], 80396, 5055),
        "C3": ([814, 461, 503, 99], [0, 0, 0, 0], 0, 119),
        "C4": (None, [0, 4096, 100, 1457, 600, 665, 824], 174370, 11101),
        "C5": (None, [0, 0, 782, 1260, 7918, 2900, 291, 1492], 612310, 38731),
    }
    for name, (q, c_head, csum, pages) in exp.items():
        _, Hq, Hkv, d, P, ql, cl, _ = synth.config_lengths(name)
        if q is not None:
            assert ql.tolist() == q
        assert cl[: len(c_head)].tolist() == c_head
        assert int(cl.sum()) == csum
        assert synth.needed_pages(ql, cl, P) == pages
    assert synth.config_lengths("C4")[5].tolist() == [2048] + [1] * 128
    assert synth.config_lengths("C5")[5].tolist() == [4096, 1024] + [1] * 256


def test_C1_layout_and_poison():
    s = synth.make_config("C1")
    assert s.num_pages == 64 and s.page_table[0, :4].tolist() == [16, 36, 27, 8]
    used = s.page_table[s.page_table >= 0]
    assert len(used) == 29 and len(set(used.tolist())) == 29
    # prior context installed, everything else poisoned
    n_valid_rows = int((s.k_pool != synth.POISON_BF16).any(axis=-1).sum())
    assert n_valid_rows == int(s.ctx_lens.sum()) * s.num_kv_heads
    assert s.q.shape == (60, 4, 64) and s.k_new.shape == (60, 4, 64)
    assert s.q_offsets.tolist() == [0, 57, 58, 59, 60]


def test_bf16_round_trip_and_rne():
    x = np.array([1.0, 1.00390625, 1.01171875, -2.5, 0.0], np.float32)  # 1+2^-8 ties to even (1.0); 1+3*2^-8 -> 1+2^-6
    b = synth.f32_to_bf16_bits(x)
    assert synth.bf16_bits_to_f32(b).tolist() == [1.0, 1.0, 1.015625, -2.5, 0.0]


def test_tiled_values_are_deterministic():
    a = synth.make_step(np.random.default_rng(5), 2, 2, 64, 16, [3, 1], [40, 100], values="tiled")
    b = synth.make_step(np.random.default_rng(5), 2, 2, 64, 16, [3, 1], [40, 100], values="tiled")
    assert np.array_equal(a.k_pool, b.k_pool) and np.array_equal(a.q, b.q)
