"""SURVEY 8(f) NEXT-4 "fuse RoPE+append": tropical_kv_append_rope against oracle.kv_append_rope over the WHOLE pool.

V rows and every untouched slot: bit-identical.  K rows are a floating-point result (fp32 in the kernel, exact fp64 in the
oracle, both rounded to bf16): bit-identical except where the kernel's one extra fp32 rounding moves a value across a
bf16 rounding boundary -- at most 1 bf16 ulp apart, and fewer than 1 in 500 elements (the bars are written below).
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_16264_b200 as tb
import synth
from tests.gpu_harness import DeviceStep, bits, to_dev

pytestmark = pytest.mark.gpu


def _ulp_distance(a_bits, b_bits):
    """Distance in bf16 steps between two arrays of finite bf16 patterns (monotone integer mapping of the sign-magnitude
    encoding)."""
    def key(x):
        x = x.astype(np.int32)
        return np.where(x & 0x8000, -(x & 0x7FFF), x & 0x7FFF)
    return np.abs(key(a_bits) - key(b_bits))


def _run(s, cos, sin):
    kp, vp = s.copy_pools()
    oracle.kv_append_rope(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new, cos, sin)
    dev = DeviceStep(s)
    tb.kv_append_rope(dev.pool, dev.batch, dev.k_new, dev.v_new, to_dev(cos), to_dev(sin))
    torch.cuda.synchronize()
    return dev, kp, vp


@pytest.mark.parametrize("Hkv,d", [(2, 64), (8, 128), (5, 128)])
def test_rope_append_whole_pool(Hkv, d):
    q = [130, 1, 1, 17, 0, 1]
    c = [3, 250, 4097, 60, 9, 0]
    s = synth.make_step(np.random.default_rng(60 + Hkv), Hkv * 2, Hkv, d, 16, q, c, poison=True)
    cos, sin = synth.make_rope_tables(int(max(a + b for a, b in zip(q, c))), d)
    dev, kp, vp = _run(s, cos, sin)
    assert np.array_equal(bits(dev.v_pool), vp), "V pool differs"
    got = bits(dev.k_pool)
    appended = np.zeros(kp.shape[:1] + kp.shape[2:3], bool)          # [page, slot] written this step
    for i in range(s.num_reqs):
        for t in range(int(s.q_lens[i])):
            pos = int(s.ctx_lens[i]) + t
            appended[s.page_table[i, pos // 16], pos % 16] = True
    mask = np.broadcast_to(appended[:, None, :, None], kp.shape)
    assert np.array_equal(got[~mask], kp[~mask]), "a slot outside the appended rows changed"
    dist = _ulp_distance(got[mask], kp[mask])
    assert dist.max() <= 1, "a rotated K value is more than one bf16 step from the oracle's"
    assert (dist != 0).mean() <= 2e-3, (dist != 0).mean()


def test_rope_identity_and_quarter_turn_tables_are_bit_exact():
    """cos = 1, sin = 0: the plain append, bit for bit.  cos = 0, sin = 1: swap and negate, bit for bit (no rounding)."""
    s = synth.make_step(np.random.default_rng(61), 8, 4, 128, 16, [200, 1, 1], [56, 700, 15], poison=True)
    table_len = 701
    half = 64
    for cs, sn in ((1.0, 0.0), (0.0, 1.0)):
        cos = np.full((table_len, half), cs, np.float32)
        sin = np.full((table_len, half), sn, np.float32)
        dev, kp, vp = _run(s, cos, sin)
        assert np.array_equal(bits(dev.k_pool), kp) and np.array_equal(bits(dev.v_pool), vp)


def test_rope_append_then_attention_equals_the_oracle_on_rotated_keys():
    """The rotated pool feeds the attention like any other: append_rope + mixed_attention against the oracle's attention
    over ITS rotated pool (q is taken as given)."""
    s = synth.make_step(np.random.default_rng(62), 8, 2, 128, 16, [150, 1, 1], [40, 300, 1000], poison=True)
    cos, sin = synth.make_rope_tables(1001, 128)
    dev, kp, vp = _run(s, cos, sin)
    ref, _ = oracle.mixed_attention(kp, vp, s.q, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table)
    tb.mixed_attention(dev.pool, dev.batch, dev.q, out=dev.out, workspace=dev.workspace)
    torch.cuda.synchronize()
    err = np.abs(dev.out_f64() - ref)
    assert err.max() <= 2e-2 and err.mean() <= 2e-3


def test_rope_append_argument_validation():
    s = synth.make_step(np.random.default_rng(63), 4, 2, 64, 16, [5, 1], [0, 40])
    dev = DeviceStep(s)
    cos, sin = synth.make_rope_tables(30, 64)        # shorter than max_kv_len = 41
    with pytest.raises(tb.TropicalError):
        tb.kv_append_rope(dev.pool, dev.batch, dev.k_new, dev.v_new, to_dev(cos), to_dev(sin))
    with pytest.raises(ValueError):
        tb.kv_append_rope(dev.pool, dev.batch, dev.k_new, dev.v_new, to_dev(cos[:, :16].copy()), to_dev(sin[:, :16].copy()))
