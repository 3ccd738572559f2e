"""Pins for the CPU oracle (oracle/tropical_oracle.c) -- none of them re-types its formula.

O1 brute-force dense attention (numpy, separate code path)          SURVEY 8(c) pin O1
O2 softmax weights sum to one                                        pin O2
O3 page-size invariance (bit-identical)                               pin O3
O4 page-permutation invariance (bit-identical)                        pin O4
O5 torch.nn.functional.scaled_dot_product_attention in fp64            pin O5
O6 closed forms                                                       pin O6
O7 chunk / decode / GQA consistency                                   pin O7
O8 needle: the softmax selects exactly one key                        pin O8
+  append vs python loops, gather vs fancy indexing, whole-pool stray-write check.
+  kv_migrate (NEXT-3): destination gathers equal source gathers, changed-row count, identity, attention invariance.
"""
import math

import numpy as np
import pytest
import torch
from hypothesis import given, settings, strategies as st

import oracle
import synth
from synth import f32_to_bf16_bits
from tests.dense_ref import (append_python_loops, bf16_to_f64, dense_attention_bruteforce,
                             gather_dense, pack_pool)


def _small_step(seed, Hq, Hkv, d, q_lens, ctx_lens, P=16, **kw):
    rng = np.random.default_rng(seed)
    return synth.make_step(rng, Hq, Hkv, d, P, q_lens, ctx_lens, **kw)


def _bruteforce_step(s, kp, vp, sm_scale=0.0):
    out = np.zeros((s.total_q, s.num_q_heads, s.head_dim))
    lse = np.zeros((s.total_q, s.num_q_heads))
    for i in range(s.num_reqs):
        ql, c = int(s.q_lens[i]), int(s.ctx_lens[i])
        if ql == 0:
            continue
        kd = gather_dense(kp, s.page_table[i], c + ql)
        vd = gather_dense(vp, s.page_table[i], c + ql)
        o, l, _ = dense_attention_bruteforce(s.q[s.q_offsets[i]:s.q_offsets[i + 1]], kd, vd, c, sm_scale)
        out[s.q_offsets[i]:s.q_offsets[i + 1]] = o
        lse[s.q_offsets[i]:s.q_offsets[i + 1]] = l
    return out, lse


# ------------------------------------------------------------------ append / gather (bit-exact)
def test_append_matches_python_loops_and_touches_nothing_else():
    s = _small_step(11, 4, 2, 64, [5, 1, 0, 33, 1], [0, 31, 7, 16, 15])
    kp, vp = s.copy_pools()
    oracle.kv_append(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    kp2, vp2 = s.copy_pools()
    append_python_loops(kp2, vp2, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    assert np.array_equal(kp, kp2) and np.array_equal(vp, vp2)
    # number of changed rows == T * Hkv exactly (poison made every target distinguishable)
    changed = (kp != s.k_pool).any(axis=-1).sum()
    assert changed == s.total_q * s.num_kv_heads
    # K and V were not swapped: V pool holds v_new rows
    i, t = 3, 32
    pos = int(s.ctx_lens[i]) + t
    assert np.array_equal(vp[s.page_table[i, pos // 16], :, pos % 16, :], s.v_new[s.q_offsets[i] + t])
    assert np.array_equal(kp[s.page_table[i, pos // 16], :, pos % 16, :], s.k_new[s.q_offsets[i] + t])


def test_gather_matches_fancy_indexing():
    s = _small_step(12, 2, 2, 64, [9, 1], [40, 77])
    kp, vp = s.copy_pools()
    oracle.kv_append(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    for i in range(2):
        n = int(s.ctx_lens[i] + s.q_lens[i])
        kd, vd = oracle.kv_gather(kp, vp, s.page_table, i, n)
        assert np.array_equal(kd, gather_dense(kp, s.page_table[i], n))
        assert np.array_equal(vd, gather_dense(vp, s.page_table[i], n))
        # the tail of the gathered K is exactly this step's new rows
        assert np.array_equal(kd[int(s.ctx_lens[i]):], s.k_new[s.q_offsets[i]:s.q_offsets[i + 1]])


# ------------------------------------------------------------------ KV migration (NEXT-3; PAPER.md:155 Path 1, :58)
def _migration_case(seed, Hkv, d, kv_lens, P=16):
    """A source step whose pools already hold kv_lens[m] tokens per request (contexts only), a poisoned destination
    pool of a different size and a fresh random destination page table."""
    rng = np.random.default_rng(seed)
    s = synth.make_step(rng, Hkv, Hkv, d, P, [0] * len(kv_lens), kv_lens)
    dst_pt, n_dst = synth.make_migration_target(rng, kv_lens, P)
    kd = np.full((n_dst, Hkv, P, d), synth.POISON_BF16, np.uint16)
    return s, dst_pt, kd, kd.copy()


def test_migrate_gather_of_destination_equals_gather_of_source():
    kv_lens = [1, 15, 16, 17, 100, 0, 255]
    s, dst_pt, kd, vd = _migration_case(21, 3, 64, kv_lens)
    k_src, v_src = s.copy_pools()
    oracle.kv_migrate(s.k_pool, s.v_pool, kd, vd, kv_lens, s.page_table, dst_pt)
    assert np.array_equal(s.k_pool, k_src) and np.array_equal(s.v_pool, v_src)      # the source is read-only
    for m, n in enumerate(kv_lens):                                                  # numpy fancy indexing, not the oracle's gather
        assert np.array_equal(gather_dense(kd, dst_pt[m], n), gather_dense(s.k_pool, s.page_table[m], n))
        assert np.array_equal(gather_dense(vd, dst_pt[m], n), gather_dense(s.v_pool, s.page_table[m], n))
    # exactly sum(kv_lens) * Hkv destination rows changed (every other slot still holds the poison pattern): token-granular,
    # nothing past a request's last token, no stray page
    assert ((kd != synth.POISON_BF16).any(axis=-1)).sum() == sum(kv_lens) * 3
    assert ((vd != synth.POISON_BF16).any(axis=-1)).sum() == sum(kv_lens) * 3
    # K went to K and V to V (the generator draws them differently)
    assert not np.array_equal(gather_dense(kd, dst_pt[4], 100), gather_dense(s.v_pool, s.page_table[4], 100))


def test_migrate_is_the_identity_when_both_tables_name_the_same_pages():
    kv_lens = [40, 7]
    s, _, _, _ = _migration_case(22, 2, 64, kv_lens)
    kd, vd = np.full_like(s.k_pool, synth.POISON_BF16), np.full_like(s.v_pool, synth.POISON_BF16)
    oracle.kv_migrate(s.k_pool, s.v_pool, kd, vd, kv_lens, s.page_table, s.page_table)
    # the installed context rows are the only non-poison rows of the source as well
    assert np.array_equal(kd, s.k_pool) and np.array_equal(vd, s.v_pool)


def test_attention_is_unchanged_by_a_migration():
    """Decoding on the destination worker sees the same cache: fp64 outputs bit-identical (same j order)."""
    rng = np.random.default_rng(23)
    s = synth.make_step(rng, 4, 2, 64, 16, [1, 1, 1], [33, 16, 250])
    kp, vp = s.copy_pools()
    oracle.kv_append(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    L = (s.q_lens + s.ctx_lens).tolist()
    dst_pt, n_dst = synth.make_migration_target(rng, L, 16)
    kd = np.full((n_dst, 2, 16, 64), synth.POISON_BF16, np.uint16)
    vd = kd.copy()
    oracle.kv_migrate(kp, vp, kd, vd, L, s.page_table, dst_pt)
    a, la = oracle.mixed_attention(kp, vp, s.q, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table)
    b, lb = oracle.mixed_attention(kd, vd, s.q, s.q_lens, s.ctx_lens, s.q_offsets, dst_pt)
    assert np.array_equal(a, b) and np.array_equal(la, lb)


# ------------------------------------------------------------------ O1 / O2
@pytest.mark.parametrize("Hq,Hkv,d", [(4, 4, 64), (8, 2, 128), (6, 1, 32)])
def test_O1_bruteforce_and_O2_rowsum(Hq, Hkv, d):
    s = _small_step(21, Hq, Hkv, d, [57, 1, 1, 1, 20, 0], [0, 17, 100, 255, 45, 9])
    out, lse, kp, vp = oracle.step(s)
    ref, ref_lse = _bruteforce_step(s, kp, vp)
    assert np.abs(out - ref).max() <= 1e-12
    assert np.abs(lse - ref_lse).max() <= 1e-12
    _, _, wsum = oracle.mixed_attention(kp, vp, s.q, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table,
                                        want_wsum=True)
    assert np.abs(wsum - 1.0).max() <= 1e-12
    assert np.isfinite(out).all()  # poison slots never leak


def test_O1_custom_scale():
    s = _small_step(22, 2, 2, 64, [7, 1], [3, 30])
    out, lse, kp, vp = oracle.step(s, sm_scale=0.37)
    ref, ref_lse = _bruteforce_step(s, kp, vp, 0.37)
    assert np.abs(out - ref).max() <= 1e-12 and np.abs(lse - ref_lse).max() <= 1e-12
    out_default, _, _, _ = oracle.step(s)
    assert np.abs(out - out_default).max() > 1e-3  # the scale is actually used


def test_C1_config_bruteforce():
    s = synth.make_config("C1")
    out, lse, kp, vp = oracle.step(s)
    ref, _ = _bruteforce_step(s, kp, vp)
    assert out.shape == (60, 4, 64) and np.abs(out - ref).max() <= 1e-12


# ------------------------------------------------------------------ O3 / O4 paging invariance
def _dense_requests(rng, lens, Hkv, d):
    return [f32_to_bf16_bits(rng.standard_normal((L, Hkv, d), dtype=np.float32)) for L in lens]


def _attend_dense(kds, vds, q_bits, q_lens, ctx_lens, P, rng, shuffle=True):
    kp, pt = pack_pool(kds, P, rng, shuffle=shuffle)
    vp = np.full_like(kp, synth.POISON_BF16)  # V placed under the same page table as K
    for i, x in enumerate(vds):
        for j in range(x.shape[0]):
            vp[pt[i, j // P], :, j % P, :] = x[j]
    q_offsets = np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32)
    return oracle.mixed_attention(kp, vp, q_bits, q_lens, ctx_lens, q_offsets, pt)


def test_O3_page_size_invariance_bit_identical():
    rng = np.random.default_rng(31)
    q_lens, ctx_lens = [19, 1, 1], [37, 64, 5]
    lens = [q + c for q, c in zip(q_lens, ctx_lens)]
    kds, vds = _dense_requests(rng, lens, 2, 64), _dense_requests(rng, lens, 2, 64)
    q_bits = f32_to_bf16_bits(rng.standard_normal((sum(q_lens), 4, 64), dtype=np.float32))
    base = None
    for P in (1, 2, 8, 16, 32, 64):
        out, lse = _attend_dense(kds, vds, q_bits, q_lens, ctx_lens, P, np.random.default_rng(P))
        if base is None:
            base = (out, lse)
        assert np.array_equal(out, base[0]) and np.array_equal(lse, base[1]), f"P={P}"


def test_O4_page_permutation_invariance_bit_identical():
    rng = np.random.default_rng(32)
    q_lens, ctx_lens = [40, 1], [50, 129]
    lens = [q + c for q, c in zip(q_lens, ctx_lens)]
    kds, vds = _dense_requests(rng, lens, 1, 64), _dense_requests(rng, lens, 1, 64)
    q_bits = f32_to_bf16_bits(rng.standard_normal((sum(q_lens), 2, 64), dtype=np.float32))
    a = _attend_dense(kds, vds, q_bits, q_lens, ctx_lens, 16, np.random.default_rng(1), shuffle=False)
    b = _attend_dense(kds, vds, q_bits, q_lens, ctx_lens, 16, np.random.default_rng(2), shuffle=True)
    c = _attend_dense(kds, vds, q_bits, q_lens, ctx_lens, 16, np.random.default_rng(3), shuffle=True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[0], c[0])


@settings(max_examples=15, deadline=None)
@given(st.integers(0, 2 ** 31 - 1), st.lists(st.tuples(st.integers(0, 40), st.integers(0, 70)), min_size=1, max_size=4),
       st.sampled_from([1, 3, 16]))
def test_hypothesis_random_batches_match_bruteforce(seed, reqs, P):
    q_lens = [q for q, _ in reqs]
    ctx_lens = [c for _, c in reqs]
    s = _small_step(seed, 4, 2, 32, q_lens, ctx_lens, P=P)
    out, lse, kp, vp = oracle.step(s)
    ref, ref_lse = _bruteforce_step(s, kp, vp)
    if s.total_q:
        assert np.abs(out - ref).max() <= 1e-12 and np.abs(lse - ref_lse).max() <= 1e-12


# ------------------------------------------------------------------ O5 library routine
def _sdpa(q_bits, kd, vd, c, causal_flag):
    q = torch.from_numpy(bf16_to_f64(q_bits)).permute(1, 0, 2)  # [Hq, q_len, d]
    k = torch.from_numpy(bf16_to_f64(kd)).permute(1, 0, 2)
    v = torch.from_numpy(bf16_to_f64(vd)).permute(1, 0, 2)
    g = q.shape[0] // k.shape[0]
    k, v = k.repeat_interleave(g, 0), v.repeat_interleave(g, 0)
    if causal_flag:
        o = torch.nn.functional.scaled_dot_product_attention(q[None], k[None], v[None], is_causal=True)
    else:
        ql, L = q.shape[1], k.shape[1]
        mask = torch.arange(L)[None, :] <= (c + torch.arange(ql))[:, None]
        o = torch.nn.functional.scaled_dot_product_attention(q[None], k[None], v[None], attn_mask=mask)
    return o[0].permute(1, 0, 2).numpy()


@pytest.mark.parametrize("Hq,Hkv", [(4, 4), (8, 2)])
def test_O5_torch_sdpa_fp64(Hq, Hkv):
    s = _small_step(41, Hq, Hkv, 64, [48, 23, 1], [0, 35, 90])
    out, _, kp, vp = oracle.step(s)
    for i in range(s.num_reqs):
        ql, c = int(s.q_lens[i]), int(s.ctx_lens[i])
        kd, vd = gather_dense(kp, s.page_table[i], c + ql), gather_dense(vp, s.page_table[i], c + ql)
        ref = _sdpa(s.q[s.q_offsets[i]:s.q_offsets[i + 1]], kd, vd, c, causal_flag=(c == 0))
        assert np.abs(out[s.q_offsets[i]:s.q_offsets[i + 1]] - ref).max() <= 1e-10


# ------------------------------------------------------------------ O6 closed forms
def test_O6_sigmoid_of_one_hand_example():
    """q=[1,0], keys k0=[0,0], k1=[1,0], scale=1: scores (0,1) -> weights (1, e)/(1+e).
    v0=[1,0], v1=[0,1] -> out = [1/(1+e), e/(1+e)] = [1-sigmoid(1), sigmoid(1)];  lse = log(1+e)."""
    d = 32
    z = np.zeros((2, 1, d), np.float32)
    k = z.copy(); k[1, 0, 0] = 1.0
    v = z.copy(); v[0, 0, 0] = 1.0; v[1, 0, 1] = 1.0
    qv = np.zeros((1, 1, d), np.float32); qv[0, 0, 0] = 1.0
    kp, pt = pack_pool([f32_to_bf16_bits(k)], 16, np.random.default_rng(0))
    vp = np.full_like(kp, synth.POISON_BF16)
    vp[pt[0, 0], :, :2, :] = f32_to_bf16_bits(v).transpose(1, 0, 2)
    out, lse = oracle.mixed_attention(kp, vp, f32_to_bf16_bits(qv), [1], [1], [0, 1], pt, sm_scale=1.0)
    assert abs(out[0, 0, 0] - 0.2689414213699951) < 1e-15
    assert abs(out[0, 0, 1] - 0.7310585786300049) < 1e-15
    assert abs(lse[0, 0] - math.log1p(math.e)) < 1e-15
    assert np.abs(out[0, 0, 2:]).max() == 0.0


def test_O6_first_row_is_v0_and_decode_on_empty_cache():
    s = _small_step(51, 4, 2, 64, [30, 1], [0, 0])
    out, lse, kp, vp = oracle.step(s)
    g = 2
    for h in range(4):
        assert np.array_equal(out[0, h], bf16_to_f64(s.v_new[0, h // g]))
        assert np.array_equal(out[30, h], bf16_to_f64(s.v_new[30, h // g]))  # q=1,c=0 (S5)


def test_O6_constant_V_and_zero_q_running_mean():
    rng = np.random.default_rng(52)
    s = synth.make_step(rng, 2, 2, 64, 16, [25, 1], [10, 40])
    s.v_new[:] = f32_to_bf16_bits(np.full(s.v_new.shape, 1.5, np.float32))
    vp_const = np.where(s.v_pool == synth.POISON_BF16, s.v_pool, f32_to_bf16_bits(np.float32(1.5).reshape(1))[0])
    s.v_pool = vp_const.astype(np.uint16)
    out, _, _, _ = oracle.step(s)
    assert np.abs(out - 1.5).max() <= 1e-14
    # q == 0 -> uniform weights -> running mean of V over j <= c + t
    s2 = synth.make_step(np.random.default_rng(53), 2, 1, 64, 16, [12], [9])
    s2.q[:] = 0
    out2, lse2, kp, vp = oracle.step(s2)
    vd = bf16_to_f64(gather_dense(vp, s2.page_table[0], 21))
    for t in range(12):
        assert np.abs(out2[t, 0] - vd[: 9 + t + 1, 0].mean(axis=0)).max() <= 1e-13
        assert abs(lse2[t, 1] - math.log(9 + t + 1)) <= 1e-13


def test_O6_key_shift_invariance():
    """Adding a fixed vector u to every key shifts each row's scores by the constant q_t.u."""
    rng = np.random.default_rng(54)
    L, ql, c, d = 37, 17, 20, 64
    grid = lambda shape: (rng.integers(-32, 33, shape) / 8.0).astype(np.float32)  # multiples of 1/8, bf16-exact
    k, u = grid((L, 1, d)), grid((1, 1, d))
    v = rng.standard_normal((L, 1, d)).astype(np.float32)
    qv = grid((ql, 2, d))
    res = []
    for kk in (k, k + u):
        assert np.array_equal(bf16_to_f64(f32_to_bf16_bits(kk)), kk.astype(np.float64))
        kp, pt = pack_pool([f32_to_bf16_bits(kk)], 16, np.random.default_rng(5))
        vp, _ = pack_pool([f32_to_bf16_bits(v)], 16, np.random.default_rng(5))
        res.append(oracle.mixed_attention(kp, vp, f32_to_bf16_bits(qv), [ql], [c], [0, ql], pt)[0])
    assert np.abs(res[0] - res[1]).max() <= 1e-11


# ------------------------------------------------------------------ O7 consistency
def test_O7_chunking_decode_and_gqa_consistency():
    rng = np.random.default_rng(61)
    L, Hq, Hkv, d = 45, 4, 2, 64
    kd = f32_to_bf16_bits(rng.standard_normal((L, Hkv, d), dtype=np.float32))
    vd = f32_to_bf16_bits(rng.standard_normal((L, Hkv, d), dtype=np.float32))
    qb = f32_to_bf16_bits(rng.standard_normal((L, Hq, d), dtype=np.float32))
    kp, pt = pack_pool([kd], 16, np.random.default_rng(7))
    vp, _ = pack_pool([vd], 16, np.random.default_rng(7))
    one, lse_one = oracle.mixed_attention(kp, vp, qb, [L], [0], [0, L], pt)
    # two chunks: rows [0,L1) with c=0 and rows [L1,L) with c=L1
    L1 = 18
    a, _ = oracle.mixed_attention(kp, vp, qb[:L1], [L1], [0], [0, L1], pt)
    b, _ = oracle.mixed_attention(kp, vp, qb[L1:], [L - L1], [L1], [0, L - L1], pt)
    assert np.array_equal(np.concatenate([a, b]), one)
    # last row == decode with c = L-1
    dec, lse_dec = oracle.mixed_attention(kp, vp, qb[L - 1:], [1], [L - 1], [0, 1], pt)
    assert np.array_equal(dec[0], one[L - 1]) and np.array_equal(lse_dec[0], lse_one[L - 1])
    # GQA == MHA with repeated kv heads
    kp_r, vp_r = np.repeat(kp, 2, axis=1), np.repeat(vp, 2, axis=1)
    mha, _ = oracle.mixed_attention(kp_r, vp_r, qb, [L], [0], [0, L], pt)
    assert np.array_equal(mha, one)
    # attention_rows subset == full
    sub, _ = oracle.attention_rows(kp, vp, qb, [L], [0], [0, L], pt, [(0, 3), (0, 44), (0, 16)])
    assert np.array_equal(sub, one[[3, 44, 16]])


# ------------------------------------------------------------------ O8 needle
def test_O8_needle_selects_exactly_one_key():
    """K rows = +-32 binary code of the logical position; q row t = code of target j*(t).
    Score gap >= 2*32*32/sqrt(d) = 256 (d=64) -> every other weight underflows to 0 in fp64 too."""
    d, c, ql = 64, 21, 30
    L = c + ql

    def code(j):
        vec = np.full(d, 32.0, np.float32)
        vec[:14] = np.where((j >> np.arange(14)) & 1, 32.0, -32.0)
        return vec

    k = np.stack([code(j) for j in range(L)])[:, None, :]
    v = np.random.default_rng(71).standard_normal((L, 1, d)).astype(np.float32)
    targets = [c + t if t % 3 == 0 else (c + t - 1 if t % 3 == 1 else (t * 7) % (c + t + 1)) for t in range(ql)]
    qv = np.stack([code(j) for j in targets])[:, None, :]
    kp, pt = pack_pool([f32_to_bf16_bits(k)], 16, np.random.default_rng(9))
    vp, _ = pack_pool([f32_to_bf16_bits(v)], 16, np.random.default_rng(9))
    out, _ = oracle.mixed_attention(kp, vp, f32_to_bf16_bits(qv), [ql], [c], [0, ql], pt)
    vb = bf16_to_f64(f32_to_bf16_bits(v))
    for t, j in enumerate(targets):
        assert np.array_equal(out[t, 0], vb[j, 0]), (t, j)
    # negative needle: aiming at the future key c+t+1 must NOT return it
    t = 4
    qf = code(c + t + 1)[None, None, :]
    o, _ = oracle.attention_rows(kp, vp, f32_to_bf16_bits(np.concatenate([qv[:t], qf, qv[t + 1:]])), [ql], [c], [0, ql], pt, [(0, t)])
    assert not np.array_equal(o[0, 0], vb[c + t + 1, 0])


# ------------------------------------------------------------------ NEXT-4: RoPE fused into the append (oracle pins)
def _rope_case(seed=50, Hq=4, Hkv=2, d=64, q_lens=(37, 1, 1), ctx_lens=(5, 100, 31)):
    s = _small_step(seed, Hq, Hkv, d, list(q_lens), list(ctx_lens))
    cos, sin = synth.make_rope_tables(int((np.asarray(q_lens) + np.asarray(ctx_lens)).max()), d)
    return s, cos, sin


def test_rope_rounding_helper_by_hand_and_against_the_fp32_route():
    """oracle_double_to_bf16: ties to even and the cases where rounding through fp32 first would go wrong.
    1 + 2^-8 is a tie -> even (1.0 = 0x3F80); 1 + 2^-8 + 2^-40 is above the tie -> 0x3F81 (fp32 would have dropped the
    2^-40 and tied down); 1 + 3 * 2^-8 is a tie between odd and even -> even 0x3F82; -2.5 = 0xC020."""
    got = oracle.double_to_bf16([1.0, 1 + 2.0 ** -8, 1 + 2.0 ** -8 + 2.0 ** -40, 1 + 3 * 2.0 ** -8, -2.5, 0.0])
    assert got.tolist() == [0x3F80, 0x3F80, 0x3F81, 0x3F82, 0xC020, 0x0000]
    # values that ARE fp32 numbers: the independent numpy fp32 -> bf16 rounding of synth must agree bit for bit
    x = np.random.default_rng(0).standard_normal(4000).astype(np.float32)
    assert np.array_equal(oracle.double_to_bf16(x.astype(np.float64)), f32_to_bf16_bits(x))


def test_rope_identity_table_is_the_plain_append():
    s, cos, sin = _rope_case()
    kp0, vp0 = s.copy_pools()
    oracle.kv_append(kp0, vp0, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    kp, vp = s.copy_pools()
    oracle.kv_append_rope(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new,
                          np.ones_like(cos), np.zeros_like(sin))
    assert np.array_equal(kp, kp0) and np.array_equal(vp, vp0)


def test_rope_quarter_turn_swaps_and_negates_and_v_is_copied():
    """cos = 0, sin = 1: k'[c] = -k[c + d/2], k'[c + d/2] = k[c], exactly (sign flip and swap of bf16 patterns): pins
    the pairing (c, c + d/2) -- an interleaved (2c, 2c + 1) convention fails -- and both signs."""
    s, cos, sin = _rope_case()
    kp, vp = s.copy_pools()
    oracle.kv_append_rope(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new,
                          np.zeros_like(cos), np.ones_like(sin))
    half = s.head_dim // 2
    for i in range(s.num_reqs):
        for t in range(int(s.q_lens[i])):
            pos = int(s.ctx_lens[i]) + t
            row = kp[s.page_table[i, pos // 16], :, pos % 16, :]
            src = s.k_new[int(s.q_offsets[i]) + t]
            assert np.array_equal(row[:, :half], src[:, half:] ^ np.uint16(0x8000))
            assert np.array_equal(row[:, half:], src[:, :half])
            assert np.array_equal(vp[s.page_table[i, pos // 16], :, pos % 16, :], s.v_new[int(s.q_offsets[i]) + t])


def test_rope_uses_the_table_row_of_the_tokens_position():
    """Only table row p* is a quarter turn, every other row the identity: exactly the token at position c_i + t == p* of
    each request is rotated."""
    s, cos, sin = _rope_case(q_lens=(37, 1, 1), ctx_lens=(5, 20, 31))
    p_star = 20
    c2, s2 = np.ones_like(cos), np.zeros_like(sin)
    c2[p_star], s2[p_star] = 0.0, 1.0
    kp, vp = s.copy_pools()
    oracle.kv_append_rope(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new, c2, s2)
    rotated = 0
    for i in range(s.num_reqs):
        for t in range(int(s.q_lens[i])):
            pos = int(s.ctx_lens[i]) + t
            row = kp[s.page_table[i, pos // 16], :, pos % 16, :]
            same = np.array_equal(row, s.k_new[int(s.q_offsets[i]) + t])
            assert same == (pos != p_star)
            rotated += not same
    assert rotated == 2     # request 0 (t = 15) and request 1 (its decode token at position 20)


def test_rope_rotation_invariants():
    """On the unrounded rotation: every (c, c + d/2) pair keeps its norm, and scores depend on the distance only:
    (R_m q) . (R_n k) = (R_{m-n} q) . (R_0 k) -- the property the embedding exists for."""
    rng = np.random.default_rng(51)
    d, n = 128, 64
    cos, sin = synth.make_rope_tables(512, d)
    rows = f32_to_bf16_bits(rng.standard_normal((n, d)).astype(np.float32))
    pos = rng.integers(0, 512, n).astype(np.int32)
    rot = oracle.rope_rotate(rows, pos, cos, sin)
    x = bf16_to_f64(rows)
    half = d // 2
    # fp32 tables: cos^2 + sin^2 = 1 to ~1e-7
    assert np.allclose(rot[:, :half] ** 2 + rot[:, half:] ** 2, x[:, :half] ** 2 + x[:, half:] ** 2, rtol=1e-6, atol=1e-9)
    q = f32_to_bf16_bits(rng.standard_normal((1, d)).astype(np.float32))
    k = f32_to_bf16_bits(rng.standard_normal((1, d)).astype(np.float32))
    for m, nn in ((300, 100), (17, 3), (511, 500)):
        lhs = float((oracle.rope_rotate(q, [m], cos, sin) @ oracle.rope_rotate(k, [nn], cos, sin).T)[0, 0])
        rhs = float((oracle.rope_rotate(q, [m - nn], cos, sin) @ oracle.rope_rotate(k, [0], cos, sin).T)[0, 0])
        assert abs(lhs - rhs) <= 2e-5 * (1 + abs(rhs))   # the fp32 tables are the only inexact part
    assert np.array_equal(oracle.rope_rotate(k, [0], cos, sin), bf16_to_f64(k))   # position 0: angle 0


def test_rope_append_equals_rotation_by_explicit_2x2_matrices():
    """A separate route to the stored bits: numpy fancy indexing for the placement, an explicit 2 x 2 rotation matrix per
    (position, pair) in float64, torch's own float64 -> bfloat16 conversion for the rounding."""
    s, cos, sin = _rope_case(seed=52, d=128, q_lens=(70, 1), ctx_lens=(9, 300))
    kp, vp = s.copy_pools()
    oracle.kv_append_rope(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new, cos, sin)
    half = s.head_dim // 2
    for i in range(s.num_reqs):
        for t in (0, int(s.q_lens[i]) - 1):
            pos = int(s.ctx_lens[i]) + t
            src = bf16_to_f64(s.k_new[int(s.q_offsets[i]) + t])          # [Hkv, d]
            want = np.empty_like(src)
            for c in range(half):
                R = np.array([[cos[pos, c], -sin[pos, c]], [sin[pos, c], cos[pos, c]]], np.float64)
                want[:, [c, c + half]] = src[:, [c, c + half]] @ R.T
            bits = torch.from_numpy(want).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
            assert np.array_equal(kp[s.page_table[i, pos // 16], :, pos % 16, :], bits)
