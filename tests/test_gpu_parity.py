"""GPU-vs-oracle parity, through the C-ABI (paper_2606_16264_b200.binding -> libtropical.so).

Bars (BASELINE.json north_star): KV append and page gather bit-exact over the WHOLE pool;
attention output max |d| <= 2e-2 and mean |d| <= 2e-3 against the fp64 oracle.
Needle tests make the page gather *through the attention kernel* bit-exact.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_16264_b200 as tb
import synth
from synth import f32_to_bf16_bits
from tests.gpu_harness import MAX_ABS_TOL, MEAN_ABS_TOL, DeviceStep, bits, errors

pytestmark = pytest.mark.gpu


def _step(seed, Hq, Hkv, d, q_lens, ctx_lens, **kw):
    return synth.make_step(np.random.default_rng(seed), Hq, Hkv, d, 16, q_lens, ctx_lens, **kw)


def _check_step(s, impl="both", sm_scale=0.0, lse_tol=2e-3):
    """impl "product": tropical_kv_append + tropical_mixed_attention; "fused": the single call tropical_mixed_step (append
    inside the step kernel, new rows read from k_new / v_new); "both" (default): each against the oracle, and the two
    outputs bit-identical to one another (same bits in, same work decomposition)."""
    ref_out, ref_lse, kp, vp = oracle.step(s, sm_scale)
    outs = []
    for one in (("product", "fused") if impl == "both" else (impl,)):
        dev = DeviceStep(s)
        out, lse = dev.step(sm_scale, one)
        # A1/A2: pool bit-identical to the oracle's over the whole pool; the attention roles never write elsewhere
        assert np.array_equal(bits(dev.k_pool), kp), f"K pool differs ({one})"
        assert np.array_equal(bits(dev.v_pool), vp), f"V pool differs ({one})"
        assert np.isfinite(out).all()
        mx, mean = errors(out, ref_out)
        assert mx <= MAX_ABS_TOL and mean <= MEAN_ABS_TOL, (one, mx, mean)
        if s.total_q:
            assert np.abs(lse - ref_lse).max() <= lse_tol
        outs.append(bits(dev.out).copy())
        del dev
    if len(outs) == 2:
        assert np.array_equal(outs[0], outs[1]), "fused step and append + attention differ"
    return mx, mean


# ------------------------------------------------------------------ BASELINE configs[0]
@pytest.mark.parametrize("impl", ["product", "fused", "auto", "simt"])
def test_C1_tiny_mixed_step(impl):
    s = synth.make_config("C1")
    mx, mean = _check_step(s, impl)
    assert mx < 1.2e-2  # diagnostic band O10: far above this signals a bug even inside tolerance


def test_C1_gather_bit_exact():
    s = synth.make_config("C1")
    _, _, kp, vp = oracle.step(s)
    dev = DeviceStep(s)
    dev.append()
    for i in range(s.num_reqs):
        n = int(s.ctx_lens[i] + s.q_lens[i])
        kd, vd = tb.kv_gather(dev.pool, dev.batch, i, n)
        ok, ov = oracle.kv_gather(kp, vp, s.page_table, i, n)
        assert np.array_equal(bits(kd), ok) and np.array_equal(bits(vd), ov)


# ------------------------------------------------------------------ edge-case matrix
EDGE_Q = [0, 1, 2, 15, 16, 17, 127, 128, 129, 255, 256, 257, 1000]
EDGE_C = [0, 1, 15, 16, 17, 127, 128, 129, 255, 256, 257, 511, 512, 513, 4095, 4096, 4097]


@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("g", [1, 4, 8])
def test_edge_matrix_q_by_c(d, g):
    """The full product EDGE_Q x EDGE_C (13 x 17 = 221 (q, c) pairs) for every (d, g): one step per q whose 17 requests
    carry all the c values, so every pairing of a chunk length with a prior-context length is compared with the oracle
    over all of its outputs."""
    Hkv = 2 if g < 8 else 1
    rng = np.random.default_rng(100 + d + g)
    for q in EDGE_Q:
        s = synth.make_step(rng, Hkv * g, Hkv, d, 16, [q] * len(EDGE_C), EDGE_C)
        _check_step(s)


@pytest.mark.parametrize("d", [64, 128])
def test_every_context_edge_as_decode(d):
    s = _step(7, 8, 2, d, [1] * len(EDGE_C), EDGE_C)
    _check_step(s)


@pytest.mark.parametrize("order", ["decode_first", "prefill_first", "interleaved", "only_decode", "only_prefill", "single", "with_skips"])
def test_request_orders(order):
    qs = {"decode_first": [1, 1, 1, 200, 33], "prefill_first": [200, 33, 1, 1, 1], "interleaved": [1, 200, 1, 33, 1],
          "only_decode": [1, 1, 1, 1], "only_prefill": [130, 64, 2], "single": [77], "with_skips": [0, 1, 0, 40, 0]}[order]
    cs = [(37 * (i + 1)) % 300 for i in range(len(qs))]
    _check_step(_step(8, 8, 4, 128, qs, cs))


def test_empty_batch_is_a_noop():
    import paper_2606_16264_b200 as tb
    kp = torch.zeros((4, 2, 16, 128), dtype=torch.int16, device="cuda")
    pool = tb.KVPool(kp, kp.clone(), 4)
    batch = tb.Batch.from_host([], [], np.zeros((0, 1), np.int32))
    q = torch.zeros((0, 4, 128), dtype=torch.int16, device="cuda")
    tb.kv_append(pool, batch, q[:, :2], q[:, :2])
    out = tb.mixed_attention(pool, batch, q)
    assert out.shape[0] == 0


def test_custom_scale_and_chunk_on_prior_context():
    """S13 variant C4b shape in small: chunk on prior context (third chunk), plus sm_scale override."""
    s = _step(9, 4, 4, 128, [256, 1, 1], [512, 100, 1023])
    _check_step(s, sm_scale=0.05)
    _check_step(s)


# ------------------------------------------------------------------ O7 on the GPU
def test_chunked_equals_unchunked_and_decode_equals_last_row():
    rng = np.random.default_rng(10)
    L, Hq, Hkv, d = 300, 4, 2, 128
    whole = synth.make_step(rng, Hq, Hkv, d, 16, [L], [0])
    ref, _, kp, vp = oracle.step(whole)
    dev = DeviceStep(whole)
    out_whole, _ = dev.step()
    # second half as a chunk over the first half as context: reuse the appended pool
    L1 = 140
    s2 = synth.StepInputs("chunk", -1, Hq, Hkv, d, 16, whole.num_pages, np.array([L - L1], np.int32),
                          np.array([L1], np.int32), np.array([0, L - L1], np.int32), whole.page_table, kp, vp,
                          whole.q[L1:].copy(), whole.k_new[L1:].copy(), whole.v_new[L1:].copy())
    out_chunk, _ = DeviceStep(s2).step()
    assert errors(out_chunk, ref[L1:])[0] <= MAX_ABS_TOL
    assert np.abs(out_chunk - out_whole[L1:]).max() <= 2e-2
    s3 = synth.StepInputs("dec", -1, Hq, Hkv, d, 16, whole.num_pages, np.array([1], np.int32),
                          np.array([L - 1], np.int32), np.array([0, 1], np.int32), whole.page_table, kp, vp,
                          whole.q[L - 1:].copy(), whole.k_new[L - 1:].copy(), whole.v_new[L - 1:].copy())
    out_dec, _ = DeviceStep(s3).step()
    assert errors(out_dec, ref[L - 1:])[0] <= MAX_ABS_TOL


# ------------------------------------------------------------------ O8 needle (bit-exact gather through attention)
def _needle_step(d, c, ql, targets_fn, Hq=2, Hkv=1, seed=0, values="normal"):
    rng = np.random.default_rng(seed)
    L = c + ql

    def code(j):
        vec = np.full(d, 32.0, np.float32)
        vec[:14] = np.where((j >> np.arange(14)) & 1, 32.0, -32.0)
        return vec

    K = np.stack([code(j) for j in range(L)])[:, None, :].repeat(Hkv, 1)
    V = rng.standard_normal((L, Hkv, d)).astype(np.float32)
    targets = [targets_fn(t) for t in range(ql)]
    Q = np.stack([code(j) for j in targets])[:, None, :].repeat(Hq, 1)
    s = synth.make_step(rng, Hq, Hkv, d, 16, [ql], [c], values=values)
    Kb, Vb = f32_to_bf16_bits(K), f32_to_bf16_bits(V)
    # install prior context rows [0,c) directly, new rows via the append under test
    for j in range(c):
        s.k_pool[s.page_table[0, j // 16], :, j % 16, :] = Kb[j]
        s.v_pool[s.page_table[0, j // 16], :, j % 16, :] = Vb[j]
    s.k_new[:], s.v_new[:], s.q[:] = Kb[c:], Vb[c:], f32_to_bf16_bits(Q)
    return s, targets, Vb


@pytest.mark.parametrize("impl", ["fused", "product"])
@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("c,ql", [(300, 200), (0, 257), (4090, 1), (1000, 1), (127, 130), (16, 129), (15, 2), (4095, 1)])
def test_needle_selects_target_row_bitwise(d, c, ql, impl):
    edges = [0, 15, 16, 17, 127, 128, 129, 255, 256, 257, 511, 512, 513, 1023, 1024, 1025]

    def target(t):
        lim = c + t
        k = t % 4
        if k == 0:
            return lim                      # own just-appended row: append->attend order, diagonal included
        if k == 1:
            return max(lim - 1, 0)
        if k == 2:
            return min(edges[(t // 4) % len(edges)], lim)
        return (t * 7919) % (lim + 1)

    s, targets, Vb = _needle_step(d, c, ql, target)
    dev = DeviceStep(s)
    dev.step(impl=impl)   # fused: the just-appended rows reach the tiles from k_new / v_new, not through the pool
    got = bits(dev.out)
    for t, j in enumerate(targets):
        for h in range(s.num_q_heads):
            assert np.array_equal(got[t, h], Vb[j, 0]), f"row {t} head {h}: expected V[{j}]"


@pytest.mark.parametrize("impl", ["fused", "product"])
def test_negative_needle_future_key_not_selected(impl):
    c, ql, d = 40, 50, 128
    s, targets, Vb = _needle_step(d, c, ql, lambda t: min(c + t + 1, c + ql - 1))
    ref, _, _, _ = oracle.step(s)
    dev = DeviceStep(s)
    out, _ = dev.step(impl=impl)
    assert errors(out, ref)[0] <= MAX_ABS_TOL
    got = bits(dev.out)
    assert not np.array_equal(got[3, 0], Vb[c + 3 + 1, 0])


def test_append_then_attention_ordering_stress():
    """Stream ordering of the step's three launches (append -> tile directory, which overlaps the append by programmatic
    dependent launch -> step kernel): a C4-sized append (2048 tokens x 40 kv heads, ~45 MB of scattered rows) directly
    followed by the attention that reads those rows, 200 times.  Before every repetition the target slots are
    overwritten with NaN patterns and V alternates between two draws, so a step kernel that started before the append
    had landed would return NaN or the other draw's rows.  Needle queries select the just-appended row: bit-exact."""
    d, ql, H = 128, 2048, 40
    s, targets, Vb = _needle_step(d, 0, ql, lambda t: t, Hq=H, Hkv=H, seed=5, values="tiled")
    assert targets == list(range(ql))
    dev = DeviceStep(s)
    rng = np.random.default_rng(6)
    v_alt = f32_to_bf16_bits(rng.standard_normal((ql, 1, d)).astype(np.float32))
    v_sets = [s.v_new.copy(), np.ascontiguousarray(np.broadcast_to(v_alt, (ql, H, d)))]
    v_dev = [torch.from_numpy(v.view(np.int16)).cuda() for v in v_sets]
    pages = dev.batch.page_table[0, : ql // 16].long()
    for rep in range(200):
        dev.k_pool[pages] = synth.POISON_BF16
        dev.v_pool[pages] = synth.POISON_BF16
        dev.out.zero_()
        tb.kv_append(dev.pool, dev.batch, dev.k_new, v_dev[rep & 1])
        tb.mixed_attention(dev.pool, dev.batch, dev.q, out=dev.out, workspace=dev.workspace)
        if rep % 20 == 19 or rep < 4:
            torch.cuda.synchronize()
            got = bits(dev.out)
            assert np.array_equal(got, v_sets[rep & 1][:, :, :]), f"repetition {rep}: stale or poisoned rows were read"
    torch.cuda.synchronize()


def test_fused_step_never_reads_the_slots_it_appends():
    """tropical_mixed_step: the attention roles take this step's rows from k_new / v_new while other warps of the same
    kernel copy them into the pool.  The target slots hold NaN patterns when the kernel starts and V alternates between
    two draws, 100 times, on a mixed batch whose chunk starts in the middle of a page (context 1000 = 62.5 pages) next to
    decode requests whose new token lands on every slot position: needle queries select just-appended rows bit-exactly,
    and after every repetition the pool holds exactly the appended rows."""
    d, H = 128, 8
    rng = np.random.default_rng(41)
    ql, c = 600, 1000
    s, targets, Vb = _needle_step(d, c, ql, lambda t: c + t, Hq=H, Hkv=H, seed=7)
    dev = DeviceStep(s)
    v_alt = f32_to_bf16_bits(rng.standard_normal((ql, 1, d)).astype(np.float32))
    v_sets = [s.v_new.copy(), np.ascontiguousarray(np.broadcast_to(v_alt, (ql, H, d)))]
    v_dev = [torch.from_numpy(v.view(np.int16)).cuda() for v in v_sets]
    pos = torch.arange(c, c + ql, device="cuda")
    pages, slots = dev.batch.page_table[0, (pos // 16).long()].long(), (pos % 16).long()
    for rep in range(100):
        dev.k_pool[pages, :, slots] = synth.POISON_BF16
        dev.v_pool[pages, :, slots] = synth.POISON_BF16
        dev.out.zero_()
        tb.debug_set_fused(1)   # the fused variant whatever the batch (this one would choose it anyway)
        try:
            tb.mixed_step(dev.pool, dev.batch, dev.q, dev.k_new, v_dev[rep & 1], out=dev.out, workspace=dev.workspace)
        finally:
            tb.debug_set_fused(-1)
        if rep % 10 == 9 or rep < 4:
            torch.cuda.synchronize()
            assert np.array_equal(bits(dev.out), v_sets[rep & 1]), f"repetition {rep}: poisoned or stale rows were read"
            assert np.array_equal(bits(dev.v_pool[pages, :, slots]), v_sets[rep & 1]), f"repetition {rep}: append incomplete"
            assert np.array_equal(bits(dev.k_pool[pages, :, slots]), s.k_new)
    torch.cuda.synchronize()
    # decode requests whose new token lands on each of the 16 slots of its page, poisoned pool, both paths
    _check_step(_step(42, 8, 2, 128, [1] * 16 + [37], [200 + k for k in range(16)] + [5], poison=True))


def test_head_sharded_step_equals_unsharded_bit_for_bit():
    """SURVEY 8(e) / P:184 (tensor parallelism 2 inside a worker): the path shards by kv head with no collective.  Two
    pools holding kv heads [0, Hkv/2) and [Hkv/2, Hkv) of the same step, each run with Hq/2 and Hkv/2: the concatenated
    outputs equal the unsharded run bit for bit (the decode split boundaries are pinned equal with the test hook,
    since the automatic split size depends on the head count), and the oracle within tolerance."""
    Hq, Hkv, d = 64, 8, 128
    rng = np.random.default_rng(31)
    ctx = np.clip(np.rint(np.exp(np.log(1500) + 1.0 * rng.standard_normal(24))), 64, 8192).astype(int).tolist()
    s = synth.make_step(rng, Hq, Hkv, d, 16, [700, 130] + [1] * 24, [0, 300] + ctx)
    ref, ref_lse, kp, vp = oracle.step(s)
    tb.debug_set_split_pages(32)
    try:
        dev = DeviceStep(s)
        out, lse = dev.step()
        whole = bits(dev.out).copy()
        assert errors(out, ref)[0] <= MAX_ABS_TOL and errors(out, ref)[1] <= MEAN_ABS_TOL
        g = Hq // Hkv
        parts, lses = [], []
        for r in range(2):
            hk = slice(r * Hkv // 2, (r + 1) * Hkv // 2)
            hq = slice(r * Hq // 2, (r + 1) * Hq // 2)
            sh = synth.StepInputs(f"shard{r}", -1, Hq // 2, Hkv // 2, d, 16, s.num_pages, s.q_lens, s.ctx_lens,
                                  s.q_offsets, s.page_table, np.ascontiguousarray(s.k_pool[:, hk]),
                                  np.ascontiguousarray(s.v_pool[:, hk]), np.ascontiguousarray(s.q[:, hq]),
                                  np.ascontiguousarray(s.k_new[:, hk]), np.ascontiguousarray(s.v_new[:, hk]))
            dsh = DeviceStep(sh)
            _, l_sh = dsh.step()
            parts.append(bits(dsh.out).copy())
            lses.append(l_sh)
            assert np.array_equal(bits(dsh.k_pool), kp[:, hk]) and np.array_equal(bits(dsh.v_pool), vp[:, hk])
        assert g == 8
        assert np.array_equal(np.concatenate(parts, axis=1), whole)
        assert np.array_equal(np.concatenate(lses, axis=1), lse)
    finally:
        tb.debug_set_split_pages(0)


# ------------------------------------------------------------------ O9 poison + stray writes, determinism
def test_poison_pool_outputs_finite_and_pool_untouched_elsewhere():
    s = _step(12, 8, 2, 128, [129, 1, 1, 17], [3, 250, 4097, 60], poison=True)
    before_k = s.k_pool.copy()
    dev = DeviceStep(s)
    out, _ = dev.step()
    assert np.isfinite(out).all()
    after = bits(dev.k_pool)
    changed_rows = (after != before_k).any(axis=-1)
    assert changed_rows.sum() == s.total_q * s.num_kv_heads  # exactly the appended rows changed


@pytest.mark.parametrize("impl", ["fused", "product"])
def test_run_to_run_deterministic(impl):
    s = _step(13, 8, 2, 128, [300, 1, 1, 1], [0, 2000, 5000, 64])
    dev = DeviceStep(s)
    dev.step(impl=impl)
    a = bits(dev.out).copy()
    for _ in range(3):
        dev.out.zero_()
        dev.step(impl=impl)
        assert np.array_equal(bits(dev.out), a)
    dev.out.zero_()
    dev.attention()     # the plain variant on the pool the step has left: the same bits as either variant
    torch.cuda.synchronize()
    assert np.array_equal(bits(dev.out), a)


def test_product_path_matches_simt_cross_check():
    s = _step(14, 16, 2, 128, [513, 1, 1, 1, 40], [0, 777, 4097, 15, 130])
    dev = DeviceStep(s)
    a, la = dev.step(impl="product")
    b, lb = dev.step(impl="simt")
    assert np.abs(a - b).max() <= 2e-2 and np.abs(la - lb).max() <= 2e-3


# ------------------------------------------------------------------ queue sequencing: many tiles per CTA
@pytest.mark.parametrize("split", [0, 16, 24, 64])
@pytest.mark.parametrize("grid", [1, 2, 5])
@pytest.mark.parametrize("shape", [(8, 1, 128), (16, 2, 128), (4, 4, 64)])
def test_few_ctas_many_tiles_per_queue(grid, shape, split):
    """With the step kernel capped to a few CTAs every role walks long sequences of prefill items and decode
    units (ring wrap-around, mailbox and barrier phases, TMEM slot reuse, both decode pipelines of a CTA)."""
    Hq, Hkv, d = shape
    qs = [300, 1, 1, 1, 1, 40, 1, 1, 1, 1, 1, 1]
    cs = [0, 777, 4097, 15, 130, 100, 2000, 128, 127, 1, 513, 3000]
    s = _step(20 + grid, Hq, Hkv, d, qs, cs)
    tb.debug_set_grid(grid)
    tb.debug_set_split_pages(split)  # 0 = automatic (one 128-key block per unit at these sizes); else multi-block units
    try:
        _check_step(s)
        # decode only: the late pipeline (prefill memory) and the dedicated one share the queue from the start
        s2 = _step(30 + grid, Hq, Hkv, d, [1] * 9, [5000, 3000, 17, 900, 256, 255, 4096, 64, 2500])
        _check_step(s2)
    finally:
        tb.debug_set_grid(0)
        tb.debug_set_split_pages(0)


# ------------------------------------------------------------------ end-to-end host entry point
def test_step_host_equals_device_path():
    import paper_2606_16264_b200 as tb
    s = _step(15, 8, 2, 128, [150, 1, 1], [10, 300, 64])
    ref, ref_lse, kp, vp = oracle.step(s)
    dev = DeviceStep(s)
    pin = lambda a: torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).pin_memory()
    h_out = torch.zeros(s.q.shape, dtype=torch.int16).pin_memory()
    h_lse = torch.zeros((s.total_q, s.num_q_heads), dtype=torch.float32).pin_memory()
    staging = torch.empty(tb.step_host_staging_bytes(dev.pool, s.num_reqs, s.total_q, s.page_table_stride) + 256,
                          dtype=torch.uint8, device="cuda")
    tb.step_host(dev.pool, pin(s.q_lens), pin(s.ctx_lens), pin(s.q_offsets), pin(s.page_table), s.max_kv_len,
                 pin(s.q), pin(s.k_new), pin(s.v_new), h_out, staging, dev.workspace, h_lse=h_lse)
    out = synth.bf16_bits_to_f32(h_out.numpy().view(np.uint16)).astype(np.float64)
    assert errors(out, ref)[0] <= MAX_ABS_TOL and errors(out, ref)[1] <= MEAN_ABS_TOL
    assert np.array_equal(bits(dev.k_pool), kp)
    assert np.abs(h_lse.numpy() - ref_lse).max() <= 2e-3
    assert tb.last_launch_count() >= 2


# ------------------------------------------------------------------ head-group shapes and seeded random batches
@pytest.mark.parametrize("Hq,Hkv", [(6, 2), (2, 1), (16, 1), (48, 3), (64, 1), (5, 5), (12, 4)])
@pytest.mark.parametrize("d", [64, 128])
def test_head_group_shapes(Hq, Hkv, d):
    """g = Hq / Hkv odd (one query tile per item), g = 2 (pairs), g = 16 / 64 (several 8-head decode blocks per kv head),
    MHA with an odd head count: same step, every shape against the oracle."""
    s = _step(50 + Hq + Hkv, Hq, Hkv, d, [130, 1, 1, 1, 40], [5, 777, 2100, 15, 130])
    _check_step(s)


@pytest.mark.parametrize("seed", range(12))
def test_seeded_random_batches(seed):
    """Random mixes of skipped / decode / prefill requests (lengths around page, tile and split edges), random head
    configuration, requests in random order."""
    rng = np.random.default_rng(1000 + seed)
    Hkv = int(rng.choice([1, 2, 4]))
    g = int(rng.choice([1, 2, 3, 4, 8]))
    d = int(rng.choice([64, 128]))
    n = int(rng.integers(1, 12))
    edges = np.array([0, 1, 2, 15, 16, 17, 31, 127, 128, 129, 255, 256, 257, 383, 700])
    qs, cs = [], []
    for _ in range(n):
        kind = rng.integers(0, 4)
        q = 0 if kind == 0 else 1 if kind == 1 else int(rng.choice(edges[2:])) + int(rng.integers(0, 3))
        c = int(rng.choice(edges)) + int(rng.integers(0, 3)) + (int(rng.integers(0, 3000)) if kind == 1 else 0)
        qs.append(q)
        cs.append(c)
    s = synth.make_step(rng, Hkv * g, Hkv, d, 16, qs, cs)
    _check_step(s)


def test_step_is_cuda_graph_capturable_and_idempotent():
    """The step has no host sync and mutates none of its metadata: append + attention captured once in a CUDA graph
    replays to the same bits (tensor maps are kernel parameters; the plan kernel's dependent launch is captured)."""
    s = _step(17, 8, 2, 128, [200, 1, 1, 1, 33], [56, 700, 2049, 17, 0])
    ref, _, kp, vp = oracle.step(s)
    dev = DeviceStep(s)
    dev.step()                                  # eager run: also warms one-time function attributes
    eager = bits(dev.out).copy()
    dev.out.zero_()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            dev.append()
            dev.attention()
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(3):
        dev.out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(bits(dev.out), eager)
    assert np.array_equal(bits(dev.k_pool), kp) and np.array_equal(bits(dev.v_pool), vp)
    assert errors(dev.out_f64(), ref)[0] <= MAX_ABS_TOL


def test_fused_step_is_cuda_graph_capturable():
    s = _step(18, 8, 2, 128, [200, 1, 1, 1, 33], [56, 700, 2049, 17, 0])
    ref, _, kp, vp = oracle.step(s)
    dev = DeviceStep(s)
    dev.step(impl="fused")
    eager = bits(dev.out).copy()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    tb.debug_set_fused(1)
    try:
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                dev.fused_step()
    finally:
        tb.debug_set_fused(-1)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(3):
        dev.out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(bits(dev.out), eager)
    assert np.array_equal(bits(dev.k_pool), kp) and np.array_equal(bits(dev.v_pool), vp)
    assert errors(dev.out_f64(), ref)[0] <= MAX_ABS_TOL


def test_mixed_step_chooses_its_variant_from_the_batch_scalars():
    """tropical_mixed_step fuses the append into the step kernel on prefill-dominated steps (>= 64 new tokens per request
    on average: 2 launches) and runs the append kernel in front of the plain variant otherwise (3 launches); both
    leave the same pool and the same output bits."""
    outs = []
    for q, c, launches in (([200, 1], [56, 700], 2), ([200] + [1] * 7, [56] + [700] * 7, 3)):
        s = _step(21, 8, 2, 128, q, c)
        ref, _, kp, vp = oracle.step(s)
        dev = DeviceStep(s)
        dev.step(impl="auto")
        assert tb.last_launch_count() == launches
        assert np.array_equal(bits(dev.k_pool), kp) and np.array_equal(bits(dev.v_pool), vp)
        assert errors(dev.out_f64(), ref)[0] <= MAX_ABS_TOL


def test_more_requests_than_plan_threads():
    """1100 requests: the plan kernel's threads own two requests each and its ticket search falls back from the
    shared-memory tables (1024 requests) to the workspace."""
    rng = np.random.default_rng(77)
    n = 1100
    qs = [1] * n
    qs[5], qs[700] = 33, 2
    cs = rng.integers(0, 40, n).tolist()
    _check_step(_step(78, 2, 2, 64, qs, cs))


def test_long_contexts():
    """Contexts far beyond the configs' 8192 tokens: a decode request on 70 001 cached tokens (4376 pages: 137 split-K
    units per kv head under the automatic split) and a 300-token chunk on 66 000 (517 KV tiles per query tile), next to a
    short request; both step variants."""
    _check_step(_step(23, 4, 2, 128, [1, 300, 1], [70001, 66000, 5]))


def test_validate_batch_finds_the_first_bad_request():
    s = _step(19, 4, 2, 64, [40, 1, 1, 0, 5], [3, 100, 17, 9, 0])
    dev = DeviceStep(s)
    assert tb.validate_batch(dev.pool, dev.batch) is None
    pt = dev.batch.page_table.clone()
    dev.batch.page_table[2, 1] = s.num_pages            # page id out of range, inside request 2's extent
    assert tb.validate_batch(dev.pool, dev.batch) == 2
    dev.batch.page_table.copy_(pt)
    dev.batch.page_table[3, 5] = -7                     # beyond request 3's extent: ignored (reading S8)
    assert tb.validate_batch(dev.pool, dev.batch) is None
    dev.batch.q_offsets[2] += 1                         # prefix sums broken at request 1
    assert tb.validate_batch(dev.pool, dev.batch) == 1
    dev.batch.q_offsets[2] -= 1
    dev.batch.ctx_lens[4] = -1
    assert tb.validate_batch(dev.pool, dev.batch) == 4


def test_predictor_and_launcher_agree_on_the_step_variant():
    """The built-in cost fits are keyed on the kernel variant tropical_mixed_step picks (csrc/step_variant.h, one rule for
    both).  Either side of the rule's boundary: the launcher's choice shows in its launch count (2 = fused variant,
    3 = append kernel + plain variant), the predictor's in the critical-path feature of an MHA prefill item (the fused
    variant pairs the top two row tiles of a head: 3 + 2 KV iterations; the plain one takes the top tile alone: 3)."""
    for q0, fused in ((316, True), (315, False)):  # 4 decode requests: T = q0 + 4 against 64 * 5
        q_lens, ctx_lens = [q0, 1, 1, 1, 1], [0, 40, 300, 17, 5]
        s = _step(50, 8, 8, 128, q_lens, ctx_lens)
        dev = DeviceStep(s)
        dev.fused_step()
        torch.cuda.synchronize()
        assert tb.last_launch_count() == (2 if fused else 3)
        _, bd = tb.step_cost(8, 8, 128, 16, q_lens, ctx_lens, require_model=False)  # features only: no fit for 8/8
        assert bd.prefill_critical_iters == (5 if fused else 3)
