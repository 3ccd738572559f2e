"""KV migration (PAPER.md:155 Path 1, :58, :101) through the C-ABI (tropical_kv_migrate) against
oracle.kv_migrate: destination pools bit-identical over the WHOLE pool, source untouched, and attention on the migrated
requests equal to attention on the originals bit for bit."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_16264_b200 as tb
import synth
from tests.gpu_harness import DeviceStep, bits, to_dev

pytestmark = pytest.mark.gpu


def _migrate_and_compare(s, kv_lens, seed, num_dst_pages=None):
    """Migrate kv_lens[m] tokens of every request of step s (whose pools already hold them) into a poisoned destination
    pool under a fresh page table; compare with the oracle over both whole pools.  Returns the device-side pieces."""
    rng = np.random.default_rng(seed)
    Hkv, P, d = s.num_kv_heads, s.page_size, s.head_dim
    dst_pt, n_dst = synth.make_migration_target(rng, kv_lens, P, num_pages=num_dst_pages)
    kd_ref = np.full((n_dst, Hkv, P, d), synth.POISON_BF16, np.uint16)
    vd_ref = kd_ref.copy()
    oracle.kv_migrate(s.k_pool, s.v_pool, kd_ref, vd_ref, kv_lens, s.page_table, dst_pt)

    k_src, v_src = to_dev(s.k_pool), to_dev(s.v_pool)
    k_dst = torch.full((n_dst, Hkv, P, d), synth.POISON_BF16, dtype=torch.int16, device="cuda")
    v_dst = k_dst.clone()
    src, dst = tb.KVPool(k_src, v_src, s.num_q_heads), tb.KVPool(k_dst, v_dst, s.num_q_heads)
    lens_d = torch.tensor(np.asarray(kv_lens, np.int32), device="cuda")
    spt, dpt = to_dev(s.page_table), to_dev(dst_pt)
    tb.kv_migrate(src, dst, lens_d, spt, dpt, int(max(kv_lens)) if len(kv_lens) else 0)
    torch.cuda.synchronize()
    assert np.array_equal(bits(k_dst), kd_ref), "destination K pool differs from the oracle's"
    assert np.array_equal(bits(v_dst), vd_ref), "destination V pool differs from the oracle's"
    assert np.array_equal(bits(k_src), s.k_pool) and np.array_equal(bits(v_src), s.v_pool), "source was written"
    return dst, dst_pt, dpt


@pytest.mark.parametrize("Hkv,d", [(1, 64), (2, 128), (3, 64), (8, 128), (5, 128), (9, 64), (40, 128)])
def test_migrate_edge_lengths_whole_pool_bit_exact(Hkv, d):
    """Lengths around page edges (ragged last pages move only their valid slots), empty requests, one long request;
    head counts that are not a multiple of the heads per copy unit (4 at d = 128, 8 at d = 64)."""
    kv_lens = [1, 15, 16, 17, 0, 31, 32, 33, 255, 256, 257, 1000, 0, 4097]
    s = synth.make_step(np.random.default_rng(60 + Hkv), Hkv, Hkv, d, 16, [0] * len(kv_lens), kv_lens)
    _migrate_and_compare(s, kv_lens, 61 + Hkv)


def test_migrate_single_request_and_empty_list():
    s = synth.make_step(np.random.default_rng(70), 8, 8, 128, 16, [0], [777])
    _migrate_and_compare(s, [777], 71)
    _migrate_and_compare(s, [0], 72)
    pool = tb.KVPool(to_dev(s.k_pool), to_dev(s.v_pool), 8)
    empty = torch.zeros((0,), dtype=torch.int32, device="cuda")
    tb.kv_migrate(pool, pool, empty, torch.zeros((0, 1), dtype=torch.int32, device="cuda"),
                  torch.zeros((0, 1), dtype=torch.int32, device="cuda"), 0)


def test_migrate_more_requests_than_one_launch_takes():
    """2500 short requests: the launcher splits the list into launches of 1024 requests."""
    rng = np.random.default_rng(73)
    kv_lens = rng.integers(0, 70, 2500).tolist()
    s = synth.make_step(rng, 2, 2, 64, 16, [0] * len(kv_lens), kv_lens)
    _migrate_and_compare(s, kv_lens, 74)
    assert tb.last_launch_count() == 3


def test_partial_migration_moves_a_prefix_only():
    """kv_lens smaller than what the source holds: only the first kv_lens[m] tokens move (e.g. a cache migrated while
    the request's last chunk is still being prefilled)."""
    have = [300, 64, 1000]
    move = [129, 64, 17]
    s = synth.make_step(np.random.default_rng(75), 4, 4, 128, 16, [0] * 3, have)
    _migrate_and_compare(s, move, 76)


def test_attention_after_migration_is_bit_identical():
    """the request decodes on the destination worker.  Same step on the migrated cache (destination pool,
    destination page table) as on the original: outputs equal bit for bit, and within tolerance of the oracle."""
    s = synth.make_step(np.random.default_rng(77), 16, 4, 128, 16, [1, 1, 1, 1, 40], [700, 16, 2500, 63, 130])
    ref, _, kp, vp = oracle.step(s)
    dev = DeviceStep(s)
    out_src, _ = dev.step()
    L = (s.q_lens + s.ctx_lens).tolist()
    # migrate the post-append caches
    s_after = synth.StepInputs(s.name, s.seed, s.num_q_heads, s.num_kv_heads, s.head_dim, 16, s.num_pages, s.q_lens,
                               s.ctx_lens, s.q_offsets, s.page_table, kp, vp, s.q, s.k_new, s.v_new)
    dst, dst_pt, dpt = _migrate_and_compare(s_after, L, 78)
    batch = tb.Batch(dev.batch.q_lens, dev.batch.ctx_lens, dev.batch.q_offsets, dpt, s.total_q, s.max_kv_len)
    out2 = torch.zeros_like(dev.q)
    ws = torch.empty(tb.workspace_bytes(dst, s.num_reqs, s.total_q, s.max_kv_len) + 256, dtype=torch.uint8, device="cuda")
    tb.mixed_attention(dst, batch, dev.q, out=out2, workspace=ws)
    torch.cuda.synchronize()
    assert np.array_equal(bits(out2), bits(dev.out))
    assert np.abs(out_src - ref).max() <= 2e-2


def test_migrate_full_C5_cache_whole_pool_bit_exact():
    """BASELINE.json configs[4] at full size: the caches of all 258 requests after the step (617 686 tokens, 2.5 GB of
    K + V) move to a second pool; both destination pools compared bit for bit with the oracle's over the whole pool."""
    s = synth.make_config("C5", poison=True, values="tiled")
    kp, vp = s.copy_pools()
    oracle.kv_append(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    L = (s.q_lens.astype(np.int64) + s.ctx_lens).tolist()
    s_after = synth.StepInputs(s.name, s.seed, s.num_q_heads, s.num_kv_heads, s.head_dim, 16, s.num_pages, s.q_lens,
                               s.ctx_lens, s.q_offsets, s.page_table, kp, vp, s.q, s.k_new, s.v_new)
    _migrate_and_compare(s_after, L, 79)


def test_migrate_rejects_mismatched_pools():
    a = torch.zeros((4, 2, 16, 128), dtype=torch.int16, device="cuda")
    b = torch.zeros((4, 4, 16, 128), dtype=torch.int16, device="cuda")
    lens = torch.ones(1, dtype=torch.int32, device="cuda")
    pt = torch.zeros((1, 1), dtype=torch.int32, device="cuda")
    with pytest.raises(tb.TropicalError):
        tb.kv_migrate(tb.KVPool(a, a.clone(), 2), tb.KVPool(b, b.clone(), 4), lens, pt, pt, 1)
    with pytest.raises(tb.TropicalError):
        tb.kv_migrate(tb.KVPool(a, a.clone(), 2), tb.KVPool(a.clone(), a.clone(), 2), lens, pt, pt, 40)  # stride < pages


# ------------------------------------------------------------------ the GPU-to-GPU hop (needs a second GPU)
def _two_gpus():
    return torch.cuda.is_available() and torch.cuda.device_count() >= 2


needs_two_gpus = pytest.mark.skipif(not _two_gpus(), reason="KV migration to a peer GPU needs 2 visible GPUs (P:155 Path 1, P:171)")


def _peer_migration(d0, d1):
    """Body of the peer test; (d0, d1) = (0, 0) runs the same code on one GPU (how it was exercised before any 2-GPU box)."""
    with torch.cuda.device(d0):
        if not tb.enable_peer_access(d1):
            pytest.skip(f"no peer path between cuda:{d0} and cuda:{d1}")
        s = synth.make_step(np.random.default_rng(90), 16, 4, 128, 16, [1, 1, 1, 1, 40], [700, 16, 2500, 63, 130])
        ref, _, kp, vp = oracle.step(s)
        dev = DeviceStep(s)
        out_src, _ = dev.step()
        L = (s.q_lens + s.ctx_lens).tolist()
        Hkv, P, d = s.num_kv_heads, s.page_size, s.head_dim
        dst_pt, n_dst = synth.make_migration_target(np.random.default_rng(91), L, P)
        kd_ref = np.full((n_dst, Hkv, P, d), synth.POISON_BF16, np.uint16)
        vd_ref = kd_ref.copy()
        oracle.kv_migrate(kp, vp, kd_ref, vd_ref, L, s.page_table, dst_pt)
        k_dst = torch.full((n_dst, Hkv, P, d), synth.POISON_BF16, dtype=torch.int16, device=f"cuda:{d1}")
        v_dst = k_dst.clone()
        torch.cuda.synchronize(d1)
        dst = tb.KVPool(k_dst, v_dst, s.num_q_heads)
        tb.kv_migrate(dev.pool, dst, torch.tensor(np.asarray(L, np.int32), device=f"cuda:{d0}"), to_dev(s.page_table),
                      to_dev(dst_pt), int(max(L)))
        torch.cuda.synchronize(d0)
        assert np.array_equal(bits(k_dst), kd_ref), "peer destination K pool differs from the oracle's"
        assert np.array_equal(bits(v_dst), vd_ref), "peer destination V pool differs from the oracle's"
        assert np.array_equal(bits(dev.k_pool), kp) and np.array_equal(bits(dev.v_pool), vp), "source was written"
        out0 = bits(dev.out).copy()
    with torch.cuda.device(d1):  # the request now decodes on the destination worker
        to1 = lambda t: t.to(f"cuda:{d1}")
        batch = tb.Batch(to1(dev.batch.q_lens), to1(dev.batch.ctx_lens), to1(dev.batch.q_offsets),
                         torch.from_numpy(dst_pt).to(f"cuda:{d1}"), s.total_q, s.max_kv_len)
        q1 = to1(dev.q)
        out1 = torch.zeros_like(q1)
        tb.mixed_attention(dst, batch, q1, out=out1)
        torch.cuda.synchronize(d1)
        assert np.array_equal(bits(out1), out0)
    assert np.abs(out_src - ref).max() <= 2e-2


def _head_shards(d0, d1):
    s = synth.make_step(np.random.default_rng(92), 16, 4, 128, 16, [300, 1, 1, 1, 17], [200, 4097, 513, 15, 0])
    tb.debug_set_split_pages(32)  # the automatic split size depends on the head count: pin the split boundaries equal
    try:
        with torch.cuda.device(d0):
            full = DeviceStep(s)
            full.step(impl="product")
            want = bits(full.out).copy()
        Hq, Hkv = s.num_q_heads, s.num_kv_heads
        shards = []
        for r, dv in enumerate((d0, d1)):
            hq = slice(r * Hq // 2, (r + 1) * Hq // 2)
            hk = slice(r * Hkv // 2, (r + 1) * Hkv // 2)
            sh = synth.StepInputs(s.name, s.seed, Hq // 2, Hkv // 2, s.head_dim, 16, s.num_pages, s.q_lens, s.ctx_lens,
                                  s.q_offsets, s.page_table, np.ascontiguousarray(s.k_pool[:, hk]),
                                  np.ascontiguousarray(s.v_pool[:, hk]), np.ascontiguousarray(s.q[:, hq]),
                                  np.ascontiguousarray(s.k_new[:, hk]), np.ascontiguousarray(s.v_new[:, hk]))
            with torch.cuda.device(dv):
                shards.append(DeviceStep(sh))
        for dv, dev in zip((d0, d1), shards):  # both GPUs busy at once: enqueue on each, then wait for both
            with torch.cuda.device(dv):
                dev.append()
                dev.attention()
        for dv in (d0, d1):
            torch.cuda.synchronize(dv)
        got = np.concatenate([bits(dev.out) for dev in shards], axis=1)
        assert np.array_equal(got, want)
    finally:
        tb.debug_set_split_pages(0)


@needs_two_gpus
def test_peer_migration_whole_destination_pool_bit_exact_and_attention_on_the_peer():
    """Source pool on cuda:0, destination pool on cuda:1, mapped into cuda:0 by tropical_enable_peer_access; the kernel
    runs on cuda:0 and its bulk stores land in peer memory over NVLink.  Destination bit-identical to oracle.kv_migrate
    over the whole pool, source untouched, and the same decode step on cuda:1 over the migrated cache gives the bits
    cuda:0 gives over the original.  NEVER RUN on two GPUs so far (every box this suite has seen had one); the body was
    run with both roles on one GPU."""
    _peer_migration(0, 1)


@needs_two_gpus
def test_head_shards_on_two_gpus_concatenate_to_the_unsharded_step():
    """TP = 2 inside a worker: kv heads [0, Hkv/2) with their q heads on cuda:0, the rest on cuda:1, both steps
    enqueued before either is waited for; the concatenated outputs equal the one-GPU step bit for bit."""
    _head_shards(0, 1)


def test_two_gpu_test_bodies_on_one_gpu():
    """The bodies of the two tests above with both roles on cuda:0, so that the code a 2-GPU box will run for the first
    time has at least run (same kernels, no NVLink hop)."""
    _peer_migration(0, 0)
    _head_shards(0, 0)
