"""the scheduler simulation (include/tropical_sim.h).

Part 1 pins the Python oracle (oracle/sim_oracle.py) to what the paper and arithmetic fix: closed forms with a
degenerate cost model, eq. (1)-(3) on a hand-worked trace, the Fig. 7 slack-check scenario, the two
guards of P:159, the no-starvation reading, conservation invariants.  Part 2 is parity: the C++ simulator in
libtropical.so against the oracle, request by request, on seeded long-tail traces for all three policies.
"""
import math
import random

import pytest

import paper_2606_16264_b200 as tb
from oracle import sim_oracle as so

FLAT = (0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 148.0)         # attention term off: iteration = overhead + linear * tokens
FIT = (35.0, 1.0e-9, 1.15e-7, 0.15, 0.13, 0.057, 148.0, 0.2)  # a B200-like fit (64/8/128), values rounded by hand


def _ocfg(policy, cm=FLAT, **kw):
    d = dict(policy=policy, num_workers=2, num_prefill_workers=1, chunk_tokens=0, ttft_slo_us=1e9, tpot_slo_us=15.0,
             decode_guard=0.9, hbm_watermark=0.9, kv_capacity_tokens=10**9, migrate_us_per_token=0.0, num_q_heads=64,
             num_kv_heads=8, head_dim=128, page_size=16, num_layers=1, attn=so.CostModel(*cm), linear_us_per_token=0.1,
             iter_overhead_us=10.0)
    d.update(kw)
    return so.Config(**d)


def _ccfg(o: so.Config):
    a = o.attn
    sh, lm = o.layer, o.linear
    return tb.SimConfig(o.policy, o.num_workers, o.num_prefill_workers, o.chunk_tokens, o.ttft_slo_us, o.tpot_slo_us,
                        o.decode_guard, o.hbm_watermark, o.kv_capacity_tokens, o.migrate_us_per_token, o.num_q_heads,
                        o.num_kv_heads, o.head_dim, o.page_size, o.num_layers,
                        tb.CostModel(a.t0_us, a.a_us_per_flop, a.b_us_per_byte, a.kappa, a.e_prefill_iter_us,
                                     a.e_decode_unit_us, a.n_sm, a.e_prefill_crit_us), o.linear_us_per_token,
                        o.iter_overhead_us,
                        tb.LayerShape(sh.d_model, sh.d_ffn, sh.gated_mlp, sh.num_layers, sh.tp),
                        tb.LinearModel(lm.g0_us, lm.f_us_per_flop, lm.w_us_per_byte, lm.kappa, lm.ar0_us, lm.ar_us_per_byte),
                        o.role_transitions, o.delay_threshold)


# ------------------------------------------------------------------------------------------ part 1: oracle pins
def test_single_request_closed_form():
    """One worker, one request (prompt 100, 5 output tokens): TTFT = overhead + linear * prompt = 10 + 10; every decode
    iteration = 10 + 0.1, so TPOT = 10.1 and finish = 20 + 4 * 10.1 (P:52 definitions)."""
    res, summ = so.simulate(_ocfg(so.COLOCATED, num_workers=1), [(3.0, 100, 5)])
    assert res[0]["ttft_us"] == pytest.approx(20.0) and res[0]["tpot_us"] == pytest.approx(10.1)
    assert res[0]["finish_us"] == pytest.approx(3.0 + 20.0 + 4 * 10.1)
    assert summ["iterations"] == 5 and summ["attainment"] == 1.0


def test_chunked_prefill_splits_the_prompt():
    """chunk 40 on a 100-token prompt: three prefill iterations of 10 + 4, 10 + 4, 10 + 2."""
    res, summ = so.simulate(_ocfg(so.COLOCATED, num_workers=1, chunk_tokens=40), [(0.0, 100, 1)])
    assert res[0]["ttft_us"] == pytest.approx(14.0 + 14.0 + 12.0) and summ["iterations"] == 3
    assert res[0]["tpot_us"] == 0.0 and res[0]["finish_us"] == res[0]["first_token_us"]


def test_attainment_follows_eq_1_to_3():
    """Two requests on one colocated worker.  r0 = (0, 100, 3) alone would decode at 10.1 per token; r1 = (25, 200, 2)
    arrives while r0 decodes and its prefill rides in r0's second decode iteration: worked by hand --
      t=0..20 prefill r0; 20..30.1 decode r0 (r1 arrives at 25, queued); 30.1..60.2 iteration {prefill r1 (200 tokens),
      decode r0}: 10 + 0.1 * 201 = 30.1 -> r0 finishes at 60.2 (TPOT (60.2 - 20) / 2 = 20.1), r1 first token at 60.2
      (TTFT 35.2); 60.2..70.3 decode r1 (TPOT 10.1).
    With TTFT_SLO = 30 and TPOT_SLO = 15: r0 meets TTFT (20) but not TPOT, r1 meets TPOT but not TTFT -> A = 0;
    with TTFT_SLO = 40: r1 in both sets -> A = 1/2."""
    reqs = [(0.0, 100, 3), (25.0, 200, 2)]
    res, summ = so.simulate(_ocfg(so.COLOCATED, num_workers=1, ttft_slo_us=30.0), reqs)
    assert res[0]["tpot_us"] == pytest.approx(20.1) and res[1]["ttft_us"] == pytest.approx(35.2)
    assert res[1]["tpot_us"] == pytest.approx(10.1) and summ["attainment"] == 0.0
    _, summ = so.simulate(_ocfg(so.COLOCATED, num_workers=1, ttft_slo_us=40.0), reqs)
    assert summ["attainment"] == 0.5


def test_fig7_slack_check():
    """P:141-145, Fig. 7.  Worker 0 prefill worker, worker 1 multiplexing worker.  R0 = (0, 10, 50) goes to the idle
    multiplexing worker (slack +inf), first token at 11, then decodes at 10.1 per token against a TPOT SLO of 15: each
    iteration banks slack.  A 200-token prefill costs 0.1 * 200 = 20 of interference:
      * arriving at t = 12 (R0 has generated nothing yet: slack = 1 * 15 - (12 - 11) = 14 < 20) it is NOT multiplexed,
      * a 100-token one at t = 12 (interference 10 <= 14) is,
      * the 200-token one arriving at t = 45 (R0 generated 3 by 41.3: slack = 4 * 15 - 34 = 26 >= 20) is -- "has
        accumulated enough slack to accommodate a prefill request" -- and R0 still meets its TPOT SLO."""
    cfg = _ocfg(so.MULTIPLEXED)
    res, _ = so.simulate(cfg, [(0.0, 10, 50), (12.0, 200, 2)])
    assert res[0]["multiplexed"] == 1 and res[0]["first_token_us"] == pytest.approx(11.0)
    assert res[1]["multiplexed"] == 0 and res[1]["prefill_worker"] == 0
    res, _ = so.simulate(cfg, [(0.0, 10, 50), (12.0, 100, 2)])
    assert res[1]["multiplexed"] == 1 and res[1]["prefill_worker"] == 1
    res, _ = so.simulate(cfg, [(0.0, 10, 50), (45.0, 200, 2)])
    assert res[1]["multiplexed"] == 1 and res[0]["tpot_us"] <= 15.0


def test_guards_of_the_toggle():
    """no multiplexing when the decode batch alone is near the TPOT SLO, nor above the HBM watermark."""
    near = _ocfg(so.MULTIPLEXED, tpot_slo_us=11.0)           # decode iteration 10.1 >= 0.9 * 11
    res, _ = so.simulate(near, [(0.0, 10, 50), (45.0, 20, 2)])
    assert res[1]["multiplexed"] == 0
    full = _ocfg(so.MULTIPLEXED, kv_capacity_tokens=100)      # 0.9 * 100 = 90 tokens of KV
    res, _ = so.simulate(full, [(0.0, 10, 50), (45.0, 85, 2), (400.0, 95, 2)])
    assert res[1]["multiplexed"] == 0 and res[2]["multiplexed"] == 0   # 10 + 3 resident + 85 > 90; 95 > 90 on an empty worker
    res, _ = so.simulate(full, [(0.0, 10, 50), (45.0, 60, 2)])
    assert res[1]["multiplexed"] == 1


def test_path1_needs_ttft_slack_and_nobody_starves():
    """a prefill worker is competent only if exec + queue < TTFT slack.  A 1000-token prompt needs 110 on a
    prefill worker; with TTFT_SLO = 50 and the multiplexing worker closed by its watermark it waits in the toggle's
    queue until its slack is gone (t = 50), then it is sent anyway."""
    cfg = _ocfg(so.MULTIPLEXED, ttft_slo_us=50.0, kv_capacity_tokens=100)
    res, _ = so.simulate(cfg, [(0.0, 1000, 1)])
    assert res[0]["multiplexed"] == 0 and res[0]["ttft_us"] == pytest.approx(50.0 + 110.0)
    cfg = _ocfg(so.MULTIPLEXED, ttft_slo_us=200.0, kv_capacity_tokens=100)
    res, _ = so.simulate(cfg, [(0.0, 1000, 1)])
    assert res[0]["ttft_us"] == pytest.approx(110.0)


def test_disaggregated_adds_migration_and_keeps_decode_off_prefill_workers():
    """prefill on worker 0, KV migration 0.5 us/token * 100, decode on worker 1 from the first iteration
    that starts after the cache has arrived."""
    cfg = _ocfg(so.DISAGGREGATED, migrate_us_per_token=0.5)
    res, _ = so.simulate(cfg, [(0.0, 100, 3)])
    assert res[0]["prefill_worker"] == 0 and res[0]["decode_worker"] == 1
    assert res[0]["ttft_us"] == pytest.approx(20.0)
    assert res[0]["finish_us"] == pytest.approx(20.0 + 50.0 + 2 * 10.1)
    assert res[0]["tpot_us"] == pytest.approx((50.0 + 2 * 10.1) / 2)   # TPOT contains the migration


def test_step_cost_closed_form_on_the_golden_batches():
    """The oracle's restatement of the step-cost form, and the library's, against values worked by hand from the feature
    counts of tests/golden/step_cost_features.txt (derived there without code) and a model with round coefficients:
    t0 = 5, a = 1e-6 us/FLOP, b = 1e-5 us/B, kappa = 0.5, e_p = 2, e_d = 3, n_sm = 4.
      A (Hq 4, Hkv 2, d 64; q = [130, 1], c = [0, 17]): F = 8737792, B = 277036, N_p = 12 iterations, N_d = 4 units:
        aF = 8.737792 >= bB = 2.77036 -> 5 + 8.737792 + 0.5 * 2.77036 + 2 * 12 / 4 + 3 * 4 / 4 = 24.122972
      B (8/8/128; q = [256], c = [300]): F = 449314816, B = 4374668, N_p = 72, N_d = 0:
        5 + 449.314816 + 0.5 * 43.74668 + 2 * 72 / 4 = 512.188156
      A with a = 1e-8 (the byte term leads): 5 + 2.77036 + 0.5 * 0.08737792 + 6 + 3 = 16.81404896"""
    cm = (5.0, 1e-6, 1e-5, 0.5, 2.0, 3.0, 4.0)
    cases = [((4, 2, 64), [130, 1], [0, 17], cm, 24.122972),
             ((8, 8, 128), [256], [300], cm, 512.188156),
             ((4, 2, 64), [130, 1], [0, 17], (5.0, 1e-8, 1e-5, 0.5, 2.0, 3.0, 4.0), 16.81404896)]
    for (Hq, Hkv, d), q, c, model, want in cases:
        cfg = _ocfg(so.COLOCATED, cm=model, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d)
        assert so.step_cost_us(cfg, q, c) == pytest.approx(want, rel=1e-12)
        got, _ = tb.step_cost(Hq, Hkv, d, 16, q, c, model=tb.CostModel(*model))
        assert got == pytest.approx(want, rel=1e-12)
        # an iteration = layers * step + linear * new tokens + overhead (tropical_sim.h "Worker iteration")
        cfg3 = _ocfg(so.COLOCATED, cm=model, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d, num_layers=3)
        assert so.iter_time_us(cfg3, q, c) == pytest.approx(3 * want + 0.1 * sum(q) + 10.0, rel=1e-12)
    # the critical-path term e_c * N_c (N_c from the golden file: A 4, B 9) with e_c = 0.5: + 2 and + 4.5
    for (Hq, Hkv, d), q, c, want in (((4, 2, 64), [130, 1], [0, 17], 24.122972 + 2.0), ((8, 8, 128), [256], [300], 512.188156 + 4.5)):
        model = cm + (0.5,)
        cfg = _ocfg(so.COLOCATED, cm=model, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d)
        assert so.step_cost_us(cfg, q, c) == pytest.approx(want, rel=1e-12)
        got, _ = tb.step_cost(Hq, Hkv, d, 16, q, c, model=tb.CostModel(*model))
        assert got == pytest.approx(want, rel=1e-12)


def test_least_unfinished_tokens_dispatch_by_hand():
    """P:186 with several non-empty candidates.  Two colocated workers, flat cost (iteration = 10 + 0.1 * tokens).
      t=0  r0 (prompt 100, 50 outputs): both empty, tie -> worker 0.           unfinished: w0 = 100 + 49 = 149
      t=1  r1 (50, 2):   w0 149, w1 0 -> worker 1.                              w1 = 50 + 1 = 51
      t=2  r2 (10, 2):   w0 149, w1 51 -> worker 1 (busier queue, fewer tokens). w1 = 51 + 10 + 1 = 62
      t=3  r3 (200, 30): w0 149, w1 62 -> worker 1.                             w1 = 62 + 200 + 29 = 291
      t=4  r4 (5, 1):    w0 149, w1 291 -> worker 0.
    Worker 1: prefill r1 1..16; then {prefill r2 (10 tokens), decode r1} = 10 + 0.1 * 11 = 11.1 -> r2's first token at
    27.1 (TTFT 25.1), r1 finished at 27.1 (TPOT 11.1)."""
    reqs = [(0.0, 100, 50), (1.0, 50, 2), (2.0, 10, 2), (3.0, 200, 30), (4.0, 5, 1)]
    cfg = _ocfg(so.COLOCATED, num_workers=2)
    res, _ = so.simulate(cfg, reqs)
    assert [r["prefill_worker"] for r in res] == [0, 1, 1, 1, 0]
    assert res[2]["ttft_us"] == pytest.approx(25.1) and res[1]["tpot_us"] == pytest.approx(11.1)
    cres, _ = tb.sim_run(_ccfg(cfg), reqs)
    assert [r.prefill_worker for r in cres] == [0, 1, 1, 1, 0] and cres[2].ttft_us == pytest.approx(25.1)


def test_path1_counts_the_iteration_in_flight_as_queueing_time():
    """P:157 "predicted queuing time in the workers" with a BUSY prefill worker.  Worker 0 prefill worker, worker 1
    multiplexing worker closed by its HBM watermark (capacity 100 tokens).  Flat cost, TTFT SLO 150.
      t=0   r0 (1000, 1): exec 110 + queue 0 < 150 -> worker 0, busy until 110.
      t=10  r1 (500, 1):  exec 60 + queue (110 - 10 = 100, the iteration in flight) = 160 >= slack 150: NOT sent.
      t=110 worker 0 idle: exec 60 + 0 >= slack 150 - 100 = 50: still not sent.
      t=160 = arrival + SLO: slack gone, sent anyway; prefill 160..220 -> TTFT 210.
    (Ignoring the iteration in flight would have sent r1 at t = 10: TTFT 160.)
      r1' (300, 1) instead: exec 40 + 100 = 140 < 150 -> sent at t = 10, runs 110..150 -> TTFT 140."""
    cfg = _ocfg(so.MULTIPLEXED, ttft_slo_us=150.0, kv_capacity_tokens=100)
    for sim in (lambda c, r: [x["ttft_us"] for x in so.simulate(c, r)[0]],
                lambda c, r: [x.ttft_us for x in tb.sim_run(_ccfg(c), r)[0]]):
        assert sim(cfg, [(0.0, 1000, 1), (10.0, 500, 1)]) == pytest.approx([110.0, 210.0])
        assert sim(cfg, [(0.0, 1000, 1), (10.0, 300, 1)]) == pytest.approx([110.0, 140.0])


def test_p90_index_by_hand():
    """P:173 "P90 latency": value at index ceil(0.9 n) - 1 of the sorted list -- the 9th smallest of 10, the 10th of 11.
    Ten requests far apart on one worker: TTFT = 10 + 0.1 * prompt = 11, 12, ..., 20 -> p90 = 19; TPOT = 10.1 each."""
    results = [dict(ttft_us=float(v), tpot_us=float(21 - v), first_token_us=0.0, finish_us=float(v), multiplexed=0)
               for v in (7, 3, 10, 1, 9, 2, 8, 4, 6, 5)]
    summ = so.summarize(_ocfg(so.COLOCATED), results, 0)
    assert summ["ttft_p90_us"] == 9.0 and summ["tpot_p90_us"] == 19.0 and summ["ttft_mean_us"] == pytest.approx(5.5)
    results.append(dict(ttft_us=11.0, tpot_us=9.0, first_token_us=0.0, finish_us=11.0, multiplexed=0))
    assert so.summarize(_ocfg(so.COLOCATED), results, 0)["ttft_p90_us"] == 10.0
    reqs = [(1000.0 * i, 10 * (i + 1), 2) for i in range(10)]
    _, csum = tb.sim_run(_ccfg(_ocfg(so.COLOCATED, num_workers=1)), reqs)
    assert csum.ttft_p90_us == pytest.approx(19.0) and csum.tpot_p90_us == pytest.approx(10.1)
    assert csum.ttft_mean_us == pytest.approx(15.5)


def test_no_starvation_wake_up_fires_despite_rounding():
    """with arrival 2724338.6555860057 and SLO 60.37494846539122 the residual slo - (now - arrival) at the
    wake-up time arrival + slo is +1e-10, not <= 0; the rule must fire on the expression the wake-up was scheduled
    with.  Multiplexing worker closed (capacity 500 < prompt), prefill worker too slow for the SLO: the request is sent
    at arrival + SLO and finishes; nobody is scored as served without being served."""
    a, slo = 2724338.6555860057, 60.37494846539122
    cfg = _ocfg(so.MULTIPLEXED, ttft_slo_us=slo, kv_capacity_tokens=500)
    ores, osum = so.simulate(cfg, [(a, 1000, 3)])
    cres, csum = tb.sim_run(_ccfg(cfg), [(a, 1000, 3)])
    want_first = (a + slo) + 110.0
    assert ores[0]["first_token_us"] == pytest.approx(want_first, rel=1e-12)
    assert cres[0].first_token_us == pytest.approx(want_first, rel=1e-12) and cres[0].finish_us > cres[0].first_token_us
    assert osum["attainment"] == 0.0 and csum.attainment == 0.0      # TTFT = slo + 110 > slo


def test_iteration_cost_worked_by_hand():
    """NEXT-4 (include/tropical.h tropical_iter_cost): golden batch A (q = [130, 1], c = [0, 17]) of a 4/2/64 model with
    TP = 2, so one GPU runs the head shard 2/1/64.  Step features of the shard, by hand from the formulas of
    tests/golden/step_cost_features.txt: F = 8737792 / 2 = 4368896; B = 4*1*64*17 + 2*(4*1*64*131) + 2*(2*2*64*131)
    + 4*11 = 4352 + 67072 + 67072 + 44 = 138540; N_p = 3 iterations x 2 heads = 6; N_d = 2 pages x 1 head = 2.
      step = 5 + 4.368896 + 0.5 * 1.3854 + 2 * 6 / 4 + 3 * 2 / 4 = 14.561596
    Linear layers of d_model 8, d_ffn 16 (gated), per GPU: QKV 8 x 256, O 128 x 8, gate+up 8 x 16, down 8 x 8:
      W = 2048 + 1024 + 128 + 64 = 3264; T = 131; F = 2 * 131 * 3264 = 855168;
      B = 2 * 3264 + 2 * 131 * (264 + 136 + 24 + 16) = 6528 + 115280 = 121808
      linear (g0 7, f 1e-5, w 1e-4, kappa 0.25) = 7 + 12.1808 + 0.25 * 8.55168 = 21.31872
      all-reduce (1.5 us + 1e-3 us/B, two per layer over 2 * 131 * 8 B) = 2 * (1.5 + 2.096) = 7.192
      iteration of 3 layers = 3 * (14.561596 + 21.31872 + 7.192) = 129.216948"""
    cm = (5.0, 1e-6, 1e-5, 0.5, 2.0, 3.0, 4.0)
    lin = (7.0, 1e-5, 1e-4, 0.25, 1.5, 1e-3)
    cfg = _ocfg(so.COLOCATED, cm=cm, num_q_heads=4, num_kv_heads=2, head_dim=64, iter_overhead_us=2.0,
                layer=so.LayerShape(8, 16, 1, 3, 2), linear=so.LinearModel(*lin))
    assert so.iter_cost_us(cfg, [130, 1], [0, 17]) == pytest.approx(129.216948, rel=1e-12)
    assert so.iter_time_us(cfg, [130, 1], [0, 17]) == pytest.approx(131.216948, rel=1e-12)
    got, bd = tb.iter_cost(tb.LayerShape(8, 16, 1, 3, 2), 4, 2, 64, 16, [130, 1], [0, 17], attn=tb.CostModel(*cm),
                           linear=tb.LinearModel(*lin))
    assert got == pytest.approx(129.216948, rel=1e-12)
    assert (bd.gemm_flops, bd.gemm_bytes) == (855168.0, 121808.0)
    assert bd.attn_us == pytest.approx(14.561596) and bd.linear_us == pytest.approx(21.31872)
    assert bd.allreduce_us == pytest.approx(7.192)
    # tp = 1: no all-reduce, whole heads: step = 24.122972 (test above); W doubles except ... by hand:
    # QKV 8 x 512, O 256 x 8, gate+up 8 x 32, down 16 x 8: W = 4096 + 2048 + 256 + 128 = 6528, F = 1710336,
    # B = 13056 + 262 * (520 + 264 + 40 + 24) = 13056 + 222176 = 235232 -> 7 + 23.5232 + 0.25 * 17.10336 = 34.79904
    got1, bd1 = tb.iter_cost(tb.LayerShape(8, 16, 1, 1, 1), 4, 2, 64, 16, [130, 1], [0, 17], attn=tb.CostModel(*cm),
                             linear=tb.LinearModel(*lin))
    assert bd1.allreduce_us == 0.0 and got1 == pytest.approx(24.122972 + 34.79904, rel=1e-12)
    cfg1 = _ocfg(so.COLOCATED, cm=cm, num_q_heads=4, num_kv_heads=2, head_dim=64,
                 layer=so.LayerShape(8, 16, 1, 1, 1), linear=so.LinearModel(*lin))
    assert so.iter_cost_us(cfg1, [130, 1], [0, 17]) == pytest.approx(24.122972 + 34.79904, rel=1e-12)
    with pytest.raises(tb.TropicalError):   # tp must divide the kv heads
        tb.iter_cost(tb.LayerShape(8, 16, 1, 1, 4), 4, 2, 64, 16, [1], [1], attn=tb.CostModel(*cm))


def test_prefill_worker_becomes_multiplexing_worker_when_every_decode_worker_is_above_the_watermark():
    """P:161, first sentence, by hand.  Workers 0, 1 prefill, worker 2 multiplexing; flat cost with 1 us per token and no
    overhead; KV capacity 100 tokens, watermark 0.5 (threshold 50 tokens); no migration time.
      t=0    A (prompt 60, 100 outputs): Path 2 refused (0 + 60 > 50), Path 1 -> worker 0 (exec 60 < SLO), runs 0..60.
      t=60   A's first token; its cache goes to worker 2 (the only multiplexing worker): worker 2 now holds 60 > 50 tokens
             = every multiplexing worker is above the watermark, two prefill workers exist -> the one with the least
             predicted queue (both 0: worker 0) becomes a multiplexing worker.  A decodes on worker 2, 1 us per token.
      t=100  B (prompt 10, 2 outputs): Path 2 candidates {0, 2} by unfinished tokens: worker 0 (0) first: empty, 0 + 10 <=
             50 -> multiplexed on worker 0: prefill 100..110 (TTFT 10), one decode iteration 110..111, stays on worker 0.
    With fixed roles B is refused by worker 2 (100 + 10 > 50) and takes Path 1: worker 0, then migrates to worker 2."""
    kw = dict(num_workers=3, num_prefill_workers=2, kv_capacity_tokens=100, hbm_watermark=0.5, linear_us_per_token=1.0,
              iter_overhead_us=0.0, tpot_slo_us=1e9)
    reqs = [(0.0, 60, 100), (100.0, 10, 2)]
    for sim in (lambda c: so.simulate(c, reqs), lambda c: _as_dicts(tb.sim_run(_ccfg(c), reqs))):
        res, summ = sim(_ocfg(so.MULTIPLEXED, role_transitions=1, delay_threshold=1000, **kw))
        assert (res[0]["prefill_worker"], res[0]["decode_worker"], res[0]["first_token_us"]) == (0, 2, 60.0)
        assert (res[1]["prefill_worker"], res[1]["decode_worker"], res[1]["multiplexed"]) == (0, 0, 1)
        assert res[1]["ttft_us"] == pytest.approx(10.0) and res[1]["finish_us"] == pytest.approx(111.0)
        assert (summ["to_multiplexing"], summ["to_prefill"]) == (1, 0)
        res, summ = sim(_ocfg(so.MULTIPLEXED, **kw))       # fixed roles
        assert (res[1]["prefill_worker"], res[1]["decode_worker"], res[1]["multiplexed"]) == (0, 2, 0)
        assert (summ["to_multiplexing"], summ["to_prefill"]) == (0, 0)


def test_multiplexing_worker_becomes_prefill_worker_when_prefills_keep_being_delayed():
    """P:161, second sentence, by hand.  Worker 0 prefill, workers 1, 2 multiplexing; flat cost, 1 us per token, no
    overhead; TTFT SLO 5 us; capacity 100, watermark 0.5, so 80-token prompts are refused by Path 2 (80 > 50) and by
    Path 1 (80 us > any slack): every request waits for the no-starvation rule at arrival + 5.  delay_threshold = 2.
      t=5  A (arrival 0) delayed -> worker 0, runs 5..85.        delayed = 1
      t=6  B (arrival 1) delayed -> worker 0's queue.             delayed = 2
      t=7  scan: 2 delayed prefills, two multiplexing workers, worker 1 holds no decode state -> worker 1 becomes a
           prefill worker.  C (arrival 2) delayed -> least predicted queue: worker 0 = (85 - 7) + 80, worker 1 = 0 ->
           worker 1, runs 7..87 (TTFT 85).  B runs 85..165 on worker 0.
    With fixed roles C queues behind B on worker 0: 165..245 (TTFT 243)."""
    kw = dict(num_workers=3, num_prefill_workers=1, kv_capacity_tokens=100, hbm_watermark=0.5, linear_us_per_token=1.0,
              iter_overhead_us=0.0, ttft_slo_us=5.0)
    reqs = [(0.0, 80, 1), (1.0, 80, 1), (2.0, 80, 1)]
    for sim in (lambda c: so.simulate(c, reqs), lambda c: _as_dicts(tb.sim_run(_ccfg(c), reqs))):
        res, summ = sim(_ocfg(so.MULTIPLEXED, role_transitions=1, delay_threshold=2, **kw))
        assert [r["prefill_worker"] for r in res] == [0, 0, 1]
        assert [r["first_token_us"] for r in res] == pytest.approx([85.0, 165.0, 87.0])
        assert (summ["to_multiplexing"], summ["to_prefill"]) == (0, 1)
        res, summ = sim(_ocfg(so.MULTIPLEXED, **kw))
        assert [r["prefill_worker"] for r in res] == [0, 0, 0] and res[2]["first_token_us"] == pytest.approx(245.0)


def _as_dicts(out):
    res, summ = out
    fields = ("ttft_us", "tpot_us", "first_token_us", "finish_us", "prefill_worker", "decode_worker", "multiplexed")
    return ([{f: getattr(r, f) for f in fields} for r in res],
            {f: getattr(summ, f) for f, _ in tb.binding.SimSummary._fields_})


def _trace(seed, n, mean_gap_us):
    rng = random.Random(seed)
    t, out = 0.0, []
    for _ in range(n):
        t += rng.expovariate(1.0 / mean_gap_us)
        out.append((t, int(min(16000, max(16, rng.lognormvariate(7.0, 1.1)))), rng.randint(1, 120)))  # long-tail prompts
    return out


@pytest.mark.parametrize("policy", [so.COLOCATED, so.DISAGGREGATED, so.MULTIPLEXED])
def test_conservation_invariants(policy):
    cfg = _ocfg(policy, cm=FIT, num_workers=4, num_prefill_workers=2, chunk_tokens=2048, ttft_slo_us=4e5, tpot_slo_us=3e4,
                kv_capacity_tokens=300000, migrate_us_per_token=0.05, num_layers=8, linear_us_per_token=1.0, iter_overhead_us=30.0)
    reqs = _trace(policy, 80, 40000.0)
    res, summ = so.simulate(cfg, reqs)
    for (a, p, o), r in zip(reqs, res):
        assert r["first_token_us"] > a and r["finish_us"] >= r["first_token_us"] and r["ttft_us"] > 0
        assert (r["tpot_us"] == 0) == (o == 1)
        if policy != so.COLOCATED and o > 1 and not r["multiplexed"]:
            assert r["prefill_worker"] < 2 <= r["decode_worker"]
        if policy == so.COLOCATED:
            assert r["prefill_worker"] == r["decode_worker"]
    assert 0.0 <= summ["attainment"] <= 1.0 and summ["makespan_us"] == max(r["finish_us"] for r in res)
    assert summ["iterations"] >= max(o for _, _, o in reqs)


# ------------------------------------------------------------------------------------------ part 2: C++ vs oracle
@pytest.mark.parametrize("policy", [so.COLOCATED, so.DISAGGREGATED, so.MULTIPLEXED])
@pytest.mark.parametrize("seed,gap,chunk", [(1, 150000.0, 2048), (2, 30000.0, 0), (3, 8000.0, 512)])
def test_cpp_simulator_matches_oracle(policy, seed, gap, chunk):
    o = _ocfg(policy, cm=FIT, num_workers=5, num_prefill_workers=2, chunk_tokens=chunk, ttft_slo_us=3e5, tpot_slo_us=2.5e4,
              kv_capacity_tokens=200000, migrate_us_per_token=0.04, num_layers=6, linear_us_per_token=0.8, iter_overhead_us=25.0)
    reqs = _trace(100 + seed, 70, gap)
    ores, osum = so.simulate(o, reqs)
    cres, csum = tb.sim_run(_ccfg(o), reqs)
    for a, b in zip(cres, ores):
        assert (a.prefill_worker, a.decode_worker, a.multiplexed) == (b["prefill_worker"], b["decode_worker"], b["multiplexed"])
        for f in ("ttft_us", "tpot_us", "first_token_us", "finish_us"):
            assert getattr(a, f) == pytest.approx(b[f], rel=1e-9, abs=1e-9)
    assert csum.iterations == osum["iterations"] and csum.multiplexed_prefills == osum["multiplexed_prefills"]
    for f in ("attainment", "ttft_mean_us", "ttft_p90_us", "tpot_mean_us", "tpot_p90_us", "makespan_us"):
        assert getattr(csum, f) == pytest.approx(osum[f], rel=1e-9)


@pytest.mark.parametrize("seed,gap,thr", [(4, 9000.0, 2), (5, 3000.0, 1), (6, 20000.0, 1)])
def test_cpp_simulator_matches_oracle_with_role_transitions_and_the_iteration_predictor(seed, gap, thr):
    """P:161 transitions + NEXT-4 iteration times (TP = 2 shard of a 64/8/128 model) on seeded long-tail traces: small
    KV capacity so that the watermark rule fires, a tight TTFT SLO so that prefills get delayed."""
    o = _ocfg(so.MULTIPLEXED, cm=FIT, num_workers=6, num_prefill_workers=3, chunk_tokens=1024, ttft_slo_us=5e3,
              tpot_slo_us=2.5e4, kv_capacity_tokens=6000, hbm_watermark=0.6, migrate_us_per_token=0.04, iter_overhead_us=25.0,
              layer=so.LayerShape(1024, 4096, 1, 4, 2), linear=so.LinearModel(20.0, 7e-10, 1.6e-7, 0.3, 8.0, 2e-6),
              role_transitions=1, delay_threshold=thr)
    reqs = _trace(200 + seed, 90, gap)
    ores, osum = so.simulate(o, reqs)
    cres, csum = _as_dicts(tb.sim_run(_ccfg(o), reqs))
    for a, b in zip(cres, ores):
        assert (a["prefill_worker"], a["decode_worker"], a["multiplexed"]) == (b["prefill_worker"], b["decode_worker"], b["multiplexed"])
        for f in ("ttft_us", "tpot_us", "first_token_us", "finish_us"):
            assert a[f] == pytest.approx(b[f], rel=1e-9, abs=1e-9)
    assert (csum["to_multiplexing"], csum["to_prefill"]) == (osum["to_multiplexing"], osum["to_prefill"])
    assert osum["to_multiplexing"] + osum["to_prefill"] > 0      # the traces do exercise the transitions
    assert csum["iterations"] == osum["iterations"]


def test_cpp_simulator_on_the_worked_examples():
    """The hand-worked traces of part 1 through the library as well."""
    res, summ = tb.sim_run(_ccfg(_ocfg(so.COLOCATED, num_workers=1, ttft_slo_us=40.0)), [(0.0, 100, 3), (25.0, 200, 2)])
    assert res[0].tpot_us == pytest.approx(20.1) and res[1].ttft_us == pytest.approx(35.2) and summ.attainment == 0.5
    res, _ = tb.sim_run(_ccfg(_ocfg(so.MULTIPLEXED)), [(0.0, 10, 50), (12.0, 200, 2)])
    assert res[1].multiplexed == 0
    res, _ = tb.sim_run(_ccfg(_ocfg(so.MULTIPLEXED)), [(0.0, 10, 50), (45.0, 200, 2)])
    assert res[1].multiplexed == 1 and res[0].tpot_us <= 15.0


def test_sim_argument_validation():
    good = _ccfg(_ocfg(so.MULTIPLEXED))
    with pytest.raises(tb.TropicalError):
        tb.sim_run(good, [(5.0, 10, 2), (1.0, 10, 2)])           # not sorted by arrival
    with pytest.raises(tb.TropicalError):
        tb.sim_run(good, [(0.0, 0, 2)])                           # empty prompt
    bad = _ccfg(_ocfg(so.MULTIPLEXED, num_prefill_workers=2))     # no multiplexing worker left
    with pytest.raises(tb.TropicalError):
        tb.sim_run(bad, [(0.0, 10, 2)])
    res, summ = tb.sim_run(good, [])
    assert res == [] and summ.iterations == 0


def test_simulate_driver_runs_on_the_builtin_fits(capsys):
    """python -m paper_2606_16264_b200.simulate: the three styles on a synthetic trace with iteration times from
    tropical_iter_cost and the compiled-in B200 fits (TP = 2 shard, role transitions on): runs, and every attainment is a
    fraction."""
    from paper_2606_16264_b200 import simulate
    assert simulate.main(["--requests", "60", "--rates", "8,24", "--tp", "2", "--role-transitions"]) == 0
    lines = [l for l in capsys.readouterr().out.splitlines() if "|" in l and l.lstrip()[0].isdigit()]
    assert len(lines) == 2
    for l in lines:
        cols = [c.split() for c in l.split("|")]
        for att in (cols[1][0], cols[2][0], cols[3][0]):
            assert 0.0 <= float(att) <= 1.0
    assert simulate.migrate_us_per_token(40, 128, 40, 900.0) == pytest.approx(40 * 4 * 40 * 128 / 900e3)   # the link is the slower hop
