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
FIT = (35.0, 1.0e-9, 1.15e-7, 0.15, 0.13, 0.057, 148.0)  # a B200-like fit (64/8/128), values rounded by hand


def _ocfg(policy, cm=FLAT, **kw):
    d = dict(policy=policy, num_workers=2, num_prefill_workers=1, chunk_tokens=0, ttft_slo_us=1e9, tpot_slo_us=15.0,
             decode_guard=0.9, hbm_watermark=0.9, kv_capacity_tokens=10**9, migrate_us_per_token=0.0, num_q_heads=64,
             num_kv_heads=8, head_dim=128, page_size=16, num_layers=1, attn=so.CostModel(*cm), linear_us_per_token=0.1,
             iter_overhead_us=10.0)
    d.update(kw)
    return so.Config(**d)


def _ccfg(o: so.Config):
    a = o.attn
    return tb.SimConfig(o.policy, o.num_workers, o.num_prefill_workers, o.chunk_tokens, o.ttft_slo_us, o.tpot_slo_us,
                        o.decode_guard, o.hbm_watermark, o.kv_capacity_tokens, o.migrate_us_per_token, o.num_q_heads,
                        o.num_kv_heads, o.head_dim, o.page_size, o.num_layers,
                        tb.CostModel(a.t0_us, a.a_us_per_flop, a.b_us_per_byte, a.kappa, a.e_prefill_iter_us,
                                     a.e_decode_unit_us, a.n_sm), o.linear_us_per_token, o.iter_overhead_us)


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
