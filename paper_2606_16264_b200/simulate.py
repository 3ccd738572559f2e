"""SLO attainment of the three serving styles of the paper on a synthetic long-tail trace.

    python -m paper_2606_16264_b200.simulate [--requests 400] [--rates 4,8,12,16] [--workers 4] [--prefill-workers 2]
                                             [--tp 2] [--role-transitions]

Drives tropical_sim_run (include/tropical_sim.h) for the 13B-like model of C4 (40/40/128 heads, d_model 5120, FFN 13824,
40 layers).  Iteration times are tropical_iter_cost (NEXT-4): per layer the step-cost fit of the head shard on this GPU
(csrc/cost_model_fit.inc, one coefficient set per kernel variant of the step: prefill-only iterations of prefill workers
run the faster fused variant; --tp 2 = the paper's TP = 2 inside a worker) plus the linear layers from the fit to
library GEMMs measured on the B200 (csrc/linear_model_fit.inc, calibration/b200_gemm.csv).  No norms / RoPE / sampling;
the all-reduce of TP > 1 is entered from NVLink's nominal 900 GB/s per direction and 5 us latency -- NOT measured (one GPU).
KV migration costs layers * (K + V bytes per token) at the rate tropical_kv_migrate reached pool to pool on
one B200 (calibration/b200_migrate.csv, half of read + write) or at --link-gbs for the NVLink hop, whichever is slower.
Arrivals are Poisson, prompt lengths lognormal (median 1500, sigma 1.1, clipped to [32, 32768]: long-tailed like P:87),
output lengths uniform in [32, 512]; no record of the paper's trace is used.  SLOs follow P:173 read as 5x the
light-load latency of each phase.  The output is qualitative context for the scheduler, not a reproduction of Fig. 8.
"""
from __future__ import annotations

import argparse
import os
import random
import re

from . import binding as tb

HERE = os.path.dirname(os.path.abspath(__file__))


def builtin_linear() -> tb.LinearModel:
    text = open(os.path.join(HERE, "csrc", "linear_model_fit.inc")).read()
    m = re.search(r"^\{([^}]*)\}", text, re.M)
    return tb.LinearModel(*[float(x) for x in m.group(1).split(",")])


def migrate_us_per_token(Hkv: int, d: int, layers: int, link_gbs: float) -> float:
    """Time to move one token's K and V of every layer: measured pool-to-pool rate on one GPU, or the link, whichever
    is slower."""
    rows = [l.strip().split(",") for l in open(os.path.join(HERE, "calibration", "b200_migrate.csv")) if l[0] not in "#H"]
    copy_gbs = float(rows[0][4]) / 2 / float(rows[0][5]) / 1e3      # bytes moved one way / us -> GB/s
    return layers * 4.0 * Hkv * d / (min(copy_gbs, link_gbs) * 1e3)


def make_trace(n: int, rate_per_s: float, seed: int):
    rng = random.Random(seed)
    t, out = 0.0, []
    for _ in range(n):
        t += rng.expovariate(rate_per_s) * 1e6
        out.append((t, int(min(32768, max(32, rng.lognormvariate(7.313, 1.1)))), rng.randint(32, 512)))
    return out


MODEL = dict(Hq=40, Hkv=40, d=128, d_model=5120, d_ffn=13824, layers=40)   # 13B-like, the heads of C4


def config(policy: int, workers: int, prefill_workers: int, ttft_slo_us: float, tpot_slo_us: float, tp: int = 1,
           link_gbs: float = 900.0, role_transitions: bool = False) -> tb.SimConfig:
    m = MODEL
    lin = builtin_linear()
    if tp > 1:  # nominal NVLink 5 figures, not measured here
        lin.ar0_us, lin.ar_us_per_byte = 5.0, 1.0 / (link_gbs * 1e3)
    shape = tb.LayerShape(m["d_model"], m["d_ffn"], 1, m["layers"], tp)
    return tb.SimConfig(policy, workers, prefill_workers, 2048, ttft_slo_us, tpot_slo_us, 0.8, 0.9, 2_000_000,
                        migrate_us_per_token(m["Hkv"] // tp, m["d"], m["layers"], link_gbs), m["Hq"], m["Hkv"], m["d"], 16,
                        m["layers"], tb.CostModel(0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0),   # n_sm = 0: the library's built-in fits
                        0.0, 0.0, shape, lin,
                        1 if role_transitions else 0, 8 if role_transitions else 0)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--requests", type=int, default=400)
    ap.add_argument("--rates", default="4,8,12,16,20,24", help="request rates (1/s), comma separated")
    ap.add_argument("--workers", type=int, default=4)
    ap.add_argument("--prefill-workers", type=int, default=2)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--tp", type=int, default=1, help="tensor-parallel degree inside a worker (P:184: 2)")
    ap.add_argument("--link-gbs", type=float, default=900.0, help="NVLink rate per direction for migration / all-reduce")
    ap.add_argument("--role-transitions", action="store_true", help="P:161 role transitions of the multiplexed style")
    a = ap.parse_args(argv)
    kw = dict(tp=a.tp, link_gbs=a.link_gbs)
    # light-load latency of each phase: one median request alone on a worker (SLO = 5x)
    probe, _ = tb.sim_run(config(tb.SIM_COLOCATED, 1, 1, 1e12, 1e12, **kw), [(0.0, 1500, 256)])
    ttft_slo, tpot_slo = 5 * probe[0].ttft_us, 5 * probe[0].tpot_us
    print(f"SLOs: TTFT {ttft_slo / 1e3:.1f} ms, TPOT {tpot_slo / 1e3:.2f} ms; {a.workers} workers "
          f"({a.prefill_workers} prefill workers where the style has them), {a.requests} requests per point")
    print(f"{'rate/s':>7} | {'colocated A':>11} {'p90 TTFT ms':>12} | {'disaggr. A':>10} {'p90 TTFT ms':>12} | "
          f"{'tropical A':>10} {'p90 TTFT ms':>12} {'multiplexed':>11}")
    for rate in [float(x) for x in a.rates.split(",")]:
        trace = make_trace(a.requests, rate, a.seed)
        cols = []
        for pol in (tb.SIM_COLOCATED, tb.SIM_DISAGGREGATED, tb.SIM_MULTIPLEXED):
            _, s = tb.sim_run(config(pol, a.workers, a.prefill_workers, ttft_slo, tpot_slo,
                                     role_transitions=a.role_transitions and pol == tb.SIM_MULTIPLEXED, **kw), trace)
            cols.append(s)
        c, d, m = cols
        print(f"{rate:7.2f} | {c.attainment:11.3f} {c.ttft_p90_us / 1e3:12.1f} | {d.attainment:10.3f} {d.ttft_p90_us / 1e3:12.1f} | "
              f"{m.attainment:10.3f} {m.ttft_p90_us / 1e3:12.1f} {m.multiplexed_prefills:11d}" +
              (f"   role transitions: {m.to_multiplexing} to multiplexing, {m.to_prefill} to prefill" if a.role_transitions else ""))
    return 0


if __name__ == "__main__":
    main()
