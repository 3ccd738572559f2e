"""SLO attainment of the three serving styles of the paper on a synthetic long-tail trace.

    python -m paper_2606_16264_b200.simulate [--requests 400] [--rates 4,8,12,16] [--workers 4] [--prefill-workers 2]

Drives tropical_sim_run (include/tropical_sim.h) with the step-cost coefficients fitted on the B200
(csrc/cost_model_fit.inc) for the 13B-like shape 40/40/128.  The linear layers of an iteration (QKV, O, gated MLP:
everything outside attention + KV append) enter as `overhead + slope * tokens` per layer, least squares on relative
error over the times `python -m paper_2606_16264_b200.gemm_probe` measured with library GEMMs on the B200
(calibration/b200_gemm.csv: ~126 us per layer to stream the weights, ~0.4 us per token per layer at large batches);
a first step towards the full-layer cost of NEXT-4, no norms / RoPE / sampling / communication.  Arrivals are Poisson, prompt lengths lognormal
(median 1500, sigma 1.1, clipped to [32, 32768]: long-tailed like P:87), output lengths uniform in [32, 512]; no record
of the paper's trace is used.  SLOs follow P:173 read as 5x the light-load latency of each phase.
The output is qualitative context for the scheduler, not a reproduction of Fig. 8.
"""
from __future__ import annotations

import argparse
import os
import random
import re

from . import binding as tb

HERE = os.path.dirname(os.path.abspath(__file__))


def builtin_model(Hq: int, Hkv: int, d: int) -> tb.CostModel:
    text = open(os.path.join(HERE, "csrc", "cost_model_fit.inc")).read()
    for m in re.finditer(r"\{(\d+), (\d+), (\d+), \{([^}]*)\}\}", text):
        if (int(m.group(1)), int(m.group(2)), int(m.group(3))) == (Hq, Hkv, d):
            return tb.CostModel(*[float(x) for x in m.group(4).split(",")])
    raise KeyError(f"no fitted coefficients for {Hq}/{Hkv}/{d}")


def linear_layer_fit():
    """(overhead_us, us_per_token) of one layer's GEMMs: weighted least squares (relative error) on b200_gemm.csv."""
    rows = [l.strip().split(",") for l in open(os.path.join(HERE, "calibration", "b200_gemm.csv"))][1:]
    T = [float(r[0]) for r in rows]
    y = [float(r[1]) for r in rows]
    w = [1.0 / v for v in y]
    s0 = sum(wi * wi for wi in w)
    s1 = sum(wi * wi * t for wi, t in zip(w, T))
    s2 = sum(wi * wi * t * t for wi, t in zip(w, T))
    b0 = sum(wi * wi * v for wi, v in zip(w, y))
    b1 = sum(wi * wi * t * v for wi, t, v in zip(w, T, y))
    det = s0 * s2 - s1 * s1
    return (b0 * s2 - b1 * s1) / det, (s0 * b1 - s1 * b0) / det


def make_trace(n: int, rate_per_s: float, seed: int):
    rng = random.Random(seed)
    t, out = 0.0, []
    for _ in range(n):
        t += rng.expovariate(rate_per_s) * 1e6
        out.append((t, int(min(32768, max(32, rng.lognormvariate(7.313, 1.1)))), rng.randint(32, 512)))
    return out


def config(policy: int, workers: int, prefill_workers: int, ttft_slo_us: float, tpot_slo_us: float) -> tb.SimConfig:
    layers = 40
    overhead, slope = linear_layer_fit()
    return tb.SimConfig(policy, workers, prefill_workers, 2048, ttft_slo_us, tpot_slo_us, 0.8, 0.9, 2_000_000, 0.05,
                        40, 40, 128, 16, layers, builtin_model(40, 40, 128), layers * slope, layers * overhead)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--requests", type=int, default=400)
    ap.add_argument("--rates", default="4,8,12,16,20,24", help="request rates (1/s), comma separated")
    ap.add_argument("--workers", type=int, default=4)
    ap.add_argument("--prefill-workers", type=int, default=2)
    ap.add_argument("--seed", type=int, default=0)
    a = ap.parse_args(argv)
    # light-load latency of each phase: one median request alone on a worker (SLO = 5x)
    probe, _ = tb.sim_run(config(tb.SIM_COLOCATED, 1, 1, 1e12, 1e12), [(0.0, 1500, 256)])
    ttft_slo, tpot_slo = 5 * probe[0].ttft_us, 5 * probe[0].tpot_us
    print(f"SLOs: TTFT {ttft_slo / 1e3:.1f} ms, TPOT {tpot_slo / 1e3:.2f} ms; {a.workers} workers "
          f"({a.prefill_workers} prefill workers where the style has them), {a.requests} requests per point")
    print(f"{'rate/s':>7} | {'colocated A':>11} {'p90 TTFT ms':>12} | {'disaggr. A':>10} {'p90 TTFT ms':>12} | "
          f"{'tropical A':>10} {'p90 TTFT ms':>12} {'multiplexed':>11}")
    for rate in [float(x) for x in a.rates.split(",")]:
        trace = make_trace(a.requests, rate, a.seed)
        cols = []
        for pol in (tb.SIM_COLOCATED, tb.SIM_DISAGGREGATED, tb.SIM_MULTIPLEXED):
            _, s = tb.sim_run(config(pol, a.workers, a.prefill_workers, ttft_slo, tpot_slo), trace)
            cols.append(s)
        c, d, m = cols
        print(f"{rate:7.2f} | {c.attainment:11.3f} {c.ttft_p90_us / 1e3:12.1f} | {d.attainment:10.3f} {d.ttft_p90_us / 1e3:12.1f} | "
              f"{m.attainment:10.3f} {m.ttft_p90_us / 1e3:12.1f} {m.multiplexed_prefills:11d}")


if __name__ == "__main__":
    main()
