"""Calibration of tropical_step_cost ("offline profiling tools").

    python -m paper_2606_16264_b200.cost_fit measure [--out calibration/b200_grid.csv]   # needs a B200
    python -m paper_2606_16264_b200.cost_fit fit     [--grid calibration/b200_grid.csv]  # CPU only

`measure` times append + attention (CUDA events, inputs resident) over a grid of synthetic batches --
prefill tokens x decode requests x decode-context median (lognormal, sigma 0.9), plus chunk-on-context points
(PAPER.md:159 chunked prefill: later chunks see more prior context) -- for each head configuration and writes
one CSV row per point.  `fit` regenerates every point's lengths from its recipe columns, fits the six
coefficients of the closed form in include/tropical.h per head configuration on 80 % of the points and
reports the error on the held-out 20 %; it rewrites csrc/cost_model_fit.inc, which step_cost.cpp compiles in.
No attention arithmetic here: lengths, timing and least squares only.
"""
from __future__ import annotations

import argparse
import csv
import math
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
DEFAULT_GRID = os.path.join(HERE, "calibration", "b200_grid.csv")
FIT_INC = os.path.join(HERE, "csrc", "cost_model_fit.inc")

SHAPES = [(32, 32, 128), (40, 40, 128), (64, 8, 128)]      # BASELINE.json configs[1..4]
PREFILL_TOKENS = [0, 256, 1024, 2048, 4096, 8192]
DECODE_REQS = [0, 16, 64, 128, 256]
CTX_MEDIANS = [256, 1024, 4096]
CHUNK_CTX = [2048, 4096, 8192]                              # prior context of a 2048-token chunk (NEXT-2 sweep)
COLUMNS = ["Hq", "Hkv", "d", "prefill_tokens", "prefill_ctx", "n_decode", "ctx_median", "seed", "us_median", "us_min"]


def grid_lengths(prefill_tokens: int, prefill_ctx: int, n_decode: int, ctx_median: int, seed: int):
    """(q_lens, ctx_lens) of one grid point; prefill split into chunks of <= 4096 tokens, first in the batch."""
    rng = np.random.default_rng(seed)
    q, c = [], []
    left = prefill_tokens
    while left > 0:
        n = min(4096, left)
        q.append(n)
        c.append(prefill_ctx)
        left -= n
    if n_decode:
        z = rng.standard_normal(n_decode)
        cd = np.clip(np.rint(np.exp(math.log(ctx_median) + 0.9 * z)), 64, 8192).astype(np.int64)
        q += [1] * n_decode
        c += cd.tolist()
    return np.asarray(q, np.int32), np.asarray(c, np.int32)


def grid_points():
    pts, seed = [], 100
    for pt in PREFILL_TOKENS:
        for nd in DECODE_REQS:
            if pt == 0 and nd == 0:
                continue
            for cm in (CTX_MEDIANS if nd else [0]):
                pts.append((pt, 0, nd, cm, seed))
                seed += 1
    for pc in CHUNK_CTX:
        for nd in (0, 128):
            pts.append((2048, pc, nd, 1024 if nd else 0, seed))
            seed += 1
    return pts


# ------------------------------------------------------------------------------------------ measure (GPU)
def measure(out_path: str, iters: int, shapes):
    import torch
    from . import binding as tb

    assert torch.cuda.is_available(), "measure needs a GPU"
    dev = torch.device("cuda")
    g = torch.Generator(device="cuda")
    g.manual_seed(1234)
    os.makedirs(os.path.dirname(os.path.abspath(out_path)), exist_ok=True)
    rows = []
    pts = grid_points()
    for Hq, Hkv, d in shapes:
        need = [int(((q.astype(np.int64) + c + 15) // 16).sum()) for q, c in (grid_lengths(*p) for p in pts)]
        num_pages = 64 * math.ceil(1.1 * max(need) / 64)
        block = torch.randn((1024, Hkv, 16, d), generator=g, device=dev).to(torch.bfloat16).view(torch.int16)
        k_pool = block.repeat((num_pages + 1023) // 1024, 1, 1, 1)[:num_pages].contiguous()
        v_pool = k_pool.roll(7, 0).contiguous()
        pool = tb.KVPool(k_pool, v_pool, Hq)
        for p in pts:
            q_lens, ctx_lens = grid_lengths(*p)
            n = len(q_lens)
            L = q_lens.astype(np.int64) + ctx_lens
            pages = (L + 15) // 16
            perm = np.random.default_rng(p[4]).permutation(num_pages)
            table = np.full((n, int(pages.max())), -1, np.int32)
            used = 0
            for i in range(n):
                table[i, :pages[i]] = perm[used:used + pages[i]]
                used += int(pages[i])
            batch = tb.Batch.from_host(q_lens.tolist(), ctx_lens.tolist(), table)
            T = int(q_lens.sum())
            rnd = lambda h: torch.randn((T, h, d), generator=g, device=dev).to(torch.bfloat16).view(torch.int16)
            qd, kn, vn = rnd(Hq), rnd(Hkv), rnd(Hkv)
            out = torch.empty_like(qd)
            ws = torch.empty(tb.workspace_bytes(pool, n, T, int(L.max())) + 256, dtype=torch.uint8, device=dev)
            stream = torch.cuda.current_stream()

            def step():
                tb.kv_append(pool, batch, kn, vn)
                tb.mixed_attention(pool, batch, qd, out=out, workspace=ws)

            for _ in range(3):
                step()
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
            torch.cuda.synchronize()
            for a, b in evs:
                a.record(stream)
                step()
                b.record(stream)
            torch.cuda.synchronize()
            us = np.array([a.elapsed_time(b) * 1e3 for a, b in evs])
            rows.append([Hq, Hkv, d, p[0], p[1], p[2], p[3], p[4], round(float(np.median(us)), 2), round(float(us.min()), 2)])
        del k_pool, v_pool, pool
        torch.cuda.empty_cache()
    with open(out_path, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(COLUMNS)
        w.writerows(rows)
    print(f"wrote {len(rows)} points to {out_path}")


# ------------------------------------------------------------------------------------------ fit (CPU)
def read_grid(path: str):
    with open(path) as f:
        rows = [r for r in csv.DictReader(l for l in f if not l.startswith("#"))]
    return [{k: (float(v) if k.startswith("us_") else int(v)) for k, v in r.items()} for r in rows]


def is_held_out(row) -> bool:
    return row["seed"] % 5 == 0


def point_features(row):
    """Exact work counts of a grid row through the library's own feature code (tropical_step_cost breakdown)."""
    from . import binding as tb
    q, c = grid_lengths(row["prefill_tokens"], row["prefill_ctx"], row["n_decode"], row["ctx_median"], row["seed"])
    _, bd = tb.step_cost(row["Hq"], row["Hkv"], row["d"], 16, q.tolist(), c.tolist(), require_model=False)
    return bd.flops, bd.bytes, float(bd.prefill_iters), float(bd.decode_units)


def predict(theta, X, n_sm=148.0):
    t0, a, b, kappa, ep, ed = theta
    F, B, Np, Nd = X.T
    tc, hb = a * F, b * B
    return t0 + np.maximum(tc, hb) + kappa * np.minimum(tc, hb) + ep * Np / n_sm + ed * Nd / n_sm


def fit_shape(rows):
    from scipy.optimize import least_squares
    X = np.array([point_features(r) for r in rows])
    y = np.array([r["us_median"] for r in rows])
    train = np.array([not is_held_out(r) for r in rows])
    scale = np.array([10.0, 1e-9, 1e-7, 1.0, 1.0, 0.01])   # parameter magnitudes (us, us/FLOP, us/byte, -, us, us)
    res_best = None
    for k0 in (0.1, 0.5, 0.9):
        x0 = np.array([1.0, 1.5, 1.6, k0, 0.5, 1.0])
        fun = lambda x: (predict(x * scale, X[train]) - y[train]) / y[train]
        res = least_squares(fun, x0, bounds=(np.zeros(6), np.array([20, 50, 50, 1, 50, 500])))
        if res_best is None or res.cost < res_best.cost:
            res_best = res
    theta = res_best.x * scale
    rel = np.abs(predict(theta, X) - y) / y
    stats = dict(n=len(rows), n_train=int(train.sum()), mape_train=float(rel[train].mean()),
                 mape_held=float(rel[~train].mean()), max_held=float(rel[~train].max()), max_all=float(rel.max()))
    return theta, stats


def fit(grid_path: str, write: bool):
    rows = read_grid(grid_path)
    shapes = sorted({(r["Hq"], r["Hkv"], r["d"]) for r in rows})
    lines = ["// Generated by `python -m paper_2606_16264_b200.cost_fit fit` from calibration/b200_grid.csv.",
             "// {Hq, Hkv, d, {t0_us, a_us_per_flop, b_us_per_byte, kappa, e_prefill_iter_us, e_decode_unit_us, n_sm}}"]
    for s in shapes:
        theta, st = fit_shape([r for r in rows if (r["Hq"], r["Hkv"], r["d"]) == s])
        print(f"shape {s}: theta={['%.4g' % t for t in theta]} {st}")
        lines.append("{%d, %d, %d, {%.6g, %.6g, %.6g, %.6g, %.6g, %.6g, 148}},  // held-out MAPE %.1f %%, max %.1f %%"
                     % (*s, *theta, 100 * st["mape_held"], 100 * st["max_held"]))
    if write:
        with open(FIT_INC, "w") as f:
            f.write("\n".join(lines) + "\n")
        print("wrote", FIT_INC)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    sub = ap.add_subparsers(dest="cmd", required=True)
    m = sub.add_parser("measure")
    m.add_argument("--out", default=DEFAULT_GRID)
    m.add_argument("--iters", type=int, default=15)
    m.add_argument("--shapes", default="all", help="'all' or e.g. 64/8/128")
    f = sub.add_parser("fit")
    f.add_argument("--grid", default=DEFAULT_GRID)
    f.add_argument("--no-write", action="store_true")
    a = ap.parse_args(argv)
    if a.cmd == "measure":
        shapes = SHAPES if a.shapes == "all" else [tuple(int(x) for x in a.shapes.split("/"))]
        measure(a.out, a.iters, shapes)
    else:
        fit(a.grid, not a.no_write)


if __name__ == "__main__":
    sys.exit(main())
