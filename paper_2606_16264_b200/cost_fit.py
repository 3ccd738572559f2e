"""Calibration of tropical_step_cost ("offline profiling tools").

    python -m paper_2606_16264_b200.cost_fit measure [--out calibration/b200_grid.csv]   # needs a B200
    python -m paper_2606_16264_b200.cost_fit measure-gemm [--out calibration/b200_gemm.csv]   # needs a B200
    python -m paper_2606_16264_b200.cost_fit sweep-split  [--out split_sweep.csv]             # needs a B200
    python -m paper_2606_16264_b200.cost_fit measure-allreduce [--world 2]                    # needs >= 2 B200s (NCCL)
    python -m paper_2606_16264_b200.cost_fit fit     [--grid calibration/b200_grid.csv]  # CPU only

`measure` times the step -- tropical_mixed_step: KV append + attention in one call -- (CUDA events, inputs resident) over a grid of synthetic batches --
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
LINEAR_INC = os.path.join(HERE, "csrc", "linear_model_fit.inc")
ALLREDUCE_GRID = os.path.join(HERE, "calibration", "b200_allreduce.csv")

SHAPES = [(32, 32, 128), (40, 40, 128), (64, 8, 128),      # BASELINE.json configs[1..4]
          (20, 20, 128), (32, 4, 128)]                      # their TP = 2 head shards (NEXT-4)
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
    # off-grid points (seeds >= 1000, always held out): recipe values drawn between and beyond the grid lines
    rng = np.random.default_rng(7)
    for k in range(24):
        pt = int(rng.choice([0, 0, 384, 768, 1536, 3072, 6144, 12288]))
        pc = int(rng.choice([0, 0, 512, 3072, 6144])) if pt else 0
        nd = int(rng.integers(0, 385)) if pt else int(rng.integers(1, 385))
        cm = int(rng.choice([128, 384, 700, 1500, 2500, 6000])) if nd else 0
        pts.append((pt, pc, nd, cm, 1000 + k))
    return pts


# ------------------------------------------------------------------------------------------ measure (GPU)
def _points_on_device(shapes, pts):
    """Yields (Hq, Hkv, d, point, step) with the point's batch resident on the GPU; step() enqueues append + attention."""
    import torch
    from . import binding as tb

    assert torch.cuda.is_available(), "needs a GPU"
    dev = torch.device("cuda")
    g = torch.Generator(device="cuda")
    g.manual_seed(1234)
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

            def step():   # the product step: one call, append fused or in front (tropical_mixed_step's own choice)
                tb.mixed_step(pool, batch, qd, kn, vn, out=out, workspace=ws)

            yield Hq, Hkv, d, p, step
        del k_pool, v_pool, pool
        torch.cuda.empty_cache()


def _time_us(step, iters):
    import torch
    stream = torch.cuda.current_stream()
    for _ in range(3):
        step()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    torch.cuda.synchronize()
    for a, b in evs:
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    return np.array([a.elapsed_time(b) * 1e3 for a, b in evs])


def measure(out_path: str, iters: int, shapes):
    os.makedirs(os.path.dirname(os.path.abspath(out_path)), exist_ok=True)
    rows = []
    for Hq, Hkv, d, p, step in _points_on_device(shapes, grid_points()):
        us = _time_us(step, iters)
        rows.append([Hq, Hkv, d, p[0], p[1], p[2], p[3], p[4], round(float(np.median(us)), 2), round(float(us.min()), 2)])
    with open(out_path, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(COLUMNS)
        w.writerows(rows)
    print(f"wrote {len(rows)} points to {out_path}")


# Decode split size (pages per split-K unit, csrc/plan.cuh): step time under forced (coarser) splits, the evidence
# behind plan_kernel's rule (profiles/r2c_split_sweep.md).  0 = the kernel's own choice.
SWEEP_SPLITS = [0, 16, 24, 32, 48, 64, 96, 128, 256]


def sweep_split(out_path: str, iters: int, shapes):
    from . import binding as tb
    pts = []
    for nd in (16, 64, 128, 256):
        for cm in (256, 1024, 4096):
            pts.append((0, 0, nd, cm, 100 + nd + cm))
    pts += [(2048, 0, 64, 1024, 71), (2048, 0, 128, 1024, 135), (4096, 0, 256, 1500, 263), (512, 0, 32, 2048, 39)]
    rows = []
    for Hq, Hkv, d, p, step in _points_on_device(shapes, pts):
        us = []
        for split in SWEEP_SPLITS:
            tb.debug_set_split_pages(split)
            us.append(round(float(np.median(_time_us(step, iters))), 1))
        tb.debug_set_split_pages(0)
        rows.append([Hq, Hkv, d, p[0], p[2], p[3]] + us)
        print(rows[-1], flush=True)
    with open(out_path, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["Hq", "Hkv", "d", "prefill_tokens", "n_decode", "ctx_median"] + [f"us_split_{s}" for s in SWEEP_SPLITS])
        w.writerows(rows)
    print(f"wrote {len(rows)} rows to {out_path}")


# ------------------------------------------------------------------------------------------ measure-gemm (GPU)
# NEXT-4: the linear layers of one transformer layer -- QKV, O, (gate +) up, down -- as library GEMMs
# (torch.matmul -> cuBLAS, bf16) on one GPU's shard of a tensor-parallel layer: heads and FFN columns split tp ways.
# Calibration data for tropical_iter_cost's linear term; these GEMMs are not kernels of this repository.
GEMM_GRID = os.path.join(HERE, "calibration", "b200_gemm.csv")
GEMM_LAYERS = [  # (d_model, d_ffn, gated, Hq, Hkv, d, tp)
    (4096, 11008, 1, 32, 32, 128, 1),   # 7B-like (C2 / C3 heads)
    (5120, 13824, 1, 40, 40, 128, 1),   # 13B-like (C4 heads)
    (5120, 13824, 1, 40, 40, 128, 2),
    (8192, 28672, 1, 64, 8, 128, 1),    # 70B-layer-like (C5 heads)
    (8192, 28672, 1, 64, 8, 128, 2),
]
GEMM_TOKENS = [1, 16, 64, 128, 256, 512, 1024, 2048, 4096, 8192]
GEMM_COLUMNS = ["d_model", "d_ffn", "gated", "Hq", "Hkv", "d", "tp", "tokens", "us_median", "us_min"]


def layer_matrices(d_model, d_ffn, gated, Hq, Hkv, d, tp):
    """(K, N) of the four weight matrices one GPU of a tp-way tensor-parallel layer holds."""
    return [(d_model, (Hq + 2 * Hkv) * d // tp), (Hq * d // tp, d_model),
            (d_model, (2 if gated else 1) * d_ffn // tp), (d_ffn // tp, d_model)]


def measure_gemm(out_path: str, iters: int):
    import torch
    assert torch.cuda.is_available(), "measure-gemm needs a GPU"
    dev = torch.device("cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    rows = []
    for layer in GEMM_LAYERS:
        mats = layer_matrices(*layer)
        w = [torch.randn(k, n, device=dev, dtype=torch.bfloat16) for k, n in mats]
        for T in GEMM_TOKENS:
            x = [torch.randn(T, k, device=dev, dtype=torch.bfloat16) for k, _ in mats]

            def run():
                for xi, wi in zip(x, w):
                    torch.matmul(xi, wi)

            for _ in range(3):
                run()
            times = []
            for k in range(iters):
                flush.fill_(k & 1)  # the weights of a real model do not stay in L2 from one layer to the next
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                run()
                e1.record()
                torch.cuda.synchronize()
                times.append(e0.elapsed_time(e1) * 1e3)
            times.sort()
            rows.append(list(layer) + [T, round(times[len(times) // 2], 2), round(times[0], 2)])
        del w
        torch.cuda.empty_cache()
    with open(out_path, "w", newline="") as f:
        wr = csv.writer(f)
        wr.writerow(GEMM_COLUMNS)
        wr.writerows(rows)
    print(f"wrote {len(rows)} points to {out_path}")


# ------------------------------------------------------------------------------------------ fit (CPU)
def read_grid(path: str):
    with open(path) as f:
        rows = [r for r in csv.DictReader(l for l in f if not l.startswith("#"))]
    return [{k: (float(v) if k.startswith("us_") else int(v)) for k, v in r.items()} for r in rows]


def is_held_out(row) -> bool:
    return row["seed"] % 5 == 0 or row["seed"] >= 1000   # every fifth grid point and every off-grid point


def point_features(row):
    """Exact work counts of a grid row through the library's own feature code (tropical_step_cost breakdown)."""
    from . import binding as tb
    q, c = grid_lengths(row["prefill_tokens"], row["prefill_ctx"], row["n_decode"], row["ctx_median"], row["seed"])
    _, bd = tb.step_cost(row["Hq"], row["Hkv"], row["d"], 16, q.tolist(), c.tolist(), require_model=False)
    return bd.flops, bd.bytes, float(bd.prefill_iters), float(bd.decode_units), float(bd.prefill_critical_iters)


def predict(theta, X, n_sm=148.0):
    t0, a, b, kappa, ep, ed, ec = theta
    F, B, Np, Nd, Nc = X.T
    tc, hb = a * F, b * B
    return t0 + np.maximum(tc, hb) + kappa * np.minimum(tc, hb) + ep * Np / n_sm + ed * Nd / n_sm + ec * Nc


# Physical lower bounds of the two roofline coefficients (nominal peaks of the part: 2250 TFLOP/s dense bf16,
# 8 TB/s HBM3e): a fit below them would predict steps faster than the hardware can run.  The measured copy figure of
# MEASURED_PEAKS.json is not used here: it is a read + write mix, and the step kernel has been measured above it on
# pure reads (6.8 TB/s of DRAM reads on C4, profiles/r3b_final.md).
A_MIN_US_PER_FLOP = 1e6 / 2250e12
B_MIN_US_PER_BYTE = 1e6 / 8000e9


FUSED_MIN_TOKENS_PER_REQ = 64   # tropical_mixed_step's choice of kernel variant (csrc/mixed.cu, csrc/step_cost.cpp)


def is_fused_step(row) -> bool:
    q, _ = grid_lengths(row["prefill_tokens"], row["prefill_ctx"], row["n_decode"], row["ctx_median"], row["seed"])
    return int(q.sum()) >= FUSED_MIN_TOKENS_PER_REQ * len(q)


def fit_shape(rows, base=None):
    """Seven coefficients by bounded least squares on relative error.  base = the plain variant's coefficients: then
    only t0, a, e_p and e_c are fitted (a fused-variant step has few decode requests: too few points to identify the
    rest)."""
    from scipy.optimize import least_squares
    X = np.array([point_features(r) for r in rows])
    y = np.array([r["us_median"] for r in rows])
    train = np.array([not is_held_out(r) for r in rows])
    off = np.array([r["seed"] >= 1000 for r in rows])
    scale = np.array([10.0, 1e-9, 1e-7, 1.0, 1.0, 0.01, 1.0])   # parameter magnitudes (us, us/FLOP, us/byte, -, us, us, us)
    lo = np.array([0, A_MIN_US_PER_FLOP / scale[1], B_MIN_US_PER_BYTE / scale[2], 0, 0, 0, 0])
    hi = np.array([20, 50, 50, 1, 50, 500, 50])
    free = np.ones(7, bool)
    if base is not None:
        free = np.array([True, True, False, False, True, False, True])
    fixed = (np.asarray(base) / scale) if base is not None else np.zeros(7)

    def full(xf):
        x = fixed.copy()
        x[free] = xf
        return x * scale

    res_best = None
    for k0 in (0.1, 0.5, 0.9):
        x0 = np.array([1.0, 1.5, 1.6, k0, 0.5, 1.0, 0.1])[free]
        fun = lambda xf: (predict(full(xf), X[train]) - y[train]) / y[train]
        res = least_squares(fun, x0, bounds=(lo[free], hi[free]))
        if res_best is None or res.cost < res_best.cost:
            res_best = res
    theta = full(res_best.x)
    rel = np.abs(predict(theta, X) - y) / y
    stats = dict(n=len(rows), n_train=int(train.sum()), mape_train=float(rel[train].mean()),
                 mape_held=float(rel[~train].mean()), max_held=float(rel[~train].max()), max_all=float(rel.max()),
                 mape_off_grid=float(rel[off].mean()) if off.any() else float("nan"),
                 max_off_grid=float(rel[off].max()) if off.any() else float("nan"))
    return theta, stats


# ---- linear layers (NEXT-4): t = g0 + max(f F, w B) + kappa min(f F, w B), one coefficient set for every layer shape
def read_gemm(path: str):
    with open(path) as f:
        return [{k: (float(v) if k.startswith("us_") else int(v)) for k, v in r.items()}
                for r in csv.DictReader(l for l in f if not l.startswith("#"))]


def gemm_features(r):
    mats = layer_matrices(r["d_model"], r["d_ffn"], r["gated"], r["Hq"], r["Hkv"], r["d"], r["tp"])
    W = float(sum(k * n for k, n in mats))
    T = float(r["tokens"])
    return 2.0 * T * W, 2.0 * W + 2.0 * T * sum(k + n for k, n in mats)


def predict_linear(theta, X):
    g0, f, w, kappa = theta
    tf, tw = f * X[:, 0], w * X[:, 1]
    return g0 + np.maximum(tf, tw) + kappa * np.minimum(tf, tw)


def fit_linear(rows):
    """Every fifth point (in file order) is held out."""
    from scipy.optimize import least_squares
    X = np.array([gemm_features(r) for r in rows])
    y = np.array([r["us_median"] for r in rows])
    train = np.array([i % 5 != 2 for i in range(len(rows))])
    scale = np.array([10.0, 1e-9, 1e-7, 1.0])
    lo = np.array([0, A_MIN_US_PER_FLOP / scale[1], B_MIN_US_PER_BYTE / scale[2], 0])
    hi = np.array([50, 50, 50, 1])
    best = None
    for k0 in (0.1, 0.5, 0.9):
        res = least_squares(lambda x: (predict_linear(x * scale, X[train]) - y[train]) / y[train],
                            np.array([2.0, 0.8, 1.8, k0]), bounds=(lo, hi))
        if best is None or res.cost < best.cost:
            best = res
    theta = best.x * scale
    rel = np.abs(predict_linear(theta, X) - y) / y
    return theta, dict(n=len(rows), mape_train=float(rel[train].mean()), mape_held=float(rel[~train].mean()),
                       max_held=float(rel[~train].max()), max_all=float(rel.max()))


# ------------------------------------------------------------------------------------------ all-reduce (NEXT-4, TP = 2)
ALLREDUCE_COLUMNS = ["world", "backend", "bytes", "us_median", "us_min"]
ALLREDUCE_D_MODEL = (4096, 5120, 8192)   # hidden sizes of the paper's model family; the payload is T x d_model bf16


def allreduce_sizes(max_tokens: int):
    """Payload bytes of the per-layer activations all-reduce of a tensor-parallel worker: T x d_model x 2."""
    sizes, t = set(), 1
    while t <= max_tokens:
        for dm in ALLREDUCE_D_MODEL:
            sizes.add(t * dm * 2)
        t *= 2
    return sorted(sizes)


def measure_allreduce(out_path: str, iters: int, world: int, backend: str, max_tokens: int) -> int:
    """Times sum-all-reduces of bf16 payloads across `world` ranks and writes one CSV row per size (rank 0).  Started
    without a launcher it starts its own ranks (torch.distributed.run, one GPU per rank).  backend "nccl" is the
    measurement (needs `world` GPUs; refused otherwise); "gloo" runs the same plumbing on CPU tensors so that the command
    can be tested without GPUs -- `fit` ignores its rows."""
    import torch
    if "WORLD_SIZE" not in os.environ:
        import socket
        import subprocess
        if backend == "nccl":
            have = torch.cuda.device_count() if torch.cuda.is_available() else 0
            if have < world:
                print(f"measure-allreduce: {world} GPUs needed for the NCCL measurement, {have} visible", file=sys.stderr)
                return 2
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
        return subprocess.call([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
                                "--master-addr", "127.0.0.1", "--master-port", str(port), "-m",
                                "paper_2606_16264_b200.cost_fit", "measure-allreduce", "--out", out_path, "--iters",
                                str(iters), "--world", str(world), "--backend", backend, "--max-tokens", str(max_tokens)])
    import time
    import torch.distributed as dist
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    cuda = backend == "nccl"
    if cuda:
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
    dist.init_process_group(backend)
    dev = "cuda" if cuda else "cpu"
    rows = []
    for nbytes in allreduce_sizes(max_tokens):
        x = torch.ones(nbytes // 2, dtype=torch.bfloat16, device=dev)
        for _ in range(3):
            dist.all_reduce(x)
        per = []
        for _ in range(iters):
            x.fill_(1.0)
            dist.barrier()
            if cuda:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                dist.all_reduce(x)
                e1.record()
                torch.cuda.synchronize()
                us = e0.elapsed_time(e1) * 1e3
            else:
                t0 = time.perf_counter()
                dist.all_reduce(x)
                us = (time.perf_counter() - t0) * 1e6
            t = torch.tensor([us], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)   # the collective is done when its slowest rank is
            per.append(float(t.item()))
        assert float(x[0].item()) == float(world), "all-reduce result"
        rows.append((world, backend, nbytes, float(np.median(per)), float(np.min(per))))
    if rank == 0:
        with open(out_path, "w", newline="") as f:
            w = csv.writer(f)
            w.writerow(ALLREDUCE_COLUMNS)
            for r in rows:
                w.writerow([r[0], r[1], r[2], "%.3f" % r[3], "%.3f" % r[4]])
        print(f"wrote {out_path}: {len(rows)} sizes, world {world}, backend {backend}")
    dist.destroy_process_group()
    return 0


def read_allreduce(path: str):
    """Rows of a measure-allreduce CSV taken with NCCL (the CPU plumbing check's gloo rows never enter a fit)."""
    if not os.path.exists(path):
        return []
    with open(path, newline="") as f:
        return [dict(world=int(r["world"]), bytes=float(r["bytes"]), us=float(r["us_median"]))
                for r in csv.DictReader(f) if r["backend"] == "nccl"]


def fit_allreduce(rows):
    """ar0_us + ar_us_per_byte x bytes, least squares on relative errors, both coefficients >= 0."""
    from scipy.optimize import nnls
    b = np.array([r["bytes"] for r in rows])
    t = np.array([r["us"] for r in rows])
    A = np.stack([np.ones_like(b), b], axis=1) / t[:, None]
    theta, _ = nnls(A, np.ones_like(t))
    rel = np.abs(A @ theta - 1.0)
    return theta, dict(n=len(rows), mape=float(rel.mean()), max=float(rel.max()))


def fit(grid_path: str, write: bool, gemm_path: str = None):
    rows = read_grid(grid_path)
    shapes = sorted({(r["Hq"], r["Hkv"], r["d"]) for r in rows})
    lines = ["// Generated by `python -m paper_2606_16264_b200.cost_fit fit` from calibration/b200_grid.csv.",
             "// {Hq, Hkv, d, fused, {t0_us, a_us_per_flop, b_us_per_byte, kappa, e_prefill_iter_us, e_decode_unit_us, n_sm, "
             "e_prefill_crit_us}}",
             "// fused = 1: steps tropical_mixed_step runs through its fused kernel variant (>= 64 new tokens per request).",
             "// a >= 1 / (2250 TFLOP/s) and b >= 1 / (8 TB/s) are enforced by the fit (nominal peaks of the part)."]
    for s in shapes:
        of_shape = [r for r in rows if (r["Hq"], r["Hkv"], r["d"]) == s]
        plain = [r for r in of_shape if not is_fused_step(r)]
        fused = [r for r in of_shape if is_fused_step(r)]
        theta, st = fit_shape(plain)
        theta_f, st_f = fit_shape(fused, base=theta)
        for tag, th, stt in ((0, theta, st), (1, theta_f, st_f)):
            print(f"shape {s} fused={tag}: theta={['%.4g' % t for t in th]} {stt}")
            lines.append("{%d, %d, %d, %d, {%.6g, %.6g, %.6g, %.6g, %.6g, %.6g, 148, %.6g}},  // %d points; held-out MAPE "
                         "%.1f %%, max over all %.1f %%; off-grid MAPE %.1f %%, max %.1f %%"
                         % (*s, tag, *th[:6], th[6], stt["n"], 100 * stt["mape_held"], 100 * stt["max_all"],
                            100 * stt["mape_off_grid"], 100 * stt["max_off_grid"]))
    gemm_path = gemm_path or GEMM_GRID
    theta_l, st_l = fit_linear(read_gemm(gemm_path))
    print(f"linear layers: theta={['%.4g' % t for t in theta_l]} {st_l}")
    lin = ["// Generated by `python -m paper_2606_16264_b200.cost_fit fit` from calibration/b200_gemm.csv.",
           "// {g0_us, f_us_per_flop, w_us_per_byte, kappa, ar0_us, ar_us_per_byte}; held-out MAPE %.1f %%, max %.1f %%;"
           % (100 * st_l["mape_held"], 100 * st_l["max_held"]),
           ]
    ar_rows = read_allreduce(ALLREDUCE_GRID)
    if ar_rows:
        theta_a, st_a = fit_allreduce(ar_rows)
        print(f"all-reduce: theta={['%.4g' % t for t in theta_a]} {st_a}")
        lin.append("// all-reduce coefficients from calibration/b200_allreduce.csv (world %d, NCCL): MAPE %.1f %%, max %.1f %%."
                   % (ar_rows[0]["world"], 100 * st_a["mape"], 100 * st_a["max"]))
        lin.append("{%.6g, %.6g, %.6g, %.6g, %.6g, %.6g}" % (*theta_l, *theta_a))
    else:
        lin.append("// all-reduce coefficients 0: not measurable on one GPU (DESIGN.md section 7); `cost_fit measure-allreduce`")
        lin.append("// on a box with two GPUs writes calibration/b200_allreduce.csv, and the next `fit` fills them in.")
        lin.append("{%.6g, %.6g, %.6g, %.6g, 0, 0}" % tuple(theta_l))
    if write:
        with open(FIT_INC, "w") as f:
            f.write("\n".join(lines) + "\n")
        with open(LINEAR_INC, "w") as f:
            f.write("\n".join(lin) + "\n")
        print("wrote", FIT_INC, "and", LINEAR_INC)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    sub = ap.add_subparsers(dest="cmd", required=True)
    m = sub.add_parser("measure")
    m.add_argument("--out", default=DEFAULT_GRID)
    m.add_argument("--iters", type=int, default=15)
    m.add_argument("--shapes", default="all", help="'all' or e.g. 64/8/128")
    sw = sub.add_parser("sweep-split")
    sw.add_argument("--out", default="split_sweep.csv")
    sw.add_argument("--iters", type=int, default=20)
    sw.add_argument("--shapes", default="all")
    mg = sub.add_parser("measure-gemm")
    mg.add_argument("--out", default=GEMM_GRID)
    mg.add_argument("--iters", type=int, default=20)
    ma = sub.add_parser("measure-allreduce")
    ma.add_argument("--out", default=ALLREDUCE_GRID)
    ma.add_argument("--iters", type=int, default=20)
    ma.add_argument("--world", type=int, default=2, help="ranks = GPUs (the paper's workers run TP = 2, P:184)")
    ma.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="gloo: CPU plumbing check, ignored by fit")
    ma.add_argument("--max-tokens", type=int, default=8192)
    f = sub.add_parser("fit")
    f.add_argument("--grid", default=DEFAULT_GRID)
    f.add_argument("--no-write", action="store_true")
    a = ap.parse_args(argv)
    if a.cmd == "measure":
        shapes = SHAPES if a.shapes == "all" else [tuple(int(x) for x in a.shapes.split("/"))]
        measure(a.out, a.iters, shapes)
    elif a.cmd == "sweep-split":
        shapes = SHAPES[:3] if a.shapes == "all" else [tuple(int(x) for x in a.shapes.split("/"))]
        sweep_split(a.out, a.iters, shapes)
    elif a.cmd == "measure-gemm":
        measure_gemm(a.out, a.iters)
    elif a.cmd == "measure-allreduce":
        return measure_allreduce(a.out, a.iters, a.world, a.backend, a.max_tokens)
    else:
        fit(a.grid, not a.no_write)


if __name__ == "__main__":
    sys.exit(main())
