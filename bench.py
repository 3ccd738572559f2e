#!/usr/bin/env python
"""bench.py -- one multiplexed-iteration step (KV append + mixed prefill/decode attention) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C5] [--impl ours|reference]

Prints ONE JSON line (contract in the task prompt).  metric = BASELINE.json's "mixed prefill+decode
attention step us"; `value` = device-timed us per step with inputs resident in HBM; `e2e` = the same
step through tropical_step_host with pinned HOST buffers (H2D/D2H inside the timed region);
`roofline` = the attention kernel against the measured HBM peak; `cpu_baseline` = the fp64 oracle
timed on this box's host cores on a bounded sample of the same workload.

N > 1 (torchrun): the path shards by request with no collective; each rank
runs its own replica of the workload (weak scaling), timing = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "mixed prefill+decode attention step time"
UNIT = "us"


# ----------------------------------------------------------------------------- roofline arithmetic
def step_counts(s_or_lengths):
    """FLOPs / algorithmic bytes of a step; attention-kernel bytes separately."""
    Hq, Hkv, d, P, q, c = s_or_lengths
    q = q.astype(np.float64)
    c = c.astype(np.float64)
    T = q.sum()
    L = q + c
    pages = np.ceil(L[q > 0] / P).sum()
    flops = 4.0 * d * Hq * (q * c + q * (q + 1) / 2).sum()
    step_bytes = 4.0 * Hkv * d * c.sum() + 2 * (4.0 * Hkv * d * T) + 2 * (2.0 * Hq * d * T) + 4.0 * pages
    attn_bytes = 4.0 * Hkv * d * L[q > 0].sum() + 2 * (2.0 * Hq * d * T) + 4.0 * pages
    return dict(flops=flops, step_bytes=step_bytes, attn_bytes=attn_bytes, new_tokens=T)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


def ncu_traffic(config: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of the step kernel, one launch, from the committed ncu capture
    of this config (profiles/ncu_traffic.csv; the .md beside it names the command); None when there is none."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        f = line.strip().split(",")
        if f and f[0] == config:
            return float(f[1])
    return None


# ----------------------------------------------------------------------------- clocks sampler
class ClockSampler(threading.Thread):
    def __init__(self, index: int, period_s: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.stop_flag = index, period_s, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------- oracle leg (CPU)
def oracle_sample_us(s: synth.StepInputs, budget_rows_flops: float = 4e11, seed: int = 0):
    """Time the fp64 oracle on a seeded random sample of rows of this workload and extrapolate to one
    full step by FLOP ratio.  Returns (us_per_step_extrapolated, description, cores, sample_seconds)."""
    import oracle
    kp, vp = s.copy_pools()
    t0 = time.perf_counter()
    oracle.kv_append(kp, vp, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    t_append = time.perf_counter() - t0
    rng = np.random.default_rng(seed)
    rows_all = [(i, t) for i in range(s.num_reqs) for t in range(int(s.q_lens[i]))]
    order = rng.permutation(len(rows_all))
    per_row = lambda i, t: 4.0 * s.head_dim * s.num_q_heads * (int(s.ctx_lens[i]) + t + 1)
    total = sum(per_row(i, t) for i, t in rows_all)
    rows, acc = [], 0.0
    for k in order:
        rows.append(rows_all[k])
        acc += per_row(*rows_all[k])
        if acc >= budget_rows_flops:
            break
    t0 = time.perf_counter()
    oracle.attention_rows(kp, vp, s.q, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, rows)
    dt = time.perf_counter() - t0
    us = (dt * total / acc + t_append) * 1e6
    desc = (f"oracle.attention_rows on {len(rows)} of {len(rows_all)} seeded-random (request,token) rows "
            f"({acc / total:.3%} of the step's FLOPs, {dt:.2f} s), extrapolated by FLOP ratio; + full oracle append")
    return us, desc, oracle.num_threads(), dt


# ----------------------------------------------------------------------------- multi-rank plumbing
def max_over_ranks(value: float, world: int, device) -> float:
    """Slowest rank's figure (the step is as slow as its slowest replica); a no-op for one rank."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tokens_per_s(new_tokens_per_replica: float, world: int, us_per_step: float) -> float:
    """Aggregate over all replicas (weak scaling: every rank runs its own copy of the workload)."""
    return new_tokens_per_replica * world / (us_per_step * 1e-6)


# ----------------------------------------------------------------------------- main legs
def make_workload(name: str, rank: int):
    t0 = time.perf_counter()
    if rank == 0:
        s = synth.make_config(name, poison=False, values="tiled")
    else:  # replica with the same lengths, different page placement / values
        seed, Hq, Hkv, d, P, q, c, _ = synth.config_lengths(name)
        s = synth.make_step(np.random.default_rng(1000 + rank), Hq, Hkv, d, P, q, c, poison=False, values="tiled",
                            name=name, seed=seed)
    return s, time.perf_counter() - t0


def run_ours(args, rank, world):
    import torch
    import torch.distributed as dist
    import paper_2606_16264_b200 as tb
    from paper_2606_16264_b200.harness import DeviceStep

    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    s, gen_s = make_workload(args.config, rank)
    cnt = step_counts((s.num_q_heads, s.num_kv_heads, s.head_dim, s.page_size, s.q_lens, s.ctx_lens))
    peaks = load_peaks()
    dev = DeviceStep(s)
    stream = torch.cuda.current_stream()

    def one_step(ev=None):
        tb.kv_append(dev.pool, dev.batch, dev.k_new, dev.v_new)
        n = tb.last_launch_count()
        if ev is not None:
            ev[0].record(stream)
        tb.mixed_attention(dev.pool, dev.batch, dev.q, out=dev.out, workspace=dev.workspace)
        n += tb.last_launch_count()
        if ev is not None:
            ev[1].record(stream)
        return n

    for _ in range(max(args.warmup, 3)):
        launches_per_step = one_step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    # A step whose working set fits the 126 MB L2 is timed cold: a 512 MB buffer is rewritten between timed steps
    # (untimed) and the per-step event times are summed.  The big configs (> 0.5 GB per step) need no flush.
    flush = cnt["step_bytes"] < 5e8
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda") if flush else None
    sampler = ClockSampler(local)
    sampler.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    st_evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for k in range(args.steps):  # the timed region: exactly K steps, nothing but the two library calls per step
        if flush:
            flush_buf.fill_(k & 0xff)
            st_evs[k][0].record(stream)
        one_step()
        if flush:
            st_evs[k][1].record(stream)
    e1.record(stream)
    torch.cuda.synchronize()
    total_ms = sum(a.elapsed_time(b) for a, b in st_evs) if flush else e0.elapsed_time(e1)
    # second pass, same steps: an event between the append and the attention call isolates the attention launches
    # for the per-kernel roofline (kept out of the timed region: the event breaks the plan kernel's overlap with
    # the append)
    n_k = min(args.steps, 50)
    for k in range(n_k):
        if flush:
            flush_buf.fill_(k & 0xff)
        one_step(evs[k])
    torch.cuda.synchronize()
    attn_ms = sum(a.elapsed_time(b) for a, b in evs[:n_k]) / n_k
    if total_ms < 400:  # keep the GPU busy long enough for the clock sampler to see it under load
        t_end = time.perf_counter() + 0.4
        while time.perf_counter() < t_end:
            one_step()
        torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    roles = tb.debug_read_profile(dev.workspace)
    total_ms = max_over_ranks(total_ms, world, "cuda")
    ms_per_step = total_ms / args.steps
    us = ms_per_step * 1e3

    # ---- e2e through tropical_step_host (pinned host buffers, H2D + D2H inside the timed region)
    pin = lambda a: torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).pin_memory()
    h = dict(ql=pin(s.q_lens), cl=pin(s.ctx_lens), qo=pin(s.q_offsets), pt=pin(s.page_table), q=pin(s.q),
             k=pin(s.k_new), v=pin(s.v_new))
    h_out = torch.zeros(s.q.shape, dtype=torch.int16).pin_memory()
    staging = torch.empty(tb.step_host_staging_bytes(dev.pool, s.num_reqs, s.total_q, s.page_table_stride) + 256,
                          dtype=torch.uint8, device="cuda")
    host_step = lambda: tb.step_host(dev.pool, h["ql"], h["cl"], h["qo"], h["pt"], s.max_kv_len, h["q"], h["k"],
                                     h["v"], h_out, staging, dev.workspace)
    for _ in range(3):
        host_step()
    torch.cuda.synchronize()
    e2e_steps = max(3, min(args.steps, 50))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        host_step()
    e2e_us = (time.perf_counter() - t0) / e2e_steps * 1e6
    e2e_us = max_over_ranks(e2e_us, world, "cuda")
    h2d = sum(int(h[k].numel() * h[k].element_size()) for k in h)
    d2h = int(h_out.numel() * 2)

    if rank != 0:
        return
    t_bytes_us = cnt["step_bytes"] / (peaks["hbm_gbs"] * 1e3)
    t_flops_us = cnt["flops"] / (peaks["bf16_tflops_sustained"] * 1e6)
    t_roof = max(t_bytes_us, t_flops_us)
    attn_us = attn_ms * 1e3
    achieved = cnt["attn_bytes"] / (attn_us * 1e3)  # GB/s
    if args.no_cpu:
        cpu_us, cpu_desc, cores = float("nan"), "skipped (--no-cpu)", 0
    else:
        cpu_us, cpu_desc, cores, _ = oracle_sample_us(s)
    line = {
        "metric": METRIC, "value": round(us, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": round(ms_per_step, 5), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": f"{args.config} ({describe(args.config)})", "replicas": world,
                   "l2": "step touches %.2f GB >> 126 MB L2, no flush needed" % (cnt["step_bytes"] / 1e9)
                   if not flush else "L2 flushed (512 MB rewritten, untimed) between timed steps; per-step event times summed",
                   "new_tokens_per_step": int(cnt["new_tokens"])},
        "tokens_per_s": round(whole_job_tokens_per_s(cnt["new_tokens"], world, us), 1),
        "step_roofline": {"t_bytes_us": round(t_bytes_us, 2), "t_flops_us": round(t_flops_us, 2),
                          "t_roof_us": round(t_roof, 2), "frac": round(t_roof / us, 4),
                          "achieved_gbs": round(cnt["step_bytes"] / (us * 1e3), 1),
                          "achieved_tflops": round(cnt["flops"] / (us * 1e6), 1),
                          "peaks": peaks},
        "roofline": {"bound": "hbm", "kernel": "launches of tropical_mixed_attention: plan + persistent step kernel (>= 95 % of it)",
                     "achieved": round(achieved, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
                     "frac": round(achieved / peaks["hbm_gbs"], 4), "traffic": ncu_traffic(args.config),
                     "kernel_us": round(attn_us, 2), "algorithmic_bytes": cnt["attn_bytes"], "of": peaks["source"]},
        "cpu_baseline": {"value": round(cpu_us, 1), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": cpu_desc},
        "e2e": {"value": round(e2e_us, 2), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(launches_per_step) * args.steps,
        "clocks": sampler.summary(),
        "gen_seconds": round(gen_s, 1),
        "role_finish_us": {k: round(v / 1e3, 1) for k, v in roles.items()} if roles else None,
    }
    print(json.dumps(line))


def describe(name):
    return {"C1": "tiny mixed 4/4/64", "C2": "decode-only 32/32/128 x64", "C3": "prefill-only 32/32/128 x4",
            "C4": "mixed 13B-like 40/40/128: 2048 chunk + 128 decodes",
            "C5": "mixed GQA 64/8/128: 4096+1024 chunks + 256 decodes"}[name]


def run_reference(args, rank, world):
    """The oracle as it stands, on host cores; each 'step' is a bounded sample of the workload sized so
    that the whole --steps K --warmup W run ends within a few minutes."""
    if rank != 0:
        return
    s, _ = make_workload(args.config, 0)
    _, _, cores, dt0 = oracle_sample_us(s, budget_rows_flops=2e8, seed=12345)  # calibrate rows/s
    per_step_s = min(10.0, max(0.05, 90.0 / max(1, args.steps + args.warmup)))
    budget = max(2e7, 2e8 * per_step_s / max(dt0, 1e-3))
    vals, desc = [], ""
    for k in range(args.warmup + args.steps):
        us, desc, cores, _ = oracle_sample_us(s, budget_rows_flops=budget, seed=k)
        if k >= args.warmup:
            vals.append(us)
    us = float(np.mean(vals)) if vals else float("nan")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": round(us, 1), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(us / 1e3, 3), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.config} ({describe(args.config)})"},
        "cpu_baseline": {"value": round(us, 1), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": round(us, 1), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default="C5", choices=synth.CONFIG_NAMES)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world)


if __name__ == "__main__":
    main()
