#!/usr/bin/env python
"""bench.py -- one multiplexed-iteration step (KV append + mixed prefill/decode attention) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C5|C1..C4|MIG] [--impl ours|reference]

Prints ONE JSON line (contract in the task prompt).  metric = BASELINE.json's "mixed prefill+decode attention step
us"; `value` = device-timed us per step over EXACTLY K back-to-back steps with inputs resident in HBM; `e2e` = the
same step through tropical_step_host with pinned HOST buffers (H2D/D2H inside the timed region); `roofline` = the
attention launches against the measured HBM peak; `cpu_baseline` = the fp64 oracle timed on this box's host cores.

Beyond the contract the line carries: `us_per_step` (median / min / max of per-step event times from a second,
instrumented pass over the same steps), `sustained` (the same step in a >= 2 s back-to-back loop: C5 runs against
the board's power limit and the clocks it holds after ~100 ms are lower than in a short burst), fractions against
the nominal peaks, and -- on the default run -- `extra.C4` (the other "mixed config" of the 70 % bar), `extra.C3`
(prefill-only: the fused kernel variant), `extra.C5_two_call` and `extra.MIG` (KV migration).  `--config MIG` makes the migration the line's own workload.

N > 1 (torchrun): the path shards by request with no collective; each rank runs its own
replica of the workload (weak scaling), timing = max over ranks.
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
NOMINAL = dict(hbm_gbs=8000.0, bf16_tflops=2250.0)  # B200 data sheet, dense


# ----------------------------------------------------------------------------- roofline arithmetic
def step_counts(s_or_lengths):
    """FLOPs / algorithmic bytes of a step; the attention call's share separately.

    step_bytes: prior K+V read once, new K/V rows read and written once, Q read, O written, page table.
    attn_bytes: what of that belongs to tropical_mixed_attention: prior K+V, Q, O, page table.  The re-read of this
    step's new rows from the pool (4 Hkv d T) is an implementation cost, not algorithmic (reading S21)."""
    Hq, Hkv, d, P, q, c = s_or_lengths
    q = q.astype(np.float64)
    c = c.astype(np.float64)
    T = q.sum()
    L = q + c
    pages = np.ceil(L[q > 0] / P).sum()
    flops = 4.0 * d * Hq * (q * c + q * (q + 1) / 2).sum()
    step_bytes = 4.0 * Hkv * d * c[q > 0].sum() + 2 * (4.0 * Hkv * d * T) + 2 * (2.0 * Hq * d * T) + 4.0 * pages
    attn_bytes = 4.0 * Hkv * d * c[q > 0].sum() + 2 * (2.0 * Hq * d * T) + 4.0 * pages
    return dict(flops=flops, step_bytes=step_bytes, attn_bytes=attn_bytes, new_tokens=T)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


KERNEL_SOURCES = ("common.cuh", "decode.cuh", "mixed.cu", "plan.cuh", "prefill.cuh", "kv_append.cu", "step_variant.h")


def kernel_source_sha() -> str:
    """Fingerprint of the step's kernel sources as they are on disk (`python bench.py --kernel-sha` prints it): an ncu
    capture is only quoted for the kernels it was taken from."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2606_16264_b200", "csrc", name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:12]


def ncu_traffic(config: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, one launch, from the committed ncu capture
    of this config (profiles/ncu_traffic.csv: config, bytes, capture file, kernel_source_sha at capture time; the .md
    beside it names the command).  None when there is no capture of THESE kernel sources: a capture of an older kernel
    is not quoted."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    sha = kernel_source_sha()
    for line in open(path):
        f = line.strip().split(",")
        if len(f) >= 4 and f[0] == config and f[3] == sha:
            return float(f[1])
    return None


def roofline_times(cnt, peaks):
    t_bytes = cnt["step_bytes"] / (peaks["hbm_gbs"] * 1e3)
    t_flops = cnt["flops"] / (peaks["bf16_tflops_sustained"] * 1e6)
    t_nom = max(cnt["step_bytes"] / (NOMINAL["hbm_gbs"] * 1e3), cnt["flops"] / (NOMINAL["bf16_tflops"] * 1e6))
    return t_bytes, t_flops, max(t_bytes, t_flops), t_nom


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

    def finish(self):
        self.stop_flag = True
        self.join()
        return self.summary()

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


def gather_over_ranks(value: float, world: int, device) -> list:
    """Every rank's figure, in rank order (reported beside the maximum)."""
    if world <= 1:
        return [float(value)]
    import torch
    import torch.distributed as dist
    mine = torch.tensor([float(value)], dtype=torch.float64, device=device)
    parts = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    return [float(p.item()) for p in parts]


def whole_job_tokens_per_s(new_tokens_per_replica: float, world: int, us_per_step: float) -> float:
    """Aggregate over all replicas (weak scaling: every rank runs its own copy of the workload)."""
    return new_tokens_per_replica * world / (us_per_step * 1e-6)


def make_workload(name: str, rank: int, part: str = "all"):
    """part = "prefill" / "decode": only those requests of the config (analysis runs: what each role costs alone)."""
    t0 = time.perf_counter()
    if rank == 0 and part == "all":
        s = synth.make_config(name, poison=False, values="tiled")
    else:  # replica with the same lengths, different page placement / values
        seed, Hq, Hkv, d, P, q, c, _ = synth.config_lengths(name)
        if part != "all":
            keep = (q > 1) if part == "prefill" else (q == 1)
            q, c = q[keep], c[keep]
        s = synth.make_step(np.random.default_rng(1000 + rank), Hq, Hkv, d, P, q, c, poison=False, values="tiled",
                            name=name, seed=seed)
    return s, time.perf_counter() - t0


def config_dict(name, part, cnt, world):
    """The line's `config`: the workload and how the L2 is kept out of the timing -- the same dict in both arms."""
    flush = cnt["step_bytes"] < 5e8
    return {"workload": f"{name} ({describe(name)})" + ("" if part == "all" else f", its {part} requests only (analysis run)"),
            "replicas": world,
            "l2": ("step touches %.2f GB >> 126 MB L2, no flush needed" % (cnt["step_bytes"] / 1e9)) if not flush else
                  "L2 flushed (512 MB rewritten, untimed) between timed steps; per-step event times summed",
            "new_tokens_per_step": int(cnt["new_tokens"])}


def describe(name):
    return {"C1": "tiny mixed 4/4/64", "C2": "decode-only 32/32/128 x64", "C3": "prefill-only 32/32/128 x4",
            "C4": "mixed 13B-like 40/40/128: 2048 chunk + 128 decodes",
            "C5": "mixed GQA 64/8/128: 4096+1024 chunks + 256 decodes",
            "MIG": "KV migration of the C5 cache (258 requests, 64/8/128) pool -> pool under a new page table"}[name]


# ----------------------------------------------------------------------------- timing of the attention step
class StepTimer:
    """The step of one config on the current device: append + attention through the C-ABI binding."""

    def __init__(self, s, tb, torch, two_call=False, dev=None):
        from paper_2606_16264_b200.harness import DeviceStep
        self.s, self.tb, self.torch = s, tb, torch
        # False (default): the step is ONE call, tropical_mixed_step (KV append fused into the step kernel);
        # True: tropical_kv_append followed by tropical_mixed_attention (three launches, the r1 / r2a chain)
        self.two_call = two_call
        self.cnt = step_counts((s.num_q_heads, s.num_kv_heads, s.head_dim, s.page_size, s.q_lens, s.ctx_lens))
        self.dev = dev if dev is not None else DeviceStep(s)
        self.stream = torch.cuda.current_stream()
        # A step whose working set fits the 126 MB L2 is timed cold: a 512 MB buffer is rewritten between timed steps
        # (untimed) and the per-step event times are summed.  The big configs (> 0.5 GB per step) need no flush.
        self.flush = self.cnt["step_bytes"] < 5e8
        self.flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda") if self.flush else None
        self.launches_per_step = 0

    def one_step(self, ev=None):
        """One step.  ev = (start, middle, end) events of the instrumented pass: when the step runs as append kernel +
        attention launches (--two-call, or tropical_mixed_step's choice on a decode-heavy step: the very same kernels)
        the middle event sits between the two, so that the attention launches are timed on their own."""
        tb, dev = self.tb, self.dev
        split = self.two_call or (ev is not None and self.launches_per_step == 3)
        if ev is not None:
            ev[0].record(self.stream)
        n = 0
        if split:
            tb.kv_append(dev.pool, dev.batch, dev.k_new, dev.v_new)
            n = tb.last_launch_count()
        if ev is not None:
            ev[1].record(self.stream)
        if split:
            tb.mixed_attention(dev.pool, dev.batch, dev.q, out=dev.out, workspace=dev.workspace)
        else:
            tb.mixed_step(dev.pool, dev.batch, dev.q, dev.k_new, dev.v_new, out=dev.out, workspace=dev.workspace)
        n += tb.last_launch_count()
        if ev is not None:
            ev[2].record(self.stream)
        self.launches_per_step = n
        return n

    def warm(self, n):
        for _ in range(max(n, 3)):
            self.one_step()
        self.torch.cuda.synchronize()

    def timed(self, steps):
        """EXACTLY `steps` steps between two events (per-step events summed when the L2 is flushed in between)."""
        torch = self.torch
        ev = lambda: torch.cuda.Event(enable_timing=True)
        st = [(ev(), ev()) for _ in range(steps)] if self.flush else None
        e0, e1 = ev(), ev()
        torch.cuda.synchronize()
        e0.record(self.stream)
        for k in range(steps):
            if self.flush:
                self.flush_buf.fill_(k & 0xff)
                st[k][0].record(self.stream)
            self.one_step()
            if self.flush:
                st[k][1].record(self.stream)
        e1.record(self.stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in st) if self.flush else e0.elapsed_time(e1)

    def timed_warm(self, steps):
        """Small configs only: the same per-step event pairs as `timed`, WITHOUT the L2 flush in between -- the step's
        working set (pages, q, workspace) is still in the 126 MB L2 from the step before.  Returns ms for `steps` steps."""
        torch = self.torch
        ev = lambda: torch.cuda.Event(enable_timing=True)
        st = [(ev(), ev()) for _ in range(steps)]
        torch.cuda.synchronize()
        for k in range(steps):
            st[k][0].record(self.stream)
            self.one_step()
            st[k][1].record(self.stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in st)

    def instrumented(self, steps):
        """Second pass over the same steps with events around every step and between its two calls: per-step times
        (median / min / max) and the attention launches' share.  Kept out of the timed region: the event between the
        append and the attention breaks the tile directory's overlap with the append."""
        torch = self.torch
        ev = lambda: torch.cuda.Event(enable_timing=True)
        evs = [(ev(), ev(), ev()) for _ in range(steps)]
        for k in range(steps):
            if self.flush:
                self.flush_buf.fill_(k & 0xff)
            self.one_step(evs[k])
        torch.cuda.synchronize()
        step_us = np.array([a.elapsed_time(c) for a, _, c in evs]) * 1e3
        attn_us = np.array([b.elapsed_time(c) for _, b, c in evs]) * 1e3
        return step_us, attn_us

    def timeline(self, reps=8):
        """Measurement builds only (-DTROPICAL_TIMELINE): when each of the step's three kernels starts and ends, median
        over `reps` steps (L2 flushed before each so that the chain of cold metadata loads is visible)."""
        tb, torch = self.tb, self.torch
        if tb.debug_timeline(reset=True) is None:
            return None
        buf = self.flush_buf if self.flush_buf is not None else torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
        rows = []
        for k in range(reps):
            tb.debug_timeline(reset=True)   # synchronises: re-arm first, then keep the GPU busy with the flush so that
            buf.fill_(k & 0xff)             # the step's launches are queued behind it (no host launch latency inside)
            self.one_step()
            t = tb.debug_timeline()
            rows.append([t.get(f, float("nan")) / 1e3 for f in tb.TIMELINE_FIELDS])
        med = np.nanmedian(np.array(rows), axis=0)
        return {f: round(float(v), 1) for f, v in zip(tb.TIMELINE_FIELDS, med) if v == v}   # no append stamps on a fused step

    def sustained(self, seconds, local):
        """The step back to back for >= `seconds`: what a long-running worker sees once the power management has
        settled (C5 runs against the 1000 W board limit; a 50 ms burst holds higher clocks)."""
        torch = self.torch
        if self.flush:
            return None
        sampler = ClockSampler(local)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n, t_end = 0, time.perf_counter() + seconds
        torch.cuda.synchronize()
        # settle first (untimed), then time the second half
        while time.perf_counter() < t_end - seconds / 2:
            for _ in range(20):
                self.one_step()
            torch.cuda.synchronize()
        e0.record(self.stream)
        while time.perf_counter() < t_end:
            for _ in range(20):
                self.one_step()
            n += 20
            torch.cuda.synchronize()
        e1.record(self.stream)
        torch.cuda.synchronize()
        clk = sampler.finish()
        return dict(us=e0.elapsed_time(e1) * 1e3 / n, steps=n, seconds=seconds, clocks=clk)


def e2e_host_step(st: StepTimer, steps, world):
    """The step through tropical_step_host: pinned host buffers, H2D + D2H inside the timed region."""
    torch, tb, s, dev = st.torch, st.tb, st.s, st.dev
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
    n = max(3, min(steps, 50))
    t0 = time.perf_counter()
    for _ in range(n):
        host_step()
    us = (time.perf_counter() - t0) / n * 1e6
    us = max_over_ranks(us, world, "cuda")
    h2d = sum(int(h[k].numel() * h[k].element_size()) for k in h)
    return us, h2d, int(h_out.numel() * 2)


# ----------------------------------------------------------------------------- KV migration (NEXT-3)
class MigrationTimer:
    """The cache of every request of a step after its append (L_i tokens each) moves from the step's pool into a second
    pool under a fresh random page table: tropical_kv_migrate."""

    def __init__(self, s, tb, torch, dst_device=None, src_pools=None):
        from paper_2606_16264_b200.harness import to_dev
        self.s, self.tb, self.torch = s, tb, torch
        self.L = (s.q_lens.astype(np.int64) + s.ctx_lens).astype(np.int32)
        self.dst_pt, n_dst = synth.make_migration_target(np.random.default_rng(77), self.L, s.page_size)
        self.k_src, self.v_src = src_pools if src_pools is not None else (to_dev(s.k_pool), to_dev(s.v_pool))
        self.src = tb.KVPool(self.k_src, self.v_src, s.num_q_heads)
        shape = (n_dst, s.num_kv_heads, s.page_size, s.head_dim)
        dd = dst_device if dst_device is not None else torch.cuda.current_device()
        self.k_dst = torch.zeros(shape, dtype=torch.int16, device=f"cuda:{dd}")
        self.v_dst = torch.zeros(shape, dtype=torch.int16, device=f"cuda:{dd}")
        self.dst = tb.KVPool(self.k_dst, self.v_dst, s.num_q_heads)
        self.lens_d, self.spt, self.dpt = to_dev(self.L), to_dev(s.page_table), to_dev(self.dst_pt)
        self.max_len = int(self.L.max())
        self.tokens = int(self.L.sum())
        # K + V, read once from the source pool and written once to the destination pool, + the two page tables
        self.bytes = 2.0 * (4.0 * s.num_kv_heads * s.head_dim * self.tokens) + 8.0 * float(np.ceil(self.L / s.page_size).sum())
        self.stream = torch.cuda.current_stream()

    def call(self):
        self.tb.kv_migrate(self.src, self.dst, self.lens_d, self.spt, self.dpt, self.max_len)
        return self.tb.last_launch_count()

    def timed(self, steps, warmup):
        torch = self.torch
        n = 0
        for _ in range(max(3, warmup)):
            n = self.call()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(self.stream)
        for _ in range(steps):
            self.call()
        e1.record(self.stream)
        torch.cuda.synchronize()
        total_ms = e0.elapsed_time(e1)
        for a, b in evs:
            a.record(self.stream)
            self.call()
            b.record(self.stream)
        torch.cuda.synchronize()
        per = np.array([a.elapsed_time(b) for a, b in evs]) * 1e3
        return total_ms, per, n


def migration_report(s, tb, torch, steps, warmup, peaks, local, world, src_pools=None):
    mt = MigrationTimer(s, tb, torch, src_pools=src_pools)
    sampler = ClockSampler(local)
    sampler.start()
    total_ms, per, launches = mt.timed(steps, warmup)
    clk = sampler.finish()
    us = max_over_ranks(total_ms * 1e3 / steps, world, "cuda")
    rep = dict(us=us, per=per, launches=launches, clocks=clk, bytes=mt.bytes, tokens=mt.tokens,
               gbs=mt.bytes / (us * 1e3), frac=mt.bytes / (us * 1e3) / peaks["hbm_gbs"])
    # the peer path: the same call with the destination pool on a second GPU, pushed over NVLink
    if world == 1 and torch.cuda.device_count() >= 2:
        peer = torch.cuda.current_device() ^ 1
        if tb.enable_peer_access(peer):
            mp = MigrationTimer(s, tb, torch, dst_device=peer, src_pools=(mt.k_src, mt.v_src))
            k = max(3, steps // 4)
            p_ms, _, _ = mp.timed(k, 3)
            p_us = p_ms * 1e3 / k
            rep["peer"] = {"us": round(p_us, 1), "link_gbs_one_direction": round(mt.bytes / 2 / (p_us * 1e3), 1),
                           "dst_device": peer}
        else:
            rep["peer"] = "not measured: no peer path between the visible GPUs"
    else:
        rep["peer"] = ("not measured: one GPU visible to this process (same kernel; the destination pointers would be "
                       "peer-mapped memory)")
    return mt, rep


# ----------------------------------------------------------------------------- main legs
def run_ours(args, rank, world):
    import torch
    import torch.distributed as dist
    import paper_2606_16264_b200 as tb

    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    peaks = load_peaks()
    if args.config == "MIG":
        return run_migration(args, rank, world, local, tb, torch, dist, peaks)
    s, gen_s = make_workload(args.config, rank, args.part)
    st = StepTimer(s, tb, torch, two_call=args.two_call)
    cnt = st.cnt
    warm = max(args.warmup, 3)
    st.warm(warm)
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    total_ms = st.timed(args.steps)                # the timed region: exactly K steps, nothing but the two library calls
    n_k = min(args.steps, 100)
    step_us, attn_us = st.instrumented(n_k)
    roles = tb.debug_read_profile(st.dev.workspace)  # of the LAST launch of the instrumented pass
    if total_ms < 400:  # keep the GPU busy long enough for the clock sampler to see it under load
        t_end = time.perf_counter() + 0.4
        while time.perf_counter() < t_end:
            st.one_step()
        torch.cuda.synchronize()
    clocks = sampler.finish()
    per_rank_us = [round(ms / args.steps * 1e3, 2) for ms in gather_over_ranks(total_ms, world, "cuda")]
    total_ms = max_over_ranks(total_ms, world, "cuda")
    ms_per_step = total_ms / args.steps
    us = ms_per_step * 1e3
    sus = st.sustained(args.sustain_seconds, local) if args.sustain_seconds > 0 else None
    e2e_us, h2d, d2h = e2e_host_step(st, args.steps, world)
    tl = st.timeline()

    extra = {}
    if args.config == "C5" and args.part == "all" and not args.no_extra and world == 1:
        extra = run_extras(args, tb, torch, peaks, local, st)
    if rank != 0:
        return
    t_bytes_us, t_flops_us, t_roof, t_nom = roofline_times(cnt, peaks)
    attn_med = float(np.median(attn_us))
    # algorithmic bytes of the dominant launch: the whole step's when the append runs inside the step kernel
    kernel_bytes = cnt["attn_bytes"] if st.launches_per_step == 3 else cnt["step_bytes"]
    # Duration of those launches IN THE TIMED REGION: the region's own mean step time times their share of a step, the
    # share taken from the event pairs of the second pass (an event between the append and the attention launches
    # cannot sit inside the timed region: it would undo the programmatic overlap of the two).  The second pass's own
    # absolute times are reported beside it: on C5 they are those of a GPU that has been under load for 0.1 s longer.
    share = float(np.median(attn_us / step_us))
    kernel_us = us * share
    achieved = kernel_bytes / (kernel_us * 1e3)  # GB/s
    if args.no_cpu:
        cpu_us, cpu_desc, cores = float("nan"), "skipped (--no-cpu)", 0
    else:
        cpu_us, cpu_desc, cores, _ = oracle_sample_us(s)
    line = {
        "metric": METRIC, "value": round(us, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warm, "ms_per_step": round(ms_per_step, 5), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": config_dict(args.config, args.part, cnt, world),
        "step_call": ("tropical_kv_append + tropical_mixed_attention (3 launches)" if args.two_call else
                      "tropical_mixed_step: one call; " +
                      ("its fused kernel variant, KV append inside the step kernel (2 launches)"
                       if st.launches_per_step == 2 else
                       "decode-heavy step: its append kernel in front of the plain step kernel (3 launches)")),
        "tokens_per_s": round(whole_job_tokens_per_s(cnt["new_tokens"], world, us), 1),
        "per_rank_us": per_rank_us,  # value = their maximum
        "us_per_step": {"mean_timed_region": round(us, 2), "median": round(float(np.median(step_us)), 2),
                        "min": round(float(step_us.min()), 2), "max": round(float(step_us.max()), 2),
                        "of": f"{n_k} per-step event pairs, second pass (rank 0)"},
        "step_roofline": {"t_bytes_us": round(t_bytes_us, 2), "t_flops_us": round(t_flops_us, 2),
                          "t_roof_us": round(t_roof, 2), "frac": round(t_roof / us, 4),
                          "frac_of_nominal_peaks": round(t_nom / us, 4), "t_roof_nominal_us": round(t_nom, 2),
                          "achieved_gbs": round(cnt["step_bytes"] / (us * 1e3), 1),
                          "achieved_tflops": round(cnt["flops"] / (us * 1e6), 1),
                          "peaks": peaks, "nominal": NOMINAL},
        "roofline": {"bound": "hbm",
                     "kernel": ("the attention launches of the step: tile directory + persistent step kernel (>= 98 % of them)"
                                if st.launches_per_step == 3 else
                                "launches of tropical_mixed_step, fused variant: tile directory + persistent step kernel with "
                                "the KV append inside (>= 98 % of them)"),
                     "achieved": round(achieved, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
                     "frac": round(achieved / peaks["hbm_gbs"], 4), "traffic": ncu_traffic(args.config),
                     "kernel_us": round(kernel_us, 2), "kernel_share_of_step": round(share, 4),
                     "kernel_us_second_pass": {"median": round(attn_med, 2), "min": round(float(attn_us.min()), 2)},
                     "algorithmic_bytes": kernel_bytes, "of": peaks["source"],
                     "timing": ("kernel_us = mean step time of the timed region x the launches' share of a step; share = median "
                                f"over {n_k} event pairs of a second pass over the same steps" +
                                (" (the same kernels, launched as append call + attention call so that an event fits between)"
                                 if st.launches_per_step == 3 else ""))},
        "cpu_baseline": {"value": round(cpu_us, 1), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": cpu_desc},
        "e2e": {"value": round(e2e_us, 2), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(st.launches_per_step) * args.steps,
        "clocks": clocks,
        "gen_seconds": round(gen_s, 1),
        "role_finish_us": (dict({k: round(v / 1e3, 1) for k, v in roles.items()},
                                launch="last step kernel of the second (instrumented) pass") if roles is not None else
                           "not stamped: product build (measurement builds: TROPICAL_NVCC_EXTRA=-DTROPICAL_ROLE_PROF)"),
    }
    if st.launches_per_step == 3:  # row A1 on its own: the append kernel between its two events of the second pass
        app_us = float(np.median(step_us - attn_us))
        app_bytes = cnt["step_bytes"] - cnt["attn_bytes"]
        line["append_kernel"] = {"us": round(app_us, 2), "bytes": app_bytes, "gbs": round(app_bytes / (app_us * 1e3), 1),
                                 "frac_of_hbm_peak": round(app_bytes / (app_us * 1e3) / peaks["hbm_gbs"], 4),
                                 "of": f"median over {n_k} event pairs of the second pass (includes the event and launch gaps around an "
                                       "11 us kernel: profiles/r3b_final.md has its ncu time); bytes = rows read + rows written"}
    if sus is not None:
        line["sustained"] = {"value": round(sus["us"], 2), "unit": UNIT, "frac": round(t_roof / sus["us"], 4),
                             "steps": sus["steps"], "clocks": sus["clocks"],
                             "how": f"back to back for {sus['seconds']:.1f} s, second half timed"}
    if tl is not None:
        line["timeline_us"] = dict(tl, note="-DTROPICAL_TIMELINE build: not a bench build; L2 flushed before each step")
    if extra:
        line["extra"] = extra
    if "WHATIF" in tb.version():
        line["invalid"] = tb.version()   # a what-if measurement build computes wrong results: never a bench value
    print(json.dumps(line))


def run_extras(args, tb, torch, peaks, local, st_c5):
    """On the default (C5) run: the other mixed config of the 70 % bar, and the KV migration of the C5 cache."""
    extra = {}
    steps = min(args.steps, 100)
    try:  # NEXT-3 on the pools that are already resident (they hold the step's rows: the timed steps appended them)
        _, rep = migration_report(st_c5.s, tb, torch, steps, 3, peaks, local, 1,
                                  src_pools=(st_c5.dev.k_pool, st_c5.dev.v_pool))
        extra["MIG"] = {"workload": describe("MIG"), "us": round(rep["us"], 1), "us_min": round(float(rep["per"].min()), 1),
                        "gbs_read_plus_write": round(rep["gbs"], 1), "frac_of_hbm_peak": round(rep["frac"], 4),
                        "bytes": rep["bytes"], "tokens": rep["tokens"],
                        "us_per_token_per_layer": round(rep["us"] / rep["tokens"], 6), "peer": rep["peer"],
                        "clocks": rep["clocks"]}
    except Exception as exc:  # an extra must never cost the headline line
        extra["MIG"] = {"error": repr(exc)}
    try:  # the same C5 step as two calls (append kernel + attention): what fusing the append is worth, same box
        st2 = StepTimer(st_c5.s, tb, torch, two_call=True, dev=st_c5.dev)   # same resident pools and inputs
        st2.warm(3)
        us2 = st2.timed(steps) * 1e3 / steps
        extra["C5_two_call"] = {"workload": "C5 as tropical_kv_append + tropical_mixed_attention (3 launches)",
                                "value": round(us2, 2), "unit": UNIT, "steps": steps}
    except Exception as exc:
        extra["C5_two_call"] = {"error": repr(exc)}
    try:
        s4, _ = make_workload("C4", 0)
        st = StepTimer(s4, tb, torch)
        st.warm(3)
        sampler = ClockSampler(local)
        sampler.start()
        us = st.timed(steps) * 1e3 / steps
        step_us, attn_us = st.instrumented(min(steps, 50))
        clk = sampler.finish()
        _, _, t_roof, t_nom = roofline_times(st.cnt, peaks)
        extra["C4"] = {"workload": f"C4 ({describe('C4')})", "value": round(us, 2), "unit": UNIT, "steps": steps,
                       "frac": round(t_roof / us, 4), "frac_of_nominal_peaks": round(t_nom / us, 4),
                       "t_roof_us": round(t_roof, 2), "median": round(float(np.median(step_us)), 2),
                       "min": round(float(step_us.min()), 2), "kernel_us": round(float(np.median(attn_us)), 2),
                       "clocks": clk}
    except Exception as exc:
        extra["C4"] = {"error": repr(exc)}
    try:  # the prefill-only config: tropical_mixed_step takes its fused kernel variant there (cold L2, as --config C3)
        s3, _ = make_workload("C3", 0)
        st = StepTimer(s3, tb, torch)
        st.warm(3)
        n3 = min(steps, 50)
        us = st.timed(n3) * 1e3 / n3
        _, _, t_roof, t_nom = roofline_times(st.cnt, peaks)
        warm_us = st.timed_warm(n3) * 1e3 / n3
        extra["C3"] = {"workload": f"C3 ({describe('C3')})", "value": round(us, 2), "unit": UNIT, "steps": n3,
                       "frac": round(t_roof / us, 4), "t_roof_us": round(t_roof, 2), "launches_per_step": st.launches_per_step,
                       "l2": "flushed between timed steps", "warm_l2": {"value": round(warm_us, 2), "frac": round(t_roof / warm_us, 4)}}
    except Exception as exc:
        extra["C3"] = {"error": repr(exc)}
    try:  # the decode-only config (bandwidth bound; 1.33 GB per step, no flush needed)
        s2, _ = make_workload("C2", 0)
        st = StepTimer(s2, tb, torch)
        st.warm(3)
        sampler = ClockSampler(local)
        sampler.start()
        us = st.timed(steps) * 1e3 / steps
        step_us, attn_us = st.instrumented(min(steps, 50))
        clk = sampler.finish()
        _, _, t_roof, t_nom = roofline_times(st.cnt, peaks)
        extra["C2"] = {"workload": f"C2 ({describe('C2')})", "value": round(us, 2), "unit": UNIT, "steps": steps,
                       "frac": round(t_roof / us, 4), "frac_of_nominal_peaks": round(t_nom / us, 4),
                       "t_roof_us": round(t_roof, 2), "median": round(float(np.median(step_us)), 2),
                       "min": round(float(step_us.min()), 2), "kernel_us": round(float(np.median(attn_us)), 2),
                       "launches_per_step": st.launches_per_step, "clocks": clk}
    except Exception as exc:
        extra["C2"] = {"error": repr(exc)}
    try:  # the tiny config: launch-latency bound; cold and warm L2 separately
        s1, _ = make_workload("C1", 0)
        st = StepTimer(s1, tb, torch)
        st.warm(3)
        n1 = min(steps, 50)
        us = st.timed(n1) * 1e3 / n1
        warm_us = st.timed_warm(n1) * 1e3 / n1
        _, _, t_roof, _ = roofline_times(st.cnt, peaks)
        extra["C1"] = {"workload": f"C1 ({describe('C1')})", "value": round(us, 2), "unit": UNIT, "steps": n1,
                       "frac": round(t_roof / us, 4), "t_roof_us": round(t_roof, 3), "launches_per_step": st.launches_per_step,
                       "l2": "flushed between timed steps", "warm_l2": {"value": round(warm_us, 2), "frac": round(t_roof / warm_us, 4)}}
    except Exception as exc:
        extra["C1"] = {"error": repr(exc)}
    return extra


def run_migration(args, rank, world, local, tb, torch, dist, peaks):
    import oracle
    s, gen_s = make_workload("C5", rank)
    oracle.kv_append(s.k_pool, s.v_pool, s.q_lens, s.ctx_lens, s.q_offsets, s.page_table, s.k_new, s.v_new)
    if world > 1:
        dist.barrier()
    mt, rep = migration_report(s, tb, torch, args.steps, args.warmup, peaks, local, world)
    # e2e: the migration's metadata (lengths and both page tables) from pinned host memory, then the call, then a sync
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h = [pin(mt.L), pin(s.page_table), pin(mt.dst_pt)]
    d = [mt.lens_d, mt.spt, mt.dpt]
    n = max(3, min(args.steps, 50))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(n):
        for a, b in zip(h, d):
            b.copy_(a, non_blocking=True)
        mt.call()
        torch.cuda.synchronize()
    e2e_us = max_over_ranks((time.perf_counter() - t0) / n * 1e6, world, "cuda")
    if rank != 0:
        return
    if args.no_cpu:
        cpu_us, cores, desc = float("nan"), 0, "skipped (--no-cpu)"
    else:
        kd, vd = np.zeros(tuple(mt.k_dst.shape), np.uint16), np.zeros(tuple(mt.k_dst.shape), np.uint16)
        t0 = time.perf_counter()
        oracle.kv_migrate(s.k_pool, s.v_pool, kd, vd, mt.L, s.page_table, mt.dst_pt)
        cpu_us, cores = (time.perf_counter() - t0) * 1e6, 1
        desc = "oracle.kv_migrate on the whole workload (single-threaded C loops)"
    us = rep["us"]
    print(json.dumps({
        "metric": "KV migration time (SURVEY 8(f) NEXT-3)", "value": round(us, 2), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": round(us / 1e3, 5), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "u16", "data": "synthetic",
        "config": {"workload": f"MIG ({describe('MIG')})", "replicas": world, "tokens": rep["tokens"],
                   "l2": "5.1 GB moved per call >> 126 MB L2, no flush needed"},
        "us_per_step": {"median": round(float(np.median(rep["per"])), 2), "min": round(float(rep["per"].min()), 2)},
        "roofline": {"bound": "hbm", "kernel": "kv_migrate_kernel", "achieved": round(rep["gbs"], 1),
                     "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": round(rep["frac"], 4), "traffic": ncu_traffic("MIG"),
                     "algorithmic_bytes": rep["bytes"], "of": peaks["source"],
                     "frac_of_nominal_peak": round(rep["gbs"] / NOMINAL["hbm_gbs"], 4)},
        "cpu_baseline": {"value": round(cpu_us, 1), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": round(e2e_us, 2), "unit": UNIT, "h2d_bytes_per_step": int(sum(x.numel() * 4 for x in h)),
                "d2h_bytes_per_step": 0},
        "gpu_launches": int(rep["launches"]) * args.steps, "clocks": rep["clocks"], "peer": rep["peer"],
        "gen_seconds": round(gen_s, 1),
    }))


def run_reference(args, rank, world):
    """The oracle as it stands, on host cores; each 'step' is a bounded sample of the workload sized so
    that the whole --steps K --warmup W run ends within a few minutes."""
    if rank != 0:
        return
    cfg = "C5" if args.config == "MIG" else args.config
    s, _ = make_workload(cfg, 0)
    _, _, cores, dt0 = oracle_sample_us(s, budget_rows_flops=2e8, seed=12345)  # calibrate rows/s
    per_step_s = min(10.0, max(0.05, 90.0 / max(1, args.steps + args.warmup)))
    budget = max(2e7, 2e8 * per_step_s / max(dt0, 1e-3))
    vals, secs, desc = [], [], ""
    for k in range(args.warmup + args.steps):
        us, desc, cores, dt = oracle_sample_us(s, budget_rows_flops=budget, seed=k)
        if k >= args.warmup:
            vals.append(us)
            secs.append(dt)
    us = float(np.mean(vals)) if vals else float("nan")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": round(us, 1), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(us / 1e3, 3), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, "all", step_counts((s.num_q_heads, s.num_kv_heads, s.head_dim, s.page_size, s.q_lens,
                                                          s.ctx_lens)), world),
        "cpu_baseline": {"value": round(us, 1), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": round(us, 1), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        # value / ms_per_step are whole-step figures EXTRAPOLATED by FLOP ratio from a bounded sample of rows per "step":
        # steps x ms_per_step is therefore not the wall time of this run, sample_seconds x steps (+ the appends) is
        "sampled": True, "sample_seconds": round(float(np.mean(secs)), 3) if secs else None,
    }))


def launch_ranks(args) -> int:
    """`python bench.py --gpus N` without torchrun around it: start N ranks of this same command line, one GPU each
    (torch.distributed.run sets RANK / LOCAL_RANK / WORLD_SIZE / MASTER_*; NCCL carries only the timing reductions).
    Refuses instead of quietly measuring fewer replicas than asked for.  P:184: 8 GPUs per node, P:186 request dispatch
    over independent workers -- the replicas share nothing."""
    import socket
    import subprocess
    if args.impl == "ours" and not args.rank_check:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            print(f"bench.py: --gpus {args.gpus} asked for, {have} CUDA device(s) visible: refusing to run fewer "
                  "replicas under the same label", file=sys.stderr)
            return 2
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def rank_check(rank: int, world: int) -> None:
    """The rank plumbing of the timed legs with no GPU in it: every rank reports a made-up step time (slower with
    rank), the job's time is the maximum, its throughput the sum over replicas; rank 0 prints one JSON line."""
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("gloo")
    mine = 100.0 + 25.0 * rank
    per_rank = gather_over_ranks(mine, world, "cpu")
    us = max_over_ranks(mine, world, "cpu")
    print(f"rank {rank} of {world}: {mine} us", file=sys.stderr, flush=True)
    if rank == 0:
        print(json.dumps({"rank_check": True, "n_gpus": world, "per_rank_us": per_rank, "value": us, "unit": UNIT,
                          "tokens_per_s": whole_job_tokens_per_s(60, world, us), "scaling": "weak"}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default="C5", choices=synth.CONFIG_NAMES + ("MIG",))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--part", default="all", choices=["all", "prefill", "decode"],
                    help="analysis runs: only the prefill (q > 1) or only the decode (q = 1) requests of the config")
    ap.add_argument("--two-call", action="store_true",
                    help="time the step as tropical_kv_append + tropical_mixed_attention instead of the fused tropical_mixed_step")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--no-extra", action="store_true", help="skip extra.C4 / extra.MIG on the default run")
    ap.add_argument("--sustain-seconds", type=float, default=2.0, help="length of the sustained loop (0 = skip)")
    ap.add_argument("--rank-check", action="store_true",
                    help="launcher check without GPU work: the ranks rendezvous over gloo, reduce a made-up time and "
                         "rank 0 prints the line's rank bookkeeping (what the CPU test of --gpus N drives)")
    ap.add_argument("--kernel-sha", action="store_true", help="print the fingerprint of the kernel sources and exit")
    args = ap.parse_args()
    if args.kernel_sha:
        print(kernel_source_sha())
        return
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        sys.exit(launch_ranks(args))
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if world != max(args.gpus, 1) and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; running {world} ranks", file=sys.stderr)
    if args.rank_check:
        return rank_check(rank, world)
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world)


if __name__ == "__main__":
    main()
