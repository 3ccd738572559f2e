"""Plain-Python restatement of the Tropical scheduler simulation -- TEST INFRASTRUCTURE (see oracle/__init__.py).

Follows the MODEL written out in include/tropical_sim.h rule by rule (section II-A: TTFT / TPOT / slack /
attainment, eq. 1-3; section IV-B, IV-C: slack check, Path 1 / Path 2, guards; P:186 least-unfinished-tokens
dispatch).  Slow and obvious on purpose: lists, linear scans, no event heap.  Shares no code with the C++
simulator (paper_2606_16264_b200/csrc/sim.cpp); it also restates the step-cost closed form (DESIGN.md
sections 6, 7) instead of calling the library.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional

COLOCATED, DISAGGREGATED, MULTIPLEXED = 0, 1, 2
INF = float("inf")


@dataclass
class CostModel:
    t0_us: float
    a_us_per_flop: float
    b_us_per_byte: float
    kappa: float
    e_prefill_iter_us: float
    e_decode_unit_us: float
    n_sm: float = 148.0
    e_prefill_crit_us: float = 0.0


@dataclass
class LayerShape:  # include/tropical.h tropical_layer_shape_t (NEXT-4)
    d_model: int = 0
    d_ffn: int = 0
    gated_mlp: int = 1
    num_layers: int = 1
    tp: int = 1


@dataclass
class LinearModel:  # include/tropical.h tropical_linear_model_t
    g0_us: float = 0.0
    f_us_per_flop: float = 0.0
    w_us_per_byte: float = 0.0
    kappa: float = 0.0
    ar0_us: float = 0.0
    ar_us_per_byte: float = 0.0


@dataclass
class Config:
    policy: int
    num_workers: int
    num_prefill_workers: int
    chunk_tokens: int
    ttft_slo_us: float
    tpot_slo_us: float
    decode_guard: float
    hbm_watermark: float
    kv_capacity_tokens: int
    migrate_us_per_token: float
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    num_layers: int
    attn: CostModel
    linear_us_per_token: float
    iter_overhead_us: float
    layer: LayerShape = field(default_factory=LayerShape)   # d_model > 0: iterations cost iter_cost_us (NEXT-4)
    linear: LinearModel = field(default_factory=LinearModel)
    role_transitions: int = 0
    delay_threshold: int = 0


def step_cost_us(cfg: Config, q_lens: List[int], ctx_lens: List[int], tp: int = 1) -> float:
    """t = t0 + max(aF, bB) + kappa min(aF, bB) + e_p N_p / n_sm + e_d N_d / n_sm + e_c N_c (DESIGN.md sections 6, 7), on the
    head shard Hq/tp, Hkv/tp (the path shards by kv head with no collective)."""
    Hq, Hkv, d, P = cfg.num_q_heads // tp, cfg.num_kv_heads // tp, cfg.head_dim, cfg.page_size
    qc = pages = T = csum = 0.0
    iters = units = crit = 0
    # the step's kernel variant: tropical_mixed_step fuses from 64 new tokens per request up (include/tropical.h)
    fused = len(q_lens) > 0 and sum(q_lens) >= 64 * len(q_lens)
    head_pairs = (Hq // Hkv) % 2 == 0
    for q, c in zip(q_lens, ctx_lens):
        if q <= 0:
            continue
        qc += float(q) * float(c) + float(q) * (float(q) + 1) / 2
        T += q
        csum += c
        L = q + c
        pages += (L + P - 1) // P
        if q == 1:
            units += ((L + P - 1) // P) * Hkv
        else:
            nt = (q + 127) // 128
            kv = []                                  # KV tiles of every 128-row tile of the chunk
            for ti in range(nt):
                last = c + min((ti + 1) * 128, q)
                kv.append((last + 127) // 128)
                iters += kv[-1] * Hq
            # heaviest item: two heads at the top tile / (fused variant, odd group) the top two row tiles / the top tile
            below = kv[-2] if nt >= 2 else 0
            crit = max(crit, 2 * kv[-1] if head_pairs else (kv[-1] + below if fused else kv[-1]))
    flops = 4.0 * d * Hq * qc
    nbytes = 2.0 * 2 * Hkv * d * csum + 2.0 * (2.0 * 2 * Hkv * d * T) + 2.0 * (2.0 * Hq * d * T) + 4.0 * pages
    m = cfg.attn
    t_tc, t_hbm = m.a_us_per_flop * flops, m.b_us_per_byte * nbytes
    hi, lo = max(t_tc, t_hbm), min(t_tc, t_hbm)
    nsm = m.n_sm if m.n_sm > 0 else 148.0
    return (m.t0_us + hi + m.kappa * lo + m.e_prefill_iter_us * iters / nsm + m.e_decode_unit_us * units / nsm +
            m.e_prefill_crit_us * crit)


def iter_cost_us(cfg: Config, q_lens: List[int], ctx_lens: List[int]) -> float:
    """include/tropical.h tropical_iter_cost: layers * (attention on the head shard + four GEMMs + two all-reduces)."""
    sh, lm = cfg.layer, cfg.linear
    T = float(sum(q_lens))
    mats = [(sh.d_model, (cfg.num_q_heads + 2 * cfg.num_kv_heads) * cfg.head_dim / sh.tp),     # QKV
            (cfg.num_q_heads * cfg.head_dim / sh.tp, sh.d_model),                               # O
            (sh.d_model, (2 if sh.gated_mlp else 1) * sh.d_ffn / sh.tp),                        # (gate and) up
            (sh.d_ffn / sh.tp, sh.d_model)]                                                     # down
    weights = sum(k * n for k, n in mats)
    flops = 2.0 * T * weights
    nbytes = 2.0 * weights + 2.0 * T * sum(k + n for k, n in mats)
    linear = allreduce = 0.0
    if T > 0:
        tf, tw = lm.f_us_per_flop * flops, lm.w_us_per_byte * nbytes
        linear = lm.g0_us + max(tf, tw) + lm.kappa * min(tf, tw)
        if sh.tp > 1:
            allreduce = 2.0 * (lm.ar0_us + lm.ar_us_per_byte * 2.0 * T * sh.d_model)
    return sh.num_layers * (step_cost_us(cfg, q_lens, ctx_lens, sh.tp) + linear + allreduce)


def iter_time_us(cfg: Config, q_lens: List[int], ctx_lens: List[int]) -> float:
    if cfg.layer.d_model > 0:
        return iter_cost_us(cfg, q_lens, ctx_lens) + cfg.iter_overhead_us
    return cfg.num_layers * step_cost_us(cfg, q_lens, ctx_lens) + cfg.linear_us_per_token * sum(q_lens) + cfg.iter_overhead_us


@dataclass
class _Req:
    arrival: float
    prompt: int
    output: int
    done_prompt: int = 0
    generated: int = 0          # decode tokens generated so far (the first token is the prefill's)
    first_token: float = -1.0
    finish: float = -1.0
    prefill_worker: int = -1
    decode_worker: int = -1
    multiplexed: int = 0


@dataclass
class _Worker:
    local_q: List[int] = field(default_factory=list)      # requests waiting for / in prefill here (FIFO)
    resident: List[int] = field(default_factory=list)     # requests decoding here
    pending: List[tuple] = field(default_factory=list)    # (available_at, rid): KV cache in migration to here
    busy_until: float = INF                               # INF = idle
    it_decodes: List[int] = field(default_factory=list)
    it_prefill: int = -1
    it_chunk: int = 0


def simulate(cfg: Config, requests: List[tuple]):
    """requests: [(arrival_us, prompt_len, output_len)] sorted by arrival.  Returns (results, summary):
    results[i] = dict(ttft_us, tpot_us, first_token_us, finish_us, prefill_worker, decode_worker, multiplexed)."""
    R = [_Req(float(a), int(p), int(o)) for a, p, o in requests]
    W = [_Worker() for _ in range(cfg.num_workers)]
    # role of each worker: True = dedicated prefill worker (disaggregated / multiplexed policies); P:161 may change it
    prefill_role = [cfg.policy != COLOCATED and w < cfg.num_prefill_workers for w in range(cfg.num_workers)]
    toggle_q: List[int] = []
    next_arrival = 0
    iterations = 0
    now = 0.0
    delayed = 0                      # prefills sent by the no-starvation rule since the last multiplexing -> prefill transition
    transitions = [0, 0]             # [to multiplexing, to prefill]

    def is_prefill_worker(w):
        return prefill_role[w]

    def prefill_workers():
        return [w for w in range(cfg.num_workers) if prefill_role[w]]

    def mux_workers():
        return [w for w in range(cfg.num_workers) if not prefill_role[w]]

    def remaining_output(r):
        return R[r].output - 1 - R[r].generated

    def unfinished_tokens(w):
        t = 0
        for r in W[w].local_q:
            t += (R[r].prompt - R[r].done_prompt) + remaining_output(r)
        for r in W[w].resident:
            t += remaining_output(r)
        for _, r in W[w].pending:
            t += remaining_output(r)
        return t

    def resident_kv(w):
        t = 0
        for r in W[w].local_q + W[w].resident + [r for _, r in W[w].pending]:
            t += R[r].done_prompt + R[r].generated
        return t

    def pred_exec(r):  # the rest of r's prompt as one iteration of its own ("execution time of a prefill request")
        return iter_time_us(cfg, [R[r].prompt - R[r].done_prompt], [R[r].done_prompt])

    def pred_queue(w):  # P:157 "queuing time when scheduling to the local worker"
        t = 0.0
        q = W[w].local_q
        if W[w].busy_until != INF:
            t += W[w].busy_until - now
            q = q[1:] if W[w].it_prefill >= 0 else q
        for r in q:
            t += pred_exec(r)
        return t

    def decode_batch(w):
        return [1] * len(W[w].resident), [R[r].prompt + R[r].generated for r in W[w].resident]

    def place_for_decode(r):  # after a prefill on a dedicated prefill worker: P:155 decode queue, P:186 dispatch
        best = min(mux_workers(), key=lambda w: (unfinished_tokens(w), w))
        W[best].pending.append((now + cfg.migrate_us_per_token * R[r].prompt, r))
        R[r].decode_worker = best

    def finish_iteration(w):
        wk = W[w]
        for r in wk.it_decodes:
            R[r].generated += 1
            if R[r].generated == R[r].output - 1:
                R[r].finish = now
                wk.resident.remove(r)
        r = wk.it_prefill
        if r >= 0:
            R[r].done_prompt += wk.it_chunk
            if R[r].done_prompt == R[r].prompt:
                wk.local_q.pop(0)
                R[r].first_token = now
                if R[r].output == 1:
                    R[r].finish = now
                    R[r].decode_worker = w
                elif is_prefill_worker(w):
                    place_for_decode(r)
                else:
                    wk.resident.append(r)
                    R[r].decode_worker = w
        wk.busy_until, wk.it_decodes, wk.it_prefill, wk.it_chunk = INF, [], -1, 0

    def try_start(w):
        nonlocal iterations
        wk = W[w]
        still = []
        for av, r in wk.pending:  # migrated caches that have arrived join the batch
            if av <= now:
                wk.resident.append(r)
            else:
                still.append((av, r))
        wk.pending = still
        q_lens, ctx_lens = [], []
        if wk.local_q:
            r = wk.local_q[0]
            rest = R[r].prompt - R[r].done_prompt
            chunk = rest if (cfg.chunk_tokens <= 0 or is_prefill_worker(w)) else min(rest, cfg.chunk_tokens)
            wk.it_prefill, wk.it_chunk = r, chunk
            q_lens.append(chunk)
            ctx_lens.append(R[r].done_prompt)
        wk.it_decodes = list(wk.resident)
        dq, dc = decode_batch(w)
        q_lens += dq
        ctx_lens += dc
        if not q_lens:
            return
        wk.busy_until = now + iter_time_us(cfg, q_lens, ctx_lens)
        iterations += 1

    def role_transitions():  # P:161, readings of include/tropical_sim.h
        nonlocal delayed
        threshold = cfg.hbm_watermark * cfg.kv_capacity_tokens
        if all(resident_kv(w) > threshold for w in mux_workers()) and len(prefill_workers()) >= 2:
            w = min(prefill_workers(), key=lambda w: (pred_queue(w), w))
            prefill_role[w] = False
            transitions[0] += 1
        if delayed >= cfg.delay_threshold and len(mux_workers()) >= 2:
            free = [w for w in mux_workers() if not W[w].resident and not W[w].pending]
            if free:
                prefill_role[free[0]] = True
                transitions[1] += 1
                delayed = 0

    def toggle_scan():
        nonlocal delayed
        if cfg.role_transitions:
            role_transitions()
        for r in list(toggle_q):
            waited = now - R[r].arrival
            target, mux = -1, 0
            # Path 2: multiplexing workers with an empty local queue, fewest unfinished tokens first
            cands = sorted((w for w in mux_workers() if not W[w].local_q), key=lambda w: (unfinished_tokens(w), w))
            for w in cands:
                dq, dc = decode_batch(w)
                t_dec = iter_time_us(cfg, dq, dc) if dq else 0.0
                if dq and not (t_dec < cfg.decode_guard * cfg.tpot_slo_us):
                    continue
                if resident_kv(w) + R[r].prompt > cfg.hbm_watermark * cfg.kv_capacity_tokens:
                    continue
                slack = INF
                for x in W[w].resident:
                    slack = min(slack, (R[x].generated + 1) * cfg.tpot_slo_us - (now - R[x].first_token))
                interference, done = 0.0, 0
                while done < R[r].prompt:
                    chunk = R[r].prompt - done if cfg.chunk_tokens <= 0 else min(R[r].prompt - done, cfg.chunk_tokens)
                    interference += iter_time_us(cfg, [chunk] + dq, [done] + dc) - t_dec
                    done += chunk
                if interference <= slack:
                    target, mux = w, 1
                    break
            if target < 0:  # Path 1, or the no-starvation rule once the TTFT slack is gone
                best = min(prefill_workers(), key=lambda w: (pred_queue(w), w))
                slack_ttft = cfg.ttft_slo_us - waited
                slack_gone = now >= R[r].arrival + cfg.ttft_slo_us  # the expression the wake-up event is scheduled with
                if slack_gone:
                    target = best
                    delayed += 1     # a delayed prefill
                elif pred_exec(r) + pred_queue(best) < slack_ttft:
                    target = best
            if target >= 0:
                toggle_q.remove(r)
                W[target].local_q.append(r)
                R[r].prefill_worker, R[r].multiplexed = target, mux

    while True:
        for w in range(cfg.num_workers):
            if W[w].busy_until <= now:
                finish_iteration(w)
        while next_arrival < len(R) and R[next_arrival].arrival <= now:
            r = next_arrival
            next_arrival += 1
            if cfg.policy == COLOCATED:
                w = min(range(cfg.num_workers), key=lambda w: (unfinished_tokens(w), w))
                W[w].local_q.append(r)
                R[r].prefill_worker = w
            elif cfg.policy == DISAGGREGATED:
                w = min(prefill_workers(), key=lambda w: (pred_queue(w), w))
                W[w].local_q.append(r)
                R[r].prefill_worker = w
            else:
                toggle_q.append(r)
        if cfg.policy == MULTIPLEXED:
            toggle_scan()
        for w in range(cfg.num_workers):
            if W[w].busy_until == INF:
                try_start(w)
        nxt = INF
        if next_arrival < len(R):
            nxt = min(nxt, R[next_arrival].arrival)
        for w in range(cfg.num_workers):
            if W[w].busy_until != INF:
                nxt = min(nxt, W[w].busy_until)
            else:
                for av, _ in W[w].pending:
                    nxt = min(nxt, av)
        for r in toggle_q:  # the moment the no-starvation rule applies
            if R[r].arrival + cfg.ttft_slo_us > now:
                nxt = min(nxt, R[r].arrival + cfg.ttft_slo_us)
        if nxt == INF:
            break
        now = nxt

    results = []
    for x in R:
        # a request the run never served violates both SLOs (guard; the model's rules serve every request)
        ttft = INF if x.first_token < 0 else x.first_token - x.arrival
        tpot = INF if x.finish < 0 else (x.finish - x.first_token) / max(1, x.output - 1)
        results.append(dict(ttft_us=ttft, tpot_us=tpot,
                            first_token_us=x.first_token, finish_us=x.finish, prefill_worker=x.prefill_worker,
                            decode_worker=x.decode_worker, multiplexed=x.multiplexed))
    summary = summarize(cfg, results, iterations)
    summary["to_multiplexing"], summary["to_prefill"] = transitions
    return results, summary


def summarize(cfg: Config, results, iterations: int):
    n = len(results)
    if n == 0:
        return dict(attainment=0.0, ttft_mean_us=0.0, ttft_p90_us=0.0, tpot_mean_us=0.0, tpot_p90_us=0.0, makespan_us=0.0,
                    iterations=iterations, multiplexed_prefills=0)
    ttft = sorted(r["ttft_us"] for r in results)
    tpot = sorted(r["tpot_us"] for r in results)
    ok = sum(1 for r in results if r["ttft_us"] <= cfg.ttft_slo_us and r["tpot_us"] <= cfg.tpot_slo_us)  # eq. (1)-(3)
    p90 = math.ceil(0.9 * n) - 1
    return dict(attainment=ok / n, ttft_mean_us=sum(ttft) / n, ttft_p90_us=ttft[p90], tpot_mean_us=sum(tpot) / n,
                tpot_p90_us=tpot[p90], makespan_us=max(r["finish_us"] for r in results), iterations=iterations,
                multiplexed_prefills=sum(r["multiplexed"] for r in results))
