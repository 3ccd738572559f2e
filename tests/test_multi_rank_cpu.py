"""N > 1 path on CPU: two processes over gloo run the rank logic bench.py uses under torchrun -- every rank builds
its own replica of the workload (same lengths, private page placement and values), steps it (here: through the
CPU oracle, since there is no GPU), and the job's time is the maximum over ranks, its throughput the sum over
replicas.  The data path has no collective: the only exchange is the timing reduction."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        import oracle
        s, _ = bench.make_workload("C1", rank)
        ref, _, kp, _ = oracle.step(s)
        fake_us = 100.0 + 25.0 * rank                      # rank 1 is the slow replica
        job_us = bench.max_over_ranks(fake_us, world, "cpu")
        info = dict(rank=rank, q=s.q_lens.tolist(), c=s.ctx_lens.tolist(), table=s.page_table.tolist(),
                    checksum=float(np.abs(ref).sum()), pool_sum=int(kp.astype(np.int64).sum()), job_us=job_us,
                    tps=bench.whole_job_tokens_per_s(s.total_q, world, job_us))
        gathered = [None] * world
        dist.all_gather_object(gathered, info)
        if rank == 0:
            out.put(gathered)
    finally:
        dist.destroy_process_group()


def test_two_ranks_run_private_replicas_and_time_is_max_over_ranks():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = out.get(timeout=180)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    a, b = sorted(got, key=lambda d: d["rank"])
    assert a["q"] == b["q"] == [57, 1, 1, 1] and a["c"] == b["c"]          # same step shape on every rank (weak scaling)
    assert a["table"] != b["table"] and a["checksum"] != b["checksum"]      # private pool placement and values
    assert a["job_us"] == b["job_us"] == 125.0                              # the slowest rank sets the step time
    assert a["tps"] == pytest.approx(2 * 60 / 125e-6)                        # whole-job aggregate over both replicas


def test_single_rank_reduction_is_identity():
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_tokens_per_s(60, 1, 100.0) == pytest.approx(6e5)


def test_bench_gpus_flag_starts_that_many_ranks():
    """`python bench.py --gpus 2` with no torchrun around it starts two ranks itself (the launcher the GPU legs use;
    --rank-check swaps the GPU work for a made-up time and NCCL for gloo, everything else is the same path)."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rank-check"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints the JSON line
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["per_rank_us"] == [100.0, 125.0] and line["value"] == 125.0
    assert line["tokens_per_s"] == pytest.approx(2 * 60 / 125e-6)
    assert "rank 0 of 2" in res.stderr and "rank 1 of 2" in res.stderr


def test_bench_refuses_more_gpus_than_visible():
    import subprocess
    n = torch.cuda.device_count() if torch.cuda.is_available() else 0
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(n + 2), "--steps", "1"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert res.returncode == 2 and "refusing" in res.stderr
    assert not [l for l in res.stdout.splitlines() if l.startswith("{")]


def test_measure_allreduce_command_runs_two_ranks_and_its_fit_recovers_a_line(tmp_path):
    """NEXT-4 (TP = 2 inside a worker): the command that will measure the all-reduce term on the first box with
    two GPUs, driven here over gloo on CPU tensors (same launcher, same loop, same CSV); its rows are marked gloo and the
    fit ignores them.  The fit itself is checked on made-up NCCL rows that lie on a known line."""
    import csv
    import subprocess
    from paper_2606_16264_b200 import cost_fit
    out = tmp_path / "ar.csv"
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, "-m", "paper_2606_16264_b200.cost_fit", "measure-allreduce", "--backend", "gloo",
                          "--out", str(out), "--iters", "2", "--max-tokens", "4"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    rows = list(csv.DictReader(open(out)))
    assert [int(r["bytes"]) for r in rows] == cost_fit.allreduce_sizes(4) and len(rows) == 7   # 3 hidden sizes x T = 1, 2, 4, merged
    assert all(r["world"] == "2" and r["backend"] == "gloo" and float(r["us_median"]) > 0 for r in rows)
    assert cost_fit.read_allreduce(str(out)) == []                     # never enters a fit
    # asking for the NCCL measurement without two GPUs is refused, not degraded
    if not (torch.cuda.is_available() and torch.cuda.device_count() >= 2):
        res = subprocess.run([sys.executable, "-m", "paper_2606_16264_b200.cost_fit", "measure-allreduce", "--out", str(out)],
                             capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
        assert res.returncode == 2 and "GPUs needed" in res.stderr
    made_up = [dict(world=2, bytes=float(b), us=9.0 + 2.5e-6 * b) for b in cost_fit.allreduce_sizes(8192)]
    theta, st = cost_fit.fit_allreduce(made_up)
    assert theta[0] == pytest.approx(9.0, rel=1e-6) and theta[1] == pytest.approx(2.5e-6, rel=1e-6) and st["max"] < 1e-9
