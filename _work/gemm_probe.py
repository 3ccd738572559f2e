"""Linear-layer time of one transformer layer on the B200 as a function of the iteration's token count (SURVEY 8(f)
NEXT-4, first step): the non-attention part of an iteration, which the scheduler simulation (simulate.py) adds to
the step-cost model.  Library GEMMs (torch.matmul -> cuBLAS, bf16) on the 13B-like shape of C4 (d_model 5120 =
40 heads x 128, FFN 13824, gated MLP); this is calibration data, not a kernel of this repository.

    python -m paper_2606_16264_b200.gemm_probe [--out calibration/b200_gemm.csv]
"""
from __future__ import annotations

import argparse
import csv
import os

HERE = os.path.dirname(os.path.abspath(__file__))
D_MODEL, D_FFN = 5120, 13824
TOKENS = [1, 8, 32, 64, 128, 256, 512, 1024, 2048, 4096, 8192]


def main(argv=None):
    import torch
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(HERE, "calibration", "b200_gemm.csv"))
    a = ap.parse_args(argv)
    dev = torch.device("cuda")
    w = [torch.randn(D_MODEL, 3 * D_MODEL, device=dev, dtype=torch.bfloat16),   # QKV
         torch.randn(D_MODEL, D_MODEL, device=dev, dtype=torch.bfloat16),       # O
         torch.randn(D_MODEL, 2 * D_FFN, device=dev, dtype=torch.bfloat16),     # gate + up
         torch.randn(D_FFN, D_MODEL, device=dev, dtype=torch.bfloat16)]         # down
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    rows = []
    for T in TOKENS:
        x = torch.randn(T, D_MODEL, device=dev, dtype=torch.bfloat16)
        h = torch.randn(T, D_FFN, device=dev, dtype=torch.bfloat16)

        def layer():
            torch.matmul(x, w[0])
            torch.matmul(x, w[1])
            torch.matmul(x, w[2])
            torch.matmul(h, w[3])

        for _ in range(3):
            layer()
        times = []
        for k in range(20):
            flush.fill_(k)  # weights of a real model do not stay in L2 between layers
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            layer()
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1) * 1e3)
        times.sort()
        rows.append([T, round(times[len(times) // 2], 2), round(times[0], 2)])
        print(rows[-1])
    os.makedirs(os.path.dirname(os.path.abspath(a.out)), exist_ok=True)
    with open(a.out, "w", newline="") as f:
        wr = csv.writer(f)
        wr.writerow(["tokens", "layer_gemm_us_median", "layer_gemm_us_min"])
        wr.writerows(rows)


if __name__ == "__main__":
    main()
