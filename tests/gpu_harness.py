"""Test-side re-exports + the parity tolerances."""
import numpy as np

from paper_2606_16264_b200.harness import DeviceStep, bits, to_dev  # noqa: F401


def errors(out_gpu: np.ndarray, out_ref: np.ndarray):
    d = np.abs(out_gpu - out_ref)
    return (float(d.max()), float(d.mean())) if d.size else (0.0, 0.0)


MAX_ABS_TOL = 2e-2   # BASELINE.json north_star: "max abs error 2e-2 and mean abs error 2e-3"
MEAN_ABS_TOL = 2e-3
