"""Row A6 checked live on whatever box runs the suite ("highly predictable"; the scheduler
acts on predicted step times).  The built-in step-cost fits were made from a grid measured on one B200
(calibration/b200_grid.csv); tests/test_cabi_cpu.py only compares them with that file.  Here fifteen points that are on
no grid line -- three native head shapes, both kernel variants of tropical_mixed_step -- are timed through the product
call and compared with tropical_step_cost.  Boxes of this pool differ by ~6 % (clocks, HBM stacks): the comparison is
made on ratios to a decode-only anchor step measured in the same test on the same shape.
Bars: SURVEY.md 8(c) step-cost model: mean absolute percentage error <= 10 %, every point within 25 %.
The file name sorts after the parity tests on purpose: this is a timing test, and pytest -x must not let a slow box hide them."""
import numpy as np
import pytest

import paper_2606_16264_b200 as tb
from paper_2606_16264_b200 import cost_fit

pytestmark = pytest.mark.gpu

SHAPES = [(32, 32, 128), (40, 40, 128), (64, 8, 128)]
ANCHOR = (0, 0, 64, 1000, 5000)           # (prefill tokens, prior context of the chunk, decode requests, ctx median, seed)
POINTS = [
    (1200, 0, 0, 0, 5001),                # prefill only, short prompt                       -> fused variant
    (3000, 1024, 20, 900, 5002),          # chunk on prior context + a few decodes            -> fused variant
    (0, 0, 200, 1800, 5003),              # decode only                                       -> plain variant
    (500, 0, 150, 1200, 5004),            # short prefill beside a decode batch               -> plain variant
    (5000, 0, 300, 600, 5005),            # two chunks beside a large decode batch            -> plain variant
]


def live_errors(iters=20):
    """[(shape, point, measured_us, predicted_us, relative error of the anchored prediction)]"""
    rows = []
    pts = [ANCHOR] + POINTS
    scale = {}
    for Hq, Hkv, d, p, step in cost_fit._points_on_device(SHAPES, pts):
        q, c = cost_fit.grid_lengths(*p)
        meas = float(np.median(cost_fit._time_us(step, iters)))
        pred = tb.step_cost(Hq, Hkv, d, 16, q.tolist(), c.tolist())[0]
        if p == ANCHOR:
            scale[(Hq, Hkv, d)] = meas / pred   # this box against the calibration box, on a bandwidth-bound step
            continue
        anchored = pred * scale[(Hq, Hkv, d)]
        rows.append(((Hq, Hkv, d), p, meas, pred, (anchored - meas) / meas))
    return rows, scale


def test_builtin_step_cost_against_live_step_times():
    rows, scale = live_errors()
    assert len(rows) == len(SHAPES) * len(POINTS)
    for s, k in scale.items():
        assert 0.8 <= k <= 1.25, f"anchor step of {s} is {k:.2f}x its prediction: this box is not the model's"
    rel = np.array([abs(r[4]) for r in rows])
    detail = "\n".join(f"{r[0]} {r[1]} measured {r[2]:.1f} us predicted {r[3]:.1f} us anchored error {r[4]:+.1%}" for r in rows)
    assert rel.mean() <= 0.10, detail
    assert rel.max() <= 0.25, detail
