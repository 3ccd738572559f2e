"""tropical_mixed_attention_static: the attention step for callers that cannot allocate device memory.

tropical_mixed_attention needs tens of MB of workspace from its caller.  A serving worker that gave all free HBM to
its KV pool at start-up, a per-iteration loop that cannot afford the device-wide synchronisation of cudaMalloc /
cudaFree, or a host program under a "no allocation after initialisation" rule has no way to provide one.  For them
the library carries a fixed 64 MiB scratch array (include/tropical.h, TROPICAL_STATIC_WORKSPACE_BYTES) and this one
entry point that uses it and allocates nothing.

What is checked here:
  * two calls in a row (a different step each time, so the second runs over what the first left in the array) give
    the outputs of the existing path -- tropical_mixed_attention with a caller workspace -- within the parity
    tolerances of the other GPU tests, and both paths sit within those tolerances of the fp64 oracle;
  * the binding takes nothing from torch's allocator during the calls (the caller passes `out`);
  * a step that needs more than the built-in array is refused with its own status before anything runs.

The file name sorts last on purpose: pytest -x stops at the first failure, so this test must not hide the others.
It has to pass in a fresh process (its first call then does the per-device set-up) and after the whole suite.
"""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import paper_2606_16264_b200 as tb
import synth
from tests.gpu_harness import MAX_ABS_TOL, MEAN_ABS_TOL, DeviceStep, errors
from paper_2606_16264_b200.harness import bf16_bits_to_f64, bits


def _mixed_step_inputs(seed, Hq, Hkv, d, q_lens, ctx_lens):
    return synth.make_step(np.random.default_rng(seed), Hq, Hkv, d, 16, q_lens, ctx_lens)


@pytest.mark.gpu
def test_static_workspace_matches_caller_workspace_on_two_calls_in_a_row():
    # call 1: prefill chunk on prior context + decode requests split over several units, GQA, d = 128;
    # call 2: another head shape and d = 64, more requests: its work lists land on top of call 1's leftovers
    steps = [
        _mixed_step_inputs(11, 16, 4, 128, [300, 1, 1, 1, 1, 17], [200, 4097, 513, 0, 15, 0]),
        _mixed_step_inputs(12, 8, 8, 64, [1] * 40 + [129, 2], [37 * (i + 1) for i in range(40)] + [0, 1000]),
    ]
    devs = []
    for s in steps:  # everything either path needs is resident before the first static call
        dev = DeviceStep(s)
        dev.append()
        dev.out_static = torch.zeros_like(dev.out)
        dev.lse_static = torch.zeros_like(dev.lse)
        devs.append(dev)
    torch.cuda.synchronize()
    reserved_before = torch.cuda.memory_reserved()

    for dev in devs:  # the two calls in a row, one stream, nothing in between
        tb.mixed_attention_static(dev.pool, dev.batch, dev.q, dev.out_static, lse=dev.lse_static)
        assert tb.last_launch_count() == 2  # tile directory + step kernel: no clearing pass, no third launch
    torch.cuda.synchronize()
    assert torch.cuda.memory_reserved() == reserved_before, "the static entry point must not take device memory"

    for s, dev in zip(steps, devs):
        dev.attention()  # the existing path: same kernels over a caller-allocated workspace
        torch.cuda.synchronize()
        got = bf16_bits_to_f64(bits(dev.out_static))
        want = dev.out_f64()
        mx, mean = errors(got, want)
        assert mx <= MAX_ABS_TOL and mean <= MEAN_ABS_TOL, (mx, mean)
        lse_got, lse_want = dev.lse_static.cpu().numpy(), dev.lse.cpu().numpy()
        assert np.abs(lse_got - lse_want).max() <= 2e-3
        # and neither is merely equal to the other: both are right
        ref_out, ref_lse, _, _ = oracle.step(s)
        mx, mean = errors(got, ref_out)
        assert mx <= MAX_ABS_TOL and mean <= MEAN_ABS_TOL, (mx, mean)
        assert np.abs(lse_got.astype(np.float64) - ref_lse).max() <= 2e-3


def test_static_workspace_refuses_a_step_beyond_its_capacity():
    """Host-side check, runs without a GPU: the size test comes before the first CUDA call."""
    L = tb.lib()
    Hq = Hkv = 64
    fake = ctypes.c_void_p(1 << 20)  # never dereferenced: the call returns before it reaches the device
    pool = tb.binding._Pool(Hq, Hkv, 128, 16, 1024, fake, fake)
    n, T = 1024, 1024
    need = L.tropical_workspace_bytes(ctypes.byref(pool), n, T, 4096)
    assert need > tb.STATIC_WORKSPACE_BYTES
    batch = tb.binding._Batch(n, T, 4096, 256, fake, fake, fake, fake)
    rc = L.tropical_mixed_attention_static(ctypes.byref(pool), ctypes.byref(batch), fake, fake, None,
                                           ctypes.c_float(0.0), None)
    assert rc == 6
    assert "static workspace" in tb.status_string(rc)
    msg = L.tropical_last_cuda_error().decode()
    assert str(need) in msg and str(tb.STATIC_WORKSPACE_BYTES) in msg
    # the five BASELINE.json configs all fit
    for cfg, (hq, hkv, d, reqs, tq) in dict(C1=(4, 4, 64, 4, 60), C2=(32, 32, 128, 64, 64), C3=(32, 32, 128, 4, 1877),
                                            C4=(40, 40, 128, 129, 2176), C5=(64, 8, 128, 258, 5376)).items():
        p = tb.binding._Pool(hq, hkv, d, 16, 64, fake, fake)
        assert 0 < L.tropical_workspace_bytes(ctypes.byref(p), reqs, tq, 100000) <= tb.STATIC_WORKSPACE_BYTES, cfg
