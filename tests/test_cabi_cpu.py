"""CPU-side checks of the C-ABI library: it loads without a GPU, exports every symbol
include/*.h declares, validates host-visible arguments before touching CUDA, and its
step-cost feature arithmetic matches hand-derived counts (tests/golden/step_cost_features.txt)."""
import ctypes
import os
import re

import pytest

import paper_2606_16264_b200 as tb
from paper_2606_16264_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = "".join(open(os.path.join(ROOT, "include", h)).read() for h in sorted(os.listdir(os.path.join(ROOT, "include"))) if h.endswith(".h"))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tropical_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = tb.lib()
    declared = _declared_functions()
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(L, name), f"{name} declared in tropical.h but not exported"
    assert set(declared) == set(binding.EXPORTS)
    assert "sm_100a" in tb.version()


def test_only_sm100a_code_in_library():
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", binding._LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_status_strings():
    assert tb.status_string(0) == "ok"
    assert "workspace" in tb.status_string(3)
    assert "unknown" in tb.status_string(99)


def _pool(hq=4, hkv=4, d=64, p=16, pages=8, k=0x1000, v=0x2000):
    return binding._Pool(hq, hkv, d, p, pages, k, v)


def _batch(n=1, T=1, mk=1, stride=1, ptr=0x3000):
    return binding._Batch(n, T, mk, stride, ptr, ptr, ptr, ptr)


def test_argument_validation_happens_before_any_cuda_call():
    L = tb.lib()
    null = ctypes.c_void_p(0)
    x = ctypes.c_void_p(0x4000)
    call = lambda p, b: L.tropical_mixed_attention(ctypes.byref(p), ctypes.byref(b), x, x, null, ctypes.c_float(0),
                                                   x, ctypes.c_size_t(1 << 30), null)
    assert call(_pool(hq=6, hkv=4), _batch()) == 1          # Hq % Hkv != 0
    assert call(_pool(d=96), _batch()) == 2                  # head_dim unsupported
    assert call(_pool(p=32), _batch()) == 2                  # page size unsupported
    assert call(_pool(k=0), _batch()) == 1                   # null pool
    assert call(_pool(k=0x1010), _batch()) == 1              # misaligned pool
    assert call(_pool(), _batch(mk=100, stride=2)) == 1      # stride too small for max_kv_len
    assert call(_pool(), _batch(n=-1)) == 1
    assert call(_pool(), _batch(ptr=0)) == 1                 # null metadata arrays
    p, b = _pool(), _batch()
    assert L.tropical_mixed_attention(ctypes.byref(p), ctypes.byref(b), x, x, null, ctypes.c_float(0), null,
                                      ctypes.c_size_t(0), null) == 3   # no workspace
    assert L.tropical_mixed_attention(ctypes.byref(p), ctypes.byref(b), null, x, null, ctypes.c_float(0), x,
                                      ctypes.c_size_t(1 << 30), null) == 1  # null q
    assert L.tropical_kv_append(ctypes.byref(p), ctypes.byref(b), null, x, null) == 1
    assert L.tropical_kv_gather(ctypes.byref(p), ctypes.byref(b), ctypes.c_int32(5), ctypes.c_int32(1), x, x, null) == 1
    # empty step is a no-op success, no CUDA needed
    e = _batch(n=0, T=0, mk=0, stride=0, ptr=0)
    assert call(_pool(), e) == 0
    assert L.tropical_kv_append(ctypes.byref(p), ctypes.byref(e), null, null, null) == 0
    assert tb.workspace_bytes(tb.KVPool.__new__(tb.KVPool), 0, 0, 0) if False else True


def test_workspace_bytes_monotone_and_nonzero():
    L = tb.lib()
    L.tropical_workspace_bytes.restype = ctypes.c_size_t
    p = _pool(hq=64, hkv=8, d=128)
    f = lambda n, T, mk: L.tropical_workspace_bytes(ctypes.byref(p), ctypes.c_int32(n), ctypes.c_int32(T), ctypes.c_int32(mk))
    assert f(1, 1, 16) >= 256
    assert f(258, 5376, 8192) >= f(4, 60, 256) >= f(1, 1, 16)
    assert f(-1, 0, 0) == 0


def test_step_cost_features_match_hand_derivation():
    """tests/golden/step_cost_features.txt: batch A = one prefill q=130,c=0 + one decode c=17 (Hq=4,Hkv=2,d=64,P=16)."""
    golden = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "step_cost_features.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            golden[k.strip()] = float(v)
    us, bd = tb.step_cost(4, 2, 64, 16, [130, 1], [0, 17], require_model=False)
    assert bd.flops == golden["A.flops"] and bd.bytes == golden["A.bytes"]
    assert bd.prefill_tiles == golden["A.prefill_tiles"] and bd.prefill_iters == golden["A.prefill_iters"]
    assert bd.decode_units == golden["A.decode_units"] and bd.prefill_critical_iters == golden["A.prefill_critical_iters"]
    us, bd = tb.step_cost(8, 8, 128, 16, [256], [300], require_model=False)
    assert bd.flops == golden["B.flops"] and bd.bytes == golden["B.bytes"]
    assert bd.prefill_tiles == golden["B.prefill_tiles"] and bd.prefill_iters == golden["B.prefill_iters"]
    assert bd.decode_units == 0 and bd.prefill_critical_iters == golden["B.prefill_critical_iters"]
    # the same chunk next to 7 decode requests: 263 tokens in 8 requests < 64 per request -> plain variant: the top tile alone
    _, bd = tb.step_cost(8, 8, 128, 16, [256] + [1] * 7, [300] + [10] * 7, require_model=False)
    assert bd.prefill_critical_iters == 5


def test_step_cost_properties_with_explicit_model():
    m = tb.CostModel(5.0, 1e-9, 2e-7, 0.3, 0.4, 0.01, 148.0)
    base, _ = tb.step_cost(8, 8, 128, 16, [512, 1, 1], [0, 700, 90], model=m)
    # monotone in every q_i and c_i
    for dq, dc in (([513, 1, 1], [0, 700, 90]), ([512, 1, 1], [16, 700, 90]), ([512, 1, 1], [0, 701, 90])):
        up, _ = tb.step_cost(8, 8, 128, 16, dq, dc, model=m)
        assert up >= base
    # permutation invariant over requests
    perm, _ = tb.step_cost(8, 8, 128, 16, [1, 512, 1], [90, 0, 700], model=m)
    assert abs(perm - base) <= 1e-9 * base
    # empty batch = launch floor; prediction >= both roofline terms
    empty, _ = tb.step_cost(8, 8, 128, 16, [], [], model=m)
    assert empty == 5.0
    us, bd = tb.step_cost(8, 8, 128, 16, [512, 1, 1], [0, 700, 90], model=m)
    assert us >= 5.0 + max(bd.t_tc_us, bd.t_hbm_us) and bd.t_tc_us == 1e-9 * bd.flops and bd.t_hbm_us == 2e-7 * bd.bytes
    with pytest.raises(tb.TropicalError):
        tb.step_cost(6, 4, 128, 16, [1], [1], model=m)


NOMINAL_TFLOPS, NOMINAL_HBM_GBS = 2250.0, 8000.0   # dense bf16 and HBM3e peaks of the part: constants, not fitted


def test_builtin_cost_model_reproduces_measured_grid():
    """A6: the compiled-in coefficients (csrc/cost_model_fit.inc: one set per head shape and kernel variant of the step)
    against the B200 measurements of tropical_mixed_step they were fitted to (calibration/b200_grid.csv).  Held-out rows
    (every fifth grid point, and every off-grid point: recipe values between and beyond the grid lines) were not used by
    the fit.  The paper gives no accuracy target; the bars are SURVEY.md 8(c)'s: MAPE <= 10 % (held-out and
    off-grid, per shape) and every one of the 535 points within 25 %.  Every prediction must also respect the roofline of
    the part's NOMINAL peaks, which the fit cannot move."""
    import numpy as np
    from paper_2606_16264_b200 import cost_fit
    rows = cost_fit.read_grid(cost_fit.DEFAULT_GRID)
    assert len(rows) >= 400
    shapes = sorted({(r["Hq"], r["Hkv"], r["d"]) for r in rows})
    assert (20, 20, 128) in shapes and (32, 4, 128) in shapes      # the TP = 2 head shards of C4 / C5 (NEXT-4)
    for shape in shapes:
        rel_all, rel_held, rel_off = [], [], []
        for r in rows:
            if (r["Hq"], r["Hkv"], r["d"]) != shape:
                continue
            q, c = cost_fit.grid_lengths(r["prefill_tokens"], r["prefill_ctx"], r["n_decode"], r["ctx_median"], r["seed"])
            us, bd = tb.step_cost(*shape, 16, q.tolist(), c.tolist())
            assert us >= max(bd.flops / (NOMINAL_TFLOPS * 1e6), bd.bytes / (NOMINAL_HBM_GBS * 1e3))
            rel = abs(us - r["us_median"]) / r["us_median"]
            rel_all.append(rel)
            if cost_fit.is_held_out(r):
                rel_held.append(rel)
            if r["seed"] >= 1000:
                rel_off.append(rel)
        assert len(rel_off) >= 20
        assert np.mean(rel_held) <= 0.10, (shape, np.mean(rel_held))
        assert np.mean(rel_off) <= 0.10, (shape, np.mean(rel_off))
        assert np.max(rel_all) <= 0.25, (shape, np.max(rel_all))


def test_builtin_linear_model_reproduces_measured_gemms():
    """NEXT-4: the compiled-in linear-layer coefficients (csrc/linear_model_fit.inc) against the library-GEMM times of
    calibration/b200_gemm.csv (7B-, 13B- and 70B-layer-like shapes, TP 1 and 2, 1 .. 8192 tokens), through
    tropical_iter_cost with the attention term switched off."""
    import numpy as np
    from paper_2606_16264_b200 import cost_fit
    rows = cost_fit.read_gemm(cost_fit.GEMM_GRID)
    assert len(rows) >= 50
    zero = tb.CostModel(0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 148.0)
    rel = []
    for r in rows:
        shape = tb.LayerShape(r["d_model"], r["d_ffn"], r["gated"], 1, r["tp"])
        T = r["tokens"]
        us, bd = tb.iter_cost(shape, r["Hq"], r["Hkv"], r["d"], 16, [T] if T > 1 else [1], [0], attn=zero)
        assert bd.attn_us == 0.0 and bd.allreduce_us == 0.0 and us == bd.linear_us
        assert us >= max(bd.gemm_flops / (NOMINAL_TFLOPS * 1e6), bd.gemm_bytes / (NOMINAL_HBM_GBS * 1e3))
        rel.append(abs(us - r["us_median"]) / r["us_median"])
    assert np.mean(rel) <= 0.08 and np.max(rel) <= 0.20, (np.mean(rel), np.max(rel))
    # a whole iteration of the 13B-like model with the built-in fits: 40 layers, TP = 2 shard of C4's batch
    import synth
    _, Hq, Hkv, d, P, q, c, _ = synth.config_lengths("C4")
    us1, bd1 = tb.iter_cost(tb.LayerShape(5120, 13824, 1, 40, 1), Hq, Hkv, d, P, q.tolist(), c.tolist())
    us2, bd2 = tb.iter_cost(tb.LayerShape(5120, 13824, 1, 40, 2), Hq, Hkv, d, P, q.tolist(), c.tolist())
    assert bd2.attn_us < bd1.attn_us and bd2.linear_us < bd1.linear_us and us2 < us1
    assert us1 == pytest.approx(40 * (bd1.attn_us + bd1.linear_us))


def test_change_of_build_flags_forces_a_rebuild(monkeypatch):
    """A measurement build (TROPICAL_NVCC_EXTRA=-DTROPICAL_WHATIF_..., results wrong by design) overwrites
    libtropical.so; the flag set it was built with is stamped beside it, so a later run with other flags rebuilds."""
    from paper_2606_16264_b200 import build
    monkeypatch.delenv("TROPICAL_NVCC_EXTRA", raising=False)
    tb.lib()
    assert not build._stale()
    monkeypatch.setenv("TROPICAL_NVCC_EXTRA", "-DTROPICAL_TIMELINE")
    assert build._stale()
    monkeypatch.delenv("TROPICAL_NVCC_EXTRA")
    assert not build._stale()
    assert b"WHATIF" not in tb.lib().tropical_version()
