"""CPU fp64 oracle for the Tropical multiplexed iteration -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports
``paper_2606_16264_b200`` and shares no code with it.  The arithmetic is in
``tropical_oracle.c`` (plain C, fp64); this file only marshals numpy arrays through ctypes.

``sim_oracle.py`` (same rules: test infrastructure only) is the plain-Python oracle of the scheduler simulation
(include/tropical_sim.h).

Citations: PAPER.md:143, :159 (the multiplexed iteration), BASELINE.json north_star (the
attention definition and tolerances), SURVEY.md section 8(c) (readings S1-S28).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tropical_oracle.c")
_LIB = os.path.join(_HERE, "libtropical_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile tropical_oracle.c -> libtropical_oracle.so (gcc, OpenMP, no fast-math)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
        _lib.oracle_attention_rows.restype = ctypes.c_int
        _lib.oracle_mixed_attention.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _u16(a) -> np.ndarray:
    a = np.asarray(a)
    assert a.dtype == np.uint16 and a.flags.c_contiguous, "bf16 tensors are passed as contiguous uint16"
    return a


def kv_append(k_pool, v_pool, q_lens, ctx_lens, q_offsets, page_table, k_new, v_new) -> None:
    """In-place append of this step's K/V rows into the pools (tropical_oracle.c: oracle_kv_append)."""
    k_pool, v_pool, k_new, v_new = _u16(k_pool), _u16(v_pool), _u16(k_new), _u16(v_new)
    assert k_pool.flags.writeable and v_pool.flags.writeable
    _, Hkv, P, d = k_pool.shape
    q_lens, ctx_lens, q_offsets, page_table = _i32(q_lens), _i32(ctx_lens), _i32(q_offsets), _i32(page_table)
    _load().oracle_kv_append(
        ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(P), ctypes.c_int(q_lens.shape[0]),
        _p(q_lens), _p(ctx_lens), _p(q_offsets), _p(page_table), ctypes.c_int(page_table.shape[1]),
        _p(k_pool), _p(v_pool), _p(k_new), _p(v_new))


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def rope_rotate(rows, pos, cos, sin) -> np.ndarray:
    """fp64 rotate-half RoPE of bf16 rows [n, d] at positions pos [n] with tables cos, sin [table_len, d/2] (fp32 values);
    unrounded (tropical_oracle.c: oracle_rope_rotate)."""
    rows, cos, sin = _u16(rows), _f32(cos), _f32(sin)
    n, d = rows.shape
    assert cos.shape == sin.shape and cos.shape[1] == d // 2
    pos = _i32(pos)
    assert pos.shape == (n,) and (n == 0 or (0 <= pos.min() and pos.max() < cos.shape[0]))
    out = np.empty((n, d), np.float64)
    _load().oracle_rope_rotate(ctypes.c_int(d), ctypes.c_int64(n), _p(rows), _p(pos), _p(cos), _p(sin), _p(out))
    return out


def double_to_bf16(values) -> np.ndarray:
    """fp64 -> bf16 bit patterns, round to nearest even straight from the double (oracle_double_to_bf16)."""
    lib = _load()
    lib.oracle_double_to_bf16.restype = ctypes.c_uint16
    v = np.ascontiguousarray(values, np.float64)
    return np.array([lib.oracle_double_to_bf16(ctypes.c_double(float(x))) for x in v.ravel()], np.uint16).reshape(v.shape)


def kv_append_rope(k_pool, v_pool, q_lens, ctx_lens, q_offsets, page_table, k_new, v_new, cos, sin) -> None:
    """In-place append with rotate-half RoPE applied to the K rows (oracle_kv_append_rope); V rows are copied."""
    k_pool, v_pool, k_new, v_new = _u16(k_pool), _u16(v_pool), _u16(k_new), _u16(v_new)
    assert k_pool.flags.writeable and v_pool.flags.writeable
    _, Hkv, P, d = k_pool.shape
    cos, sin = _f32(cos), _f32(sin)
    q_lens, ctx_lens, q_offsets, page_table = _i32(q_lens), _i32(ctx_lens), _i32(q_offsets), _i32(page_table)
    need = int((q_lens.astype(np.int64) + ctx_lens).max()) if q_lens.size else 0
    assert cos.shape == sin.shape and cos.shape[1] == d // 2 and cos.shape[0] >= need
    _load().oracle_kv_append_rope(
        ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(P), ctypes.c_int(q_lens.shape[0]),
        _p(q_lens), _p(ctx_lens), _p(q_offsets), _p(page_table), ctypes.c_int(page_table.shape[1]),
        _p(k_pool), _p(v_pool), _p(k_new), _p(v_new), _p(cos), _p(sin))


def kv_gather(k_pool, v_pool, page_table, req: int, n_keys: int) -> Tuple[np.ndarray, np.ndarray]:
    """Dense bf16 copy-out [n_keys, Hkv, d] of request req's first n_keys keys/values."""
    k_pool, v_pool = _u16(k_pool), _u16(v_pool)
    _, Hkv, P, d = k_pool.shape
    page_table = _i32(page_table)
    kd = np.empty((n_keys, Hkv, d), np.uint16)
    vd = np.empty((n_keys, Hkv, d), np.uint16)
    _load().oracle_kv_gather(
        ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(P), _p(page_table),
        ctypes.c_int(page_table.shape[1]), ctypes.c_int(req), ctypes.c_int(n_keys),
        _p(k_pool), _p(v_pool), _p(kd), _p(vd))
    return kd, vd


def kv_migrate(k_src, v_src, k_dst, v_dst, kv_lens, src_page_table, dst_page_table) -> None:
    """In-place migration of the first kv_lens[m] tokens of every request m from the source pools (through
    src_page_table) into the destination pools (under dst_page_table): tropical_oracle.c: oracle_kv_migrate."""
    k_src, v_src, k_dst, v_dst = _u16(k_src), _u16(v_src), _u16(k_dst), _u16(v_dst)
    assert k_dst.flags.writeable and v_dst.flags.writeable
    _, Hkv, P, d = k_src.shape
    assert k_dst.shape[1:] == (Hkv, P, d)
    kv_lens, src_page_table, dst_page_table = _i32(kv_lens), _i32(src_page_table), _i32(dst_page_table)
    _load().oracle_kv_migrate(
        ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(P), ctypes.c_int(kv_lens.shape[0]), _p(kv_lens),
        _p(src_page_table), ctypes.c_int(src_page_table.shape[1]), _p(dst_page_table),
        ctypes.c_int(dst_page_table.shape[1]), _p(k_src), _p(v_src), _p(k_dst), _p(v_dst))


def attention_rows(k_pool, v_pool, q, q_lens, ctx_lens, q_offsets, page_table,
                   rows: Sequence[Tuple[int, int]], sm_scale: float = 0.0, want_wsum: bool = False):
    """fp64 attention for chosen (request, new-token index) rows; all q heads of each row.

    Returns (out [n, Hq, d] f64, lse [n, Hq] f64[, wsum [n, Hq] f64])."""
    k_pool, v_pool, q = _u16(k_pool), _u16(v_pool), _u16(q)
    _, Hkv, P, d = k_pool.shape
    Hq = q.shape[1]
    q_lens, ctx_lens, q_offsets, page_table = _i32(q_lens), _i32(ctx_lens), _i32(q_offsets), _i32(page_table)
    rows = list(rows)
    n = len(rows)
    row_req = _i32([r for r, _ in rows])
    row_t = _i32([t for _, t in rows])
    for r, t in rows:
        assert 0 <= r < q_lens.shape[0] and 0 <= t < q_lens[r], (r, t)
    out = np.zeros((n, Hq, d), np.float64)
    lse = np.zeros((n, Hq), np.float64)
    wsum = np.zeros((n, Hq), np.float64) if want_wsum else None
    rc = _load().oracle_attention_rows(
        ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(P),
        _p(q_lens), _p(ctx_lens), _p(q_offsets), _p(page_table), ctypes.c_int(page_table.shape[1]),
        _p(k_pool), _p(v_pool), _p(q), ctypes.c_double(sm_scale), ctypes.c_int(n),
        _p(row_req), _p(row_t), _p(out), _p(lse), _p(wsum))
    if rc != 0:
        raise MemoryError("oracle scratch allocation failed")
    return (out, lse, wsum) if want_wsum else (out, lse)


def mixed_attention(k_pool, v_pool, q, q_lens, ctx_lens, q_offsets, page_table,
                    sm_scale: float = 0.0, want_wsum: bool = False):
    """fp64 attention for every row of the step (pools must already hold this step's rows).

    Returns (out [T, Hq, d] f64, lse [T, Hq] f64[, wsum])."""
    k_pool, v_pool, q = _u16(k_pool), _u16(v_pool), _u16(q)
    _, Hkv, P, d = k_pool.shape
    T, Hq = q.shape[0], q.shape[1]
    q_lens, ctx_lens, q_offsets, page_table = _i32(q_lens), _i32(ctx_lens), _i32(q_offsets), _i32(page_table)
    assert int(q_offsets[-1]) == T
    out = np.zeros((T, Hq, d), np.float64)
    lse = np.zeros((T, Hq), np.float64)
    wsum = np.zeros((T, Hq), np.float64) if want_wsum else None
    rc = _load().oracle_mixed_attention(
        ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(d), ctypes.c_int(P), ctypes.c_int(q_lens.shape[0]),
        _p(q_lens), _p(ctx_lens), _p(q_offsets), _p(page_table), ctypes.c_int(page_table.shape[1]),
        _p(k_pool), _p(v_pool), _p(q), ctypes.c_double(sm_scale), _p(out), _p(lse), _p(wsum))
    if rc != 0:
        raise MemoryError("oracle scratch allocation failed")
    return (out, lse, wsum) if want_wsum else (out, lse)


def step(inputs, sm_scale: float = 0.0):
    """Whole step on a synth.StepInputs: append into COPIES of the pools, then attend.

    Returns (out f64 [T,Hq,d], lse f64 [T,Hq], k_pool_after, v_pool_after)."""
    kp, vp = inputs.copy_pools()
    kv_append(kp, vp, inputs.q_lens, inputs.ctx_lens, inputs.q_offsets, inputs.page_table,
              inputs.k_new, inputs.v_new)
    out, lse = mixed_attention(kp, vp, inputs.q, inputs.q_lens, inputs.ctx_lens, inputs.q_offsets,
                               inputs.page_table, sm_scale)
    return out, lse, kp, vp
