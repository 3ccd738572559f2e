"""ctypes binding with the same names as include/tropical.h.  No arithmetic here."""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtropical.so")
_lib = None


class TropicalError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        detail = lib().tropical_last_cuda_error().decode() if status in (4, 6) else ""
        super().__init__(f"{where}: {status_string(status)} (status {status}) {detail}".strip())


class _Pool(ctypes.Structure):
    _fields_ = [("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("page_size", ctypes.c_int32), ("num_pages", ctypes.c_int32),
                ("k_pool", ctypes.c_void_p), ("v_pool", ctypes.c_void_p)]


class _Batch(ctypes.Structure):
    _fields_ = [("num_reqs", ctypes.c_int32), ("total_q", ctypes.c_int32), ("max_kv_len", ctypes.c_int32),
                ("page_table_stride", ctypes.c_int32),
                ("q_lens", ctypes.c_void_p), ("ctx_lens", ctypes.c_void_p), ("q_offsets", ctypes.c_void_p),
                ("page_table", ctypes.c_void_p)]


class CostModel(ctypes.Structure):
    _fields_ = [("t0_us", ctypes.c_double), ("a_us_per_flop", ctypes.c_double), ("b_us_per_byte", ctypes.c_double),
                ("kappa", ctypes.c_double), ("e_prefill_iter_us", ctypes.c_double),
                ("e_decode_unit_us", ctypes.c_double), ("n_sm", ctypes.c_double), ("e_prefill_crit_us", ctypes.c_double)]


class CostBreakdown(ctypes.Structure):
    _fields_ = [("flops", ctypes.c_double), ("bytes", ctypes.c_double), ("t_tc_us", ctypes.c_double),
                ("t_hbm_us", ctypes.c_double), ("prefill_tiles", ctypes.c_int64), ("prefill_iters", ctypes.c_int64),
                ("decode_units", ctypes.c_int64), ("prefill_critical_iters", ctypes.c_int64)]


class LayerShape(ctypes.Structure):
    """include/tropical.h: tropical_layer_shape_t (NEXT-4)."""
    _fields_ = [("d_model", ctypes.c_int32), ("d_ffn", ctypes.c_int32), ("gated_mlp", ctypes.c_int32),
                ("num_layers", ctypes.c_int32), ("tp", ctypes.c_int32)]


class LinearModel(ctypes.Structure):
    _fields_ = [("g0_us", ctypes.c_double), ("f_us_per_flop", ctypes.c_double), ("w_us_per_byte", ctypes.c_double),
                ("kappa", ctypes.c_double), ("ar0_us", ctypes.c_double), ("ar_us_per_byte", ctypes.c_double)]


class IterBreakdown(ctypes.Structure):
    _fields_ = [("attn_us", ctypes.c_double), ("linear_us", ctypes.c_double), ("allreduce_us", ctypes.c_double),
                ("gemm_flops", ctypes.c_double), ("gemm_bytes", ctypes.c_double), ("total_us", ctypes.c_double)]


class SimRequest(ctypes.Structure):
    _fields_ = [("arrival_us", ctypes.c_double), ("prompt_len", ctypes.c_int32), ("output_len", ctypes.c_int32)]


class SimConfig(ctypes.Structure):
    """include/tropical_sim.h: tropical_sim_config_t."""
    _fields_ = [("policy", ctypes.c_int32), ("num_workers", ctypes.c_int32), ("num_prefill_workers", ctypes.c_int32),
                ("chunk_tokens", ctypes.c_int32), ("ttft_slo_us", ctypes.c_double), ("tpot_slo_us", ctypes.c_double),
                ("decode_guard", ctypes.c_double), ("hbm_watermark", ctypes.c_double),
                ("kv_capacity_tokens", ctypes.c_int64), ("migrate_us_per_token", ctypes.c_double),
                ("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("page_size", ctypes.c_int32), ("num_layers", ctypes.c_int32), ("attn", CostModel),
                ("linear_us_per_token", ctypes.c_double), ("iter_overhead_us", ctypes.c_double),
                ("layer", LayerShape), ("linear", LinearModel), ("role_transitions", ctypes.c_int32),
                ("delay_threshold", ctypes.c_int32)]


class SimResult(ctypes.Structure):
    _fields_ = [("ttft_us", ctypes.c_double), ("tpot_us", ctypes.c_double), ("first_token_us", ctypes.c_double),
                ("finish_us", ctypes.c_double), ("prefill_worker", ctypes.c_int32), ("decode_worker", ctypes.c_int32),
                ("multiplexed", ctypes.c_int32)]


class SimSummary(ctypes.Structure):
    _fields_ = [("attainment", ctypes.c_double), ("ttft_mean_us", ctypes.c_double), ("ttft_p90_us", ctypes.c_double),
                ("tpot_mean_us", ctypes.c_double), ("tpot_p90_us", ctypes.c_double), ("makespan_us", ctypes.c_double),
                ("iterations", ctypes.c_int64), ("multiplexed_prefills", ctypes.c_int64),
                ("to_multiplexing", ctypes.c_int64), ("to_prefill", ctypes.c_int64)]


SIM_COLOCATED, SIM_DISAGGREGATED, SIM_MULTIPLEXED = 0, 1, 2

EXPORTS = (
    "tropical_kv_append", "tropical_kv_append_rope", "tropical_kv_gather", "tropical_kv_migrate", "tropical_enable_peer_access", "tropical_validate_batch", "tropical_workspace_bytes", "tropical_mixed_attention", "tropical_mixed_attention_static", "tropical_mixed_step",
    "tropical_step_host_staging_bytes", "tropical_step_host", "tropical_step_cost", "tropical_iter_cost",
    "tropical_last_launch_count", "tropical_status_string", "tropical_last_cuda_error", "tropical_version",
    "tropical_debug_attention_simt", "tropical_debug_set_grid", "tropical_debug_set_split_pages", "tropical_debug_set_fused", "tropical_debug_wait_profile", "tropical_debug_read_profile", "tropical_debug_timeline",
    "tropical_sim_run",
)


def lib():
    """Load libtropical.so; build it in-tree with nvcc when it is missing or stale.  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    try:
        path = _build.build()
    except Exception as exc:  # no silent fallback: there is no other implementation
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"libtropical.so is missing and could not be built: {exc}") from exc
        path = _LIB_PATH
    L = ctypes.CDLL(path)
    for name in EXPORTS:
        getattr(L, name)  # AttributeError here = header and library disagree
    L.tropical_workspace_bytes.restype = ctypes.c_size_t
    L.tropical_step_host_staging_bytes.restype = ctypes.c_size_t
    L.tropical_status_string.restype = ctypes.c_char_p
    L.tropical_last_cuda_error.restype = ctypes.c_char_p
    L.tropical_version.restype = ctypes.c_char_p
    if b"WHATIF" in L.tropical_version() and "WHATIF" not in os.environ.get("TROPICAL_NVCC_EXTRA", ""):
        # a measurement build whose attention results are wrong by design must be asked for, never picked up
        raise ImportError(f"{path} is a what-if measurement build ({L.tropical_version().decode()}); "
                          "rebuild without TROPICAL_NVCC_EXTRA, or set it to load this library on purpose")
    for name in ("tropical_kv_append", "tropical_kv_append_rope", "tropical_kv_gather", "tropical_kv_migrate", "tropical_enable_peer_access", "tropical_validate_batch", "tropical_mixed_attention", "tropical_mixed_attention_static", "tropical_mixed_step", "tropical_step_host",
                 "tropical_step_cost", "tropical_iter_cost", "tropical_last_launch_count", "tropical_debug_attention_simt",
                 "tropical_debug_read_profile"):
        getattr(L, name).restype = ctypes.c_int
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().tropical_status_string(int(status)).decode()


def version() -> str:
    return lib().tropical_version().decode()


def debug_set_grid(num_ctas: int) -> None:
    """Test hook: cap the CTAs of the persistent step kernel (0 = one per SM)."""
    lib().tropical_debug_set_grid(ctypes.c_int(int(num_ctas)))


def debug_set_fused(mode: int) -> None:
    """Test hook: tropical_mixed_step's kernel variant: 1 = always the fused one, 0 = never, -1 = its own choice."""
    lib().tropical_debug_set_fused(ctypes.c_int(int(mode)))


def debug_set_split_pages(pages: int) -> None:
    """Test hook: force the decode split size in pages (0 = automatic)."""
    lib().tropical_debug_set_split_pages(ctypes.c_int(int(pages)))


def debug_wait_profile(reset: bool = True):
    """{tag: (cycles, calls)} of the step kernel's mbarrier waits; None unless built with -DTROPICAL_WAIT_PROF."""
    cyc = (ctypes.c_uint64 * 512)()
    cnt = (ctypes.c_uint64 * 512)()
    rc = lib().tropical_debug_wait_profile(cyc, cnt, ctypes.c_int32(512), ctypes.c_int32(1 if reset else 0))
    if rc == 2:
        return None
    _check(rc, "tropical_debug_wait_profile")
    return {t: (int(cyc[t]), int(cnt[t])) for t in range(512) if cnt[t]}


def debug_read_profile(workspace: torch.Tensor, stream=None):
    """Role timestamps (ns, relative to kernel start) of the last fused step kernel run with `workspace`:
    dict(prefill_done, decode_done, late_decode_done); 0 = that role never ran.  None unless the library was built
    with -DTROPICAL_ROLE_PROF (the product kernel carries no stamps)."""
    out = (ctypes.c_uint64 * 4)()
    _check(lib().tropical_debug_read_profile(_ptr(_aligned(workspace)), out, _stream(stream)), "debug_read_profile")
    t0 = int(out[0])
    if t0 == 2 ** 64 - 1:  # the tile directory's initial value: nobody stamped the kernel start
        return None
    rel = lambda v: int(v) - t0 if int(v) else 0
    return {"prefill_done": rel(out[1]), "decode_done": rel(out[2]), "late_decode_done": rel(out[3])}


TIMELINE_FIELDS = ("append_start", "append_end", "plan_start", "plan_body_end", "plan_end", "step_start",
                   "step_prologue_end", "step_main_start", "step_end")


def debug_timeline(reset: bool = False):
    """{field: ns relative to the append's start} of the step(s) since the last reset; None unless built with
    -DTROPICAL_TIMELINE.  debug_timeline(reset=True) before a step, debug_timeline() after it."""
    out = (ctypes.c_uint64 * 9)()
    rc = lib().tropical_debug_timeline(None if reset else out, ctypes.c_int32(1 if reset else 0))
    if rc == 2:
        return None
    _check(rc, "tropical_debug_timeline")
    if reset:
        return {}
    # relative to the first kernel of the step: the append's start, or -- when the step has no append kernel (the fused
    # variant of tropical_mixed_step) -- the tile directory's; stamps that were never written stay out
    unset = (0, 2 ** 64 - 1)
    vals = {k: int(out[i]) for i, k in enumerate(TIMELINE_FIELDS) if int(out[i]) not in unset}
    t0 = vals.get("append_start", vals.get("plan_start", 0))
    return {k: v - t0 for k, v in vals.items()}


def last_launch_count() -> int:
    return int(lib().tropical_last_launch_count())


def _check(status: int, where: str):
    if status != 0:
        raise TropicalError(status, where)


def _ptr(t: Optional[torch.Tensor]):
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _stream(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _dev2(t: torch.Tensor, name: str):
    if not (t.is_cuda and t.is_contiguous() and t.element_size() == 2):
        raise ValueError(f"{name} must be a contiguous 2-byte (bf16) CUDA tensor")


@dataclass
class KVPool:
    """Paged KV pool: k_pool / v_pool are CUDA tensors [num_pages, Hkv, page_size, head_dim], 2-byte dtype."""
    k_pool: torch.Tensor
    v_pool: torch.Tensor
    num_q_heads: int

    def c(self) -> _Pool:
        _dev2(self.k_pool, "k_pool"); _dev2(self.v_pool, "v_pool")
        n, hkv, p, d = self.k_pool.shape
        assert tuple(self.v_pool.shape) == (n, hkv, p, d)
        return _Pool(self.num_q_heads, hkv, d, p, n, self.k_pool.data_ptr(), self.v_pool.data_ptr())


@dataclass
class Batch:
    """One multiplexed iteration; the four arrays are int32 CUDA tensors."""
    q_lens: torch.Tensor
    ctx_lens: torch.Tensor
    q_offsets: torch.Tensor
    page_table: torch.Tensor
    total_q: int
    max_kv_len: int

    @staticmethod
    def from_host(q_lens: Sequence[int], ctx_lens: Sequence[int], page_table, device="cuda") -> "Batch":
        ql = torch.as_tensor(q_lens, dtype=torch.int32)
        cl = torch.as_tensor(ctx_lens, dtype=torch.int32)
        qo = torch.zeros(ql.numel() + 1, dtype=torch.int32)
        qo[1:] = torch.cumsum(ql, 0)
        pt = torch.as_tensor(page_table, dtype=torch.int32).contiguous()
        mk = int((ql.long() + cl.long()).max()) if ql.numel() else 0
        return Batch(ql.to(device), cl.to(device), qo.to(device), pt.to(device), int(qo[-1]), mk)

    def c(self) -> _Batch:
        for t in (self.q_lens, self.ctx_lens, self.q_offsets, self.page_table):
            if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
                raise ValueError("batch arrays must be contiguous int32 CUDA tensors")
        n = self.q_lens.numel()
        stride = self.page_table.shape[1] if self.page_table.dim() == 2 else 0
        return _Batch(n, self.total_q, self.max_kv_len, stride, self.q_lens.data_ptr(), self.ctx_lens.data_ptr(),
                      self.q_offsets.data_ptr(), self.page_table.data_ptr())


def kv_append(pool: KVPool, batch: Batch, k_new: torch.Tensor, v_new: torch.Tensor, stream=None) -> None:
    _dev2(k_new, "k_new"); _dev2(v_new, "v_new")
    p, b = pool.c(), batch.c()
    _check(lib().tropical_kv_append(ctypes.byref(p), ctypes.byref(b), _ptr(k_new), _ptr(v_new), _stream(stream)),
           "tropical_kv_append")


def kv_append_rope(pool: KVPool, batch: Batch, k_new: torch.Tensor, v_new: torch.Tensor, cos: torch.Tensor,
                   sin: torch.Tensor, stream=None) -> None:
    """tropical_kv_append_rope: the append with rotate-half RoPE on the K rows; cos, sin: float32 CUDA [table_len, d/2]."""
    _dev2(k_new, "k_new"); _dev2(v_new, "v_new")
    for t, name in ((cos, "cos"), (sin, "sin")):
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.dim() == 2):
            raise ValueError(f"{name} must be a contiguous float32 CUDA tensor [table_len, d/2]")
    if cos.shape != sin.shape or cos.shape[1] * 2 != pool.k_pool.shape[3]:
        raise ValueError("cos / sin must both be [table_len, head_dim / 2]")
    p, b = pool.c(), batch.c()
    _check(lib().tropical_kv_append_rope(ctypes.byref(p), ctypes.byref(b), _ptr(k_new), _ptr(v_new), _ptr(cos), _ptr(sin),
                                         ctypes.c_int32(cos.shape[0]), _stream(stream)), "tropical_kv_append_rope")


def kv_gather(pool: KVPool, batch: Batch, req: int, n_keys: int, stream=None):
    p, b = pool.c(), batch.c()
    hkv, d = pool.k_pool.shape[1], pool.k_pool.shape[3]
    kd = torch.empty((n_keys, hkv, d), dtype=pool.k_pool.dtype, device=pool.k_pool.device)
    vd = torch.empty_like(kd)
    _check(lib().tropical_kv_gather(ctypes.byref(p), ctypes.byref(b), ctypes.c_int32(req), ctypes.c_int32(n_keys),
                                    _ptr(kd), _ptr(vd), _stream(stream)), "tropical_kv_gather")
    return kd, vd


class _Migration(ctypes.Structure):
    _fields_ = [("num_reqs", ctypes.c_int32), ("max_kv_len", ctypes.c_int32), ("src_page_table_stride", ctypes.c_int32),
                ("dst_page_table_stride", ctypes.c_int32), ("kv_lens", ctypes.c_void_p),
                ("src_page_table", ctypes.c_void_p), ("dst_page_table", ctypes.c_void_p)]


def kv_migrate(src_pool: KVPool, dst_pool: KVPool, kv_lens: torch.Tensor, src_page_table: torch.Tensor,
               dst_page_table: torch.Tensor, max_kv_len: int, stream=None) -> None:
    """KV migration (include/tropical.h: tropical_kv_migrate).  kv_lens int32 [n], page tables int32 [n, stride], all on
    the CURRENT device (the owner of src_pool); dst_pool may be on a peer device (enable_peer_access first)."""
    for t in (kv_lens, src_page_table, dst_page_table):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
            raise ValueError("migration arrays must be contiguous int32 CUDA tensors")
    sp, dp = src_pool.c(), dst_pool.c()
    n = kv_lens.numel()
    m = _Migration(n, int(max_kv_len), src_page_table.shape[1] if src_page_table.dim() == 2 else 0,
                   dst_page_table.shape[1] if dst_page_table.dim() == 2 else 0, kv_lens.data_ptr(),
                   src_page_table.data_ptr(), dst_page_table.data_ptr())
    _check(lib().tropical_kv_migrate(ctypes.byref(sp), ctypes.byref(dp), ctypes.byref(m), _stream(stream)),
           "tropical_kv_migrate")


def enable_peer_access(peer_device: int) -> bool:
    """True when peer_device's memory is (now) mapped into the current device; False when there is no peer path."""
    rc = lib().tropical_enable_peer_access(ctypes.c_int32(int(peer_device)))
    if rc == 2:
        return False
    _check(rc, "tropical_enable_peer_access")
    return True


def validate_batch(pool: KVPool, batch: Batch, scratch: Optional[torch.Tensor] = None, stream=None):
    """Opt-in debug check of the batch's device arrays (syncs).  Returns None if valid, else the first bad request.
    scratch: any CUDA tensor of >= 4 bytes (e.g. the attention workspace); allocated here when omitted."""
    bad = ctypes.c_int32(-1)
    p, b = pool.c(), batch.c()
    if scratch is None:
        scratch = torch.empty(1, dtype=torch.int32, device=batch.q_lens.device)
    rc = lib().tropical_validate_batch(ctypes.byref(p), ctypes.byref(b), ctypes.byref(bad), _ptr(scratch),
                                       _stream(stream))
    if rc == 1 and bad.value >= 0:
        return bad.value
    _check(rc, "tropical_validate_batch")
    return None


def workspace_bytes(pool: KVPool, num_reqs: int, total_q: int, max_kv_len: int) -> int:
    p = pool.c()
    return int(lib().tropical_workspace_bytes(ctypes.byref(p), ctypes.c_int32(num_reqs), ctypes.c_int32(total_q),
                                              ctypes.c_int32(max_kv_len)))


def _alloc_ws(nbytes: int, device) -> torch.Tensor:
    return torch.empty(max(nbytes, 256) + 256, dtype=torch.uint8, device=device)


def _aligned(t: torch.Tensor) -> torch.Tensor:
    off = (-t.data_ptr()) % 256
    return t[off:]


def mixed_attention(pool: KVPool, batch: Batch, q: torch.Tensor, out: Optional[torch.Tensor] = None,
                    lse: Optional[torch.Tensor] = None, sm_scale: float = 0.0,
                    workspace: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    _dev2(q, "q")
    if out is None:
        out = torch.empty_like(q)
    _dev2(out, "out")
    p, b = pool.c(), batch.c()
    if workspace is None:
        workspace = _alloc_ws(workspace_bytes(pool, b.num_reqs, b.total_q, b.max_kv_len), q.device)
    ws = _aligned(workspace)
    if lse is not None and not (lse.is_cuda and lse.dtype == torch.float32 and lse.is_contiguous()):
        raise ValueError("lse must be a contiguous float32 CUDA tensor")
    _check(lib().tropical_mixed_attention(ctypes.byref(p), ctypes.byref(b), _ptr(q), _ptr(out), _ptr(lse),
                                          ctypes.c_float(sm_scale), _ptr(ws), ctypes.c_size_t(ws.numel()),
                                          _stream(stream)), "tropical_mixed_attention")
    return out


STATIC_WORKSPACE_BYTES = 64 << 20  # TROPICAL_STATIC_WORKSPACE_BYTES in include/tropical.h


def mixed_attention_static(pool: KVPool, batch: Batch, q: torch.Tensor, out: torch.Tensor,
                           lse: Optional[torch.Tensor] = None, sm_scale: float = 0.0, stream=None) -> torch.Tensor:
    """tropical_mixed_attention_static: mixed_attention for a caller that cannot allocate a workspace.

    The scratch comes from a 64 MiB array built into the library (one per GPU, shared by all calls: do not let two
    of these calls overlap on one GPU), so nothing is allocated here either: `out` is required, not created.  A
    step that needs more than STATIC_WORKSPACE_BYTES raises TropicalError (status 6).  Make the first call on each
    device during start-up.  Details and the list of callers this is for: include/tropical.h."""
    _dev2(q, "q")
    _dev2(out, "out")
    p, b = pool.c(), batch.c()
    if lse is not None and not (lse.is_cuda and lse.dtype == torch.float32 and lse.is_contiguous()):
        raise ValueError("lse must be a contiguous float32 CUDA tensor")
    _check(lib().tropical_mixed_attention_static(ctypes.byref(p), ctypes.byref(b), _ptr(q), _ptr(out), _ptr(lse),
                                                 ctypes.c_float(sm_scale), _stream(stream)),
           "tropical_mixed_attention_static")
    return out


def mixed_step(pool: KVPool, batch: Batch, q: torch.Tensor, k_new: torch.Tensor, v_new: torch.Tensor,
               out: Optional[torch.Tensor] = None, lse: Optional[torch.Tensor] = None, sm_scale: float = 0.0,
               workspace: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """One multiplexed iteration in one call: KV append fused into the attention step (tropical_mixed_step)."""
    _dev2(q, "q")
    _dev2(k_new, "k_new")
    _dev2(v_new, "v_new")
    if out is None:
        out = torch.empty_like(q)
    _dev2(out, "out")
    p, b = pool.c(), batch.c()
    if workspace is None:
        workspace = _alloc_ws(workspace_bytes(pool, b.num_reqs, b.total_q, b.max_kv_len), q.device)
    ws = _aligned(workspace)
    if lse is not None and not (lse.is_cuda and lse.dtype == torch.float32 and lse.is_contiguous()):
        raise ValueError("lse must be a contiguous float32 CUDA tensor")
    _check(lib().tropical_mixed_step(ctypes.byref(p), ctypes.byref(b), _ptr(q), _ptr(k_new), _ptr(v_new), _ptr(out),
                                     _ptr(lse), ctypes.c_float(sm_scale), _ptr(ws), ctypes.c_size_t(ws.numel()),
                                     _stream(stream)), "tropical_mixed_step")
    return out


def debug_attention_simt(pool: KVPool, batch: Batch, q: torch.Tensor, lse: Optional[torch.Tensor] = None,
                         sm_scale: float = 0.0, stream=None) -> torch.Tensor:
    """The plain CUDA-core kernel, exposed for cross-checking the tile kernels in tests."""
    out = torch.empty_like(q)
    p, b = pool.c(), batch.c()
    _check(lib().tropical_debug_attention_simt(ctypes.byref(p), ctypes.byref(b), _ptr(q), _ptr(out), _ptr(lse),
                                               ctypes.c_float(sm_scale), _stream(stream)),
           "tropical_debug_attention_simt")
    return out


class _HostBatch(ctypes.Structure):
    _fields_ = _Batch._fields_


def step_host_staging_bytes(pool: KVPool, num_reqs: int, total_q: int, stride: int) -> int:
    p = pool.c()
    return int(lib().tropical_step_host_staging_bytes(ctypes.byref(p), ctypes.c_int32(num_reqs),
                                                      ctypes.c_int32(total_q), ctypes.c_int32(stride)))


def step_host(pool: KVPool, q_lens, ctx_lens, q_offsets, page_table, max_kv_len: int, h_q, h_k_new, h_v_new, h_out,
              staging: torch.Tensor, workspace: torch.Tensor, h_lse=None, sm_scale: float = 0.0, stream=None) -> None:
    """End-to-end step from HOST (ideally pinned) torch tensors; synchronises the stream before returning."""
    for t in (q_lens, ctx_lens, q_offsets, page_table, h_q, h_k_new, h_v_new, h_out):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("step_host takes contiguous host tensors")
    p = pool.c()
    n = q_lens.numel()
    hb = _HostBatch(n, int(h_q.shape[0]), int(max_kv_len), int(page_table.shape[1]) if page_table.dim() == 2 else 0,
                    q_lens.data_ptr(), ctx_lens.data_ptr(), q_offsets.data_ptr(), page_table.data_ptr())
    st, ws = _aligned(staging), _aligned(workspace)
    _check(lib().tropical_step_host(ctypes.byref(p), ctypes.byref(hb), _ptr(h_q), _ptr(h_k_new), _ptr(h_v_new),
                                    _ptr(h_out), _ptr(h_lse), ctypes.c_float(sm_scale), _ptr(st),
                                    ctypes.c_size_t(st.numel()), _ptr(ws), ctypes.c_size_t(ws.numel()),
                                    _stream(stream)), "tropical_step_host")


def step_cost(num_q_heads: int, num_kv_heads: int, head_dim: int, page_size: int, q_lens: Sequence[int],
              ctx_lens: Sequence[int], model: Optional[CostModel] = None, require_model: bool = True):
    """(predicted_us or None, CostBreakdown).  Host only; works without a GPU."""
    n = len(q_lens)
    ql = (ctypes.c_int32 * max(n, 1))(*[int(x) for x in q_lens])
    cl = (ctypes.c_int32 * max(n, 1))(*[int(x) for x in ctx_lens])
    us = ctypes.c_double(0.0)
    bd = CostBreakdown()
    rc = lib().tropical_step_cost(ctypes.byref(model) if model is not None else None, ctypes.c_int32(num_q_heads),
                                  ctypes.c_int32(num_kv_heads), ctypes.c_int32(head_dim), ctypes.c_int32(page_size),
                                  ctypes.c_int32(n), ql, cl, ctypes.byref(us), ctypes.byref(bd))
    if rc == 5 and not require_model:
        return None, bd
    _check(rc, "tropical_step_cost")
    return us.value, bd


def iter_cost(shape: LayerShape, num_q_heads: int, num_kv_heads: int, head_dim: int, page_size: int,
              q_lens: Sequence[int], ctx_lens: Sequence[int], attn: Optional[CostModel] = None,
              linear: Optional[LinearModel] = None):
    """(predicted us of a whole iteration, IterBreakdown): include/tropical.h tropical_iter_cost.  Host only."""
    n = len(q_lens)
    ql = (ctypes.c_int32 * max(n, 1))(*[int(x) for x in q_lens])
    cl = (ctypes.c_int32 * max(n, 1))(*[int(x) for x in ctx_lens])
    us = ctypes.c_double(0.0)
    bd = IterBreakdown()
    _check(lib().tropical_iter_cost(ctypes.byref(attn) if attn is not None else None,
                                    ctypes.byref(linear) if linear is not None else None, ctypes.byref(shape),
                                    ctypes.c_int32(num_q_heads), ctypes.c_int32(num_kv_heads), ctypes.c_int32(head_dim),
                                    ctypes.c_int32(page_size), ctypes.c_int32(n), ql, cl, ctypes.byref(us),
                                    ctypes.byref(bd)), "tropical_iter_cost")
    return us.value, bd


def sim_run(config: SimConfig, requests: Sequence[tuple]):
    """Scheduler simulation (include/tropical_sim.h).  requests: (arrival_us, prompt_len, output_len) sorted by
    arrival.  Returns (list of SimResult, SimSummary).  Host only; works without a GPU."""
    n = len(requests)
    reqs = (SimRequest * max(n, 1))(*[SimRequest(float(a), int(p), int(o)) for a, p, o in requests])
    res = (SimResult * max(n, 1))()
    summ = SimSummary()
    _check(lib().tropical_sim_run(ctypes.byref(config), ctypes.c_int32(n), reqs, res, ctypes.byref(summ)), "tropical_sim_run")
    return [res[i] for i in range(n)], summ
