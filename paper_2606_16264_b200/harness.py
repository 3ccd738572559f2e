"""Device-resident copy of one step's inputs + convenience calls (marshalling only, no arithmetic).

Takes any object with the fields of synth.StepInputs (duck-typed; this package does not import synth
or oracle).  Used by tests/, bench.py and __graft_entry__.smoke()."""
from __future__ import annotations

import numpy as np
import torch

from . import binding as tb


def to_dev(a: np.ndarray) -> torch.Tensor:
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).cuda()
    return torch.from_numpy(a).cuda()


def bits(t: torch.Tensor) -> np.ndarray:
    """2-byte tensor -> numpy uint16 bit patterns on the host."""
    return t.detach().cpu().numpy().view(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


class DeviceStep:
    def __init__(self, s):
        self.s = s
        self.k_pool, self.v_pool = to_dev(s.k_pool), to_dev(s.v_pool)
        self.pool = tb.KVPool(self.k_pool, self.v_pool, s.num_q_heads)
        self.batch = tb.Batch(to_dev(s.q_lens), to_dev(s.ctx_lens), to_dev(s.q_offsets), to_dev(s.page_table),
                              s.total_q, s.max_kv_len)
        self.q, self.k_new, self.v_new = to_dev(s.q), to_dev(s.k_new), to_dev(s.v_new)
        nbytes = tb.workspace_bytes(self.pool, s.num_reqs, s.total_q, s.max_kv_len)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        self.out = torch.zeros_like(self.q)
        self.lse = torch.zeros((s.total_q, s.num_q_heads), dtype=torch.float32, device="cuda")

    def append(self):
        tb.kv_append(self.pool, self.batch, self.k_new, self.v_new)

    def attention(self, sm_scale=0.0, impl="product"):
        if impl == "simt":
            self.out = tb.debug_attention_simt(self.pool, self.batch, self.q, lse=self.lse, sm_scale=sm_scale)
        else:
            tb.mixed_attention(self.pool, self.batch, self.q, out=self.out, lse=self.lse, sm_scale=sm_scale,
                               workspace=self.workspace)
        return self.out

    def fused_step(self, sm_scale=0.0):
        """tropical_mixed_step: the append fused into the attention step (one call)."""
        tb.mixed_step(self.pool, self.batch, self.q, self.k_new, self.v_new, out=self.out, lse=self.lse,
                      sm_scale=sm_scale, workspace=self.workspace)
        return self.out

    def step(self, sm_scale=0.0, impl="fused"):
        """One iteration, synchronised; returns (out f64 [T,Hq,d], lse f64 [T,Hq]) on the host.  impl "fused": the single
        call tropical_mixed_step with its fused kernel variant forced (append inside the step kernel); "auto": the same
        call with its own choice of variant; "product" / "simt": tropical_kv_append followed by the attention call."""
        if impl in ("fused", "auto"):
            tb.debug_set_fused(1 if impl == "fused" else -1)
            try:
                self.fused_step(sm_scale)
            finally:
                tb.debug_set_fused(-1)
        else:
            self.append()
            self.attention(sm_scale, impl)
        torch.cuda.synchronize()
        return self.out_f64(), self.lse.cpu().numpy().astype(np.float64)

    def out_f64(self) -> np.ndarray:
        return bf16_bits_to_f64(bits(self.out))
