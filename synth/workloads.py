"""Seeded generators for one multiplexed iteration (a prefill
chunk piggy-backed on the running decode batch of one worker).

Notation: request i has q_i new tokens this step (1 = decode
token, >= 2 = prefill chunk, 0 = skipped), c_i tokens already in the cache,
L_i = c_i + q_i.  T = sum q_i.  Hq / Hkv query / kv heads, d head dim, P page size.

Layouts produced (all host numpy, bf16 carried as uint16 bit patterns):
  q            uint16 [T, Hq, d]        request-major ragged rows
  k_new, v_new uint16 [T, Hkv, d]
  k_pool/v_pool uint16 [num_pages, Hkv, P, d]   ("HND": one (page, head) is contiguous)
  page_table   int32  [num_reqs, stride]        entries past ceil(L_i/P) are -1
  q_lens, ctx_lens int32 [num_reqs];  q_offsets int32 [num_reqs + 1]

No attention / softmax / append arithmetic lives here.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np

POISON_BF16 = 0x7FC0  # quiet-NaN bf16 pattern written to every unused pool slot

CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")


# ----------------------------------------------------------------------------- bf16 helpers
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even.  Finite inputs only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounded = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return rounded.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> float32 (exact)."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


# ----------------------------------------------------------------------------- containers
@dataclasses.dataclass
class StepInputs:
    name: str
    seed: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    num_pages: int
    q_lens: np.ndarray
    ctx_lens: np.ndarray
    q_offsets: np.ndarray
    page_table: np.ndarray
    k_pool: np.ndarray
    v_pool: np.ndarray
    q: np.ndarray
    k_new: np.ndarray
    v_new: np.ndarray

    @property
    def num_reqs(self) -> int:
        return int(self.q_lens.shape[0])

    @property
    def total_q(self) -> int:
        return int(self.q_offsets[-1])

    @property
    def max_kv_len(self) -> int:
        if self.num_reqs == 0:
            return 0
        return int((self.q_lens.astype(np.int64) + self.ctx_lens).max())

    @property
    def page_table_stride(self) -> int:
        return int(self.page_table.shape[1])

    def copy_pools(self):
        return self.k_pool.copy(), self.v_pool.copy()


def needed_pages(q_lens: Sequence[int], ctx_lens: Sequence[int], page_size: int) -> int:
    return int(sum((int(q) + int(c) + page_size - 1) // page_size for q, c in zip(q_lens, ctx_lens)))


# ----------------------------------------------------------------------------- lengths of C1..C5
def _lognormal_lengths(rng, n, median, sigma, lo, hi):
    z = rng.standard_normal(n)
    return np.clip(np.rint(np.exp(math.log(median) + sigma * z)), lo, hi).astype(np.int64)


def config_lengths(name: str):
    """(seed, Hq, Hkv, d, P, q_lens, ctx_lens, rng) for BASELINE.json configs[0..4].

    The returned rng has consumed exactly the length draws, so that make_config continues
    with the page permutation and then the values (draw order fixed by SURVEY.md 8(d))."""
    if name == "C1":  # tiny mixed step
        seed, Hq, Hkv, d = 0, 4, 4, 64
        rng = np.random.default_rng(seed)
        q = [57, 1, 1, 1]
        c = [0, 17, 100, 255]
    elif name == "C2":  # decode-only, 7B-like MHA
        seed, Hq, Hkv, d = 1, 32, 32, 128
        rng = np.random.default_rng(seed)
        c = rng.integers(512, 2049, 64).tolist()
        q = [1] * 64
    elif name == "C3":  # prefill-only, 7B-like MHA
        seed, Hq, Hkv, d = 2, 32, 32, 128
        rng = np.random.default_rng(seed)
        q = _lognormal_lengths(rng, 4, 700, 0.8, 64, 4096).tolist()
        c = [0] * 4
    elif name == "C4":  # multiplexed mixed step, 13B-like MHA
        seed, Hq, Hkv, d = 3, 40, 40, 128
        rng = np.random.default_rng(seed)
        cd = _lognormal_lengths(rng, 128, 1000, 0.9, 64, 4096).tolist()
        q = [2048] + [1] * 128
        c = [0] + cd
    elif name == "C5":  # multiplexed mixed step, GQA 70B-layer-like
        seed, Hq, Hkv, d = 4, 64, 8, 128
        rng = np.random.default_rng(seed)
        cd = _lognormal_lengths(rng, 256, 1500, 1.0, 64, 8192).tolist()
        q = [4096, 1024] + [1] * 256
        c = [0, 0] + cd
    else:
        raise KeyError(f"unknown config {name!r}; expected one of {CONFIG_NAMES}")
    return seed, Hq, Hkv, d, 16, np.asarray(q, np.int32), np.asarray(c, np.int32), rng


# ----------------------------------------------------------------------------- value sources
class _Values:
    """N(0,1) -> bf16 bits.  'normal': every value freshly drawn.  'tiled': one drawn block of
    2^22 values reused cyclically (multi-GB pools for timing; still ordinary data for parity)."""

    def __init__(self, rng, mode: str):
        if mode not in ("normal", "tiled"):
            raise ValueError(mode)
        self.rng, self.mode = rng, mode
        self._block = None
        self._pos = 0

    def draw(self, n: int) -> np.ndarray:
        if self.mode == "normal":
            out = np.empty(n, np.uint16)
            step = 1 << 24
            for s in range(0, n, step):
                m = min(step, n - s)
                out[s:s + m] = f32_to_bf16_bits(self.rng.standard_normal(m, dtype=np.float32))
            return out
        if self._block is None:
            self._block = f32_to_bf16_bits(self.rng.standard_normal(1 << 22, dtype=np.float32))
        blk = self._block
        idx = (self._pos + np.arange(n, dtype=np.int64)) % blk.shape[0] if n < blk.shape[0] else None
        if idx is not None:
            out = blk[idx]
        else:
            reps = -(-(n + self._pos % blk.shape[0]) // blk.shape[0])
            out = np.tile(blk, reps)[self._pos % blk.shape[0]:][:n].copy()
        self._pos += n + 977  # de-phase consecutive draws
        return out


# ----------------------------------------------------------------------------- one step
def make_step(
    rng,
    num_q_heads: int,
    num_kv_heads: int,
    head_dim: int,
    page_size: int,
    q_lens: Sequence[int],
    ctx_lens: Sequence[int],
    *,
    num_pages: Optional[int] = None,
    poison: bool = True,
    values: str = "normal",
    shuffle_pages: bool = True,
    name: str = "custom",
    seed: int = -1,
) -> StepInputs:
    """Build one multiplexed iteration.  rng: numpy Generator (already past any length draws).

    Draw order: page permutation -> q -> k_new -> v_new -> prior-context K rows, V rows per request.
    Prior context is installed by writing the pool directly, so an append under test only handles
    this step's rows.  Unused slots hold POISON_BF16 when poison=True (else 0)."""
    q_lens = np.asarray(q_lens, np.int32)
    ctx_lens = np.asarray(ctx_lens, np.int32)
    assert q_lens.shape == ctx_lens.shape and q_lens.ndim == 1
    n = int(q_lens.shape[0])
    Hq, Hkv, d, P = num_q_heads, num_kv_heads, head_dim, page_size
    L = q_lens.astype(np.int64) + ctx_lens
    pages_per_req = (L + P - 1) // P
    need = int(pages_per_req.sum())
    if num_pages is None:
        num_pages = 64 * max(1, math.ceil(1.25 * need / 64))
    assert num_pages >= need, "pool too small"
    perm = rng.permutation(num_pages) if shuffle_pages else np.arange(num_pages)
    stride = max(1, int(pages_per_req.max()) if n else 1)
    page_table = np.full((n, stride), -1, np.int32)
    used = 0
    for i in range(n):
        k = int(pages_per_req[i])
        page_table[i, :k] = perm[used:used + k]
        used += k
    q_offsets = np.zeros(n + 1, np.int32)
    np.cumsum(q_lens, out=q_offsets[1:])
    T = int(q_offsets[-1])

    src = _Values(rng, values)
    q = src.draw(T * Hq * d).reshape(T, Hq, d)
    k_new = src.draw(T * Hkv * d).reshape(T, Hkv, d)
    v_new = src.draw(T * Hkv * d).reshape(T, Hkv, d)

    fill = POISON_BF16 if poison else 0
    k_pool = np.full((num_pages, Hkv, P, d), fill, np.uint16)
    v_pool = np.full((num_pages, Hkv, P, d), fill, np.uint16)
    for i in range(n):
        c = int(ctx_lens[i])
        if c == 0:
            continue
        for pool in (k_pool, v_pool):
            rows = src.draw(c * Hkv * d).reshape(c, Hkv, d)
            full = c // P
            if full:
                pool[page_table[i, :full]] = rows[: full * P].reshape(full, P, Hkv, d).transpose(0, 2, 1, 3)
            rem = c - full * P
            if rem:
                pool[page_table[i, full], :, :rem, :] = rows[full * P:].transpose(1, 0, 2)
    return StepInputs(name, seed, Hq, Hkv, d, P, int(num_pages), q_lens, ctx_lens, q_offsets,
                      page_table, k_pool, v_pool, q, k_new, v_new)


def make_config(name: str, *, poison: bool = True, values: str = "normal") -> StepInputs:
    """BASELINE.json configs[0..4] (C1..C5) with the seeds / pool sizes of SURVEY.md 8(c) S18-S19."""
    seed, Hq, Hkv, d, P, q_lens, ctx_lens, rng = config_lengths(name)
    num_pages = 64 if name == "C1" else None
    return make_step(rng, Hq, Hkv, d, P, q_lens, ctx_lens, num_pages=num_pages, poison=poison,
                     values=values, name=name, seed=seed)


# ----------------------------------------------------------------------------- KV migration
def make_migration_target(rng, kv_lens: Sequence[int], page_size: int, *, num_pages: Optional[int] = None,
                          shuffle_pages: bool = True):
    """Destination side of a KV migration (PAPER.md:155 Path 1: the cache of a prefilled request moves to the
    worker that will decode it): a page table into a second pool for requests holding kv_lens[m] tokens.
    Returns (dst_page_table int32 [n, stride] with -1 past ceil(len/P), num_dst_pages).  Placement only."""
    kv_lens = np.asarray(kv_lens, np.int64)
    pages_per_req = (kv_lens + page_size - 1) // page_size
    need = int(pages_per_req.sum())
    if num_pages is None:
        num_pages = 64 * max(1, math.ceil(1.25 * need / 64))
    assert num_pages >= need, "destination pool too small"
    perm = rng.permutation(num_pages) if shuffle_pages else np.arange(num_pages)
    n = int(kv_lens.shape[0])
    stride = max(1, int(pages_per_req.max()) if n else 1)
    table = np.full((n, stride), -1, np.int32)
    used = 0
    for m in range(n):
        k = int(pages_per_req[m])
        table[m, :k] = perm[used:used + k]
        used += k
    return table, int(num_pages)


# ----------------------------------------------------------------------------- RoPE tables
def make_rope_tables(table_len: int, head_dim: int, base: float = 10000.0):
    """The caller-side INPUT of a RoPE-fused append: cos / sin tables fp32 [table_len, head_dim / 2] of the angles
    pos * base^(-2 c / head_dim), evaluated in float64 and rounded to fp32 once.  Input generation only: the rotation
    itself is the library's (and, independently, the oracle's)."""
    pos = np.arange(table_len, dtype=np.float64)[:, None]
    freq = base ** (-2.0 * np.arange(head_dim // 2, dtype=np.float64) / head_dim)[None, :]
    ang = pos * freq
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)
