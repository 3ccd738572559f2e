"""Test-side helpers that are independent of BOTH oracle/ and the CUDA path.

* brute-force dense attention (numpy fp64, full score matrix with -inf mask) -- pin O1
* logical (dense) K/V  <->  paged pool packing for arbitrary page sizes -- pins O3/O4
* a python-loop KV append -- pin for oracle_kv_append

Nothing here is imported by oracle/ or paper_2606_16264_b200/.
"""
from __future__ import annotations

import numpy as np

from synth import POISON_BF16, bf16_bits_to_f32


def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    return bf16_bits_to_f32(bits).astype(np.float64)


def gather_dense(pool: np.ndarray, page_row: np.ndarray, n_keys: int) -> np.ndarray:
    """pool uint16 [pages, Hkv, P, d] -> dense uint16 [n_keys, Hkv, d] by fancy indexing."""
    P = pool.shape[2]
    j = np.arange(n_keys)
    return pool[page_row[j // P], :, j % P, :]


def dense_attention_bruteforce(q_bits, k_dense_bits, v_dense_bits, ctx_len: int, sm_scale: float = 0.0):
    """One request.  q_bits [q_len, Hq, d]; k/v_dense_bits [ctx_len + q_len, Hkv, d] (already appended).

    Full [q_len, L] score matrix per head, additive -inf mask for j > ctx_len + t, row softmax,
    matmul.  Returns (out [q_len, Hq, d], lse [q_len, Hq], weights [Hq, q_len, L])."""
    q = bf16_to_f64(q_bits)
    k = bf16_to_f64(k_dense_bits)
    v = bf16_to_f64(v_dense_bits)
    q_len, Hq, d = q.shape
    L, Hkv, _ = k.shape
    assert L == ctx_len + q_len
    g = Hq // Hkv
    scale = sm_scale if sm_scale > 0 else 1.0 / np.sqrt(d)
    out = np.zeros((q_len, Hq, d))
    lse = np.zeros((q_len, Hq))
    weights = np.zeros((Hq, q_len, L))
    mask = np.where(np.arange(L)[None, :] <= ctx_len + np.arange(q_len)[:, None], 0.0, -np.inf)
    for h in range(Hq):
        hk = h // g
        s = scale * (q[:, h, :] @ k[:, hk, :].T) + mask
        m = s.max(axis=1, keepdims=True)
        e = np.exp(s - m)
        z = e.sum(axis=1, keepdims=True)
        w = e / z
        weights[h] = w
        out[:, h, :] = w @ v[:, hk, :]
        lse[:, h] = (m + np.log(z))[:, 0]
    return out, lse, weights


def pack_pool(dense_list, page_size: int, rng, num_pages=None, shuffle=True, fill=POISON_BF16):
    """dense_list: per request uint16 [L_i, Hkv, d] -> (pool [pages,Hkv,P,d], page_table [n, stride])."""
    P = page_size
    Hkv, d = dense_list[0].shape[1:]
    per = [(x.shape[0] + P - 1) // P for x in dense_list]
    need = sum(per)
    if num_pages is None:
        num_pages = need + 3
    ids = rng.permutation(num_pages) if shuffle else np.arange(num_pages)
    stride = max(1, max(per))
    pt = np.full((len(dense_list), stride), -1, np.int32)
    pool = np.full((num_pages, Hkv, P, d), fill, np.uint16)
    used = 0
    for i, x in enumerate(dense_list):
        pt[i, :per[i]] = ids[used:used + per[i]]
        used += per[i]
        for j in range(x.shape[0]):
            pool[pt[i, j // P], :, j % P, :] = x[j]
    return pool, pt


def append_python_loops(k_pool, v_pool, q_lens, ctx_lens, q_offsets, page_table, k_new, v_new):
    """Scalar-loop restatement of SURVEY 8(a) row A1 (in place)."""
    P = k_pool.shape[2]
    for i in range(len(q_lens)):
        for t in range(int(q_lens[i])):
            pos = int(ctx_lens[i]) + t
            pg, sl = int(page_table[i, pos // P]), pos % P
            k_pool[pg, :, sl, :] = k_new[int(q_offsets[i]) + t]
            v_pool[pg, :, sl, :] = v_new[int(q_offsets[i]) + t]
