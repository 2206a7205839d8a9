"""Planted retrieval needle for BASELINE.json configs[4] (c5), the synthetic stand-in for the paper's needle-in-a-haystack
probe (section 5.3).  Test helper: builds an INPUT with the oracle's own RoPE / pooling (DESIGN.md
section 3); the result is fed identically to the oracle and to the CUDA path.  It never touches the CUDA path.

Recipe: group g* = floor(depth * n_g).  With q_hat the unit pooled rotated query of the final block
(per KV head), the needle's rotated keys are  k_rot_t = rho * (0.9 * q_hat + sqrt(0.19) * z_t),  z_t a unit vector
orthogonal to q_hat, rho = sqrt(D + 4) * gain (the typical key norm of the clustered workload); K_raw_t = R(-p_t) k_rot_t,
rounded to the workload's storage dtype.  Cosine(k_rot_t, q_hat) = 0.9 before rounding.
"""
from __future__ import annotations

import numpy as np

import hga_workloads as W
import oracle

DEPTHS = (0.10, 0.50, 0.90)


def needle_group(w: W.Workload, depth: float) -> int:
    return int(np.floor(depth * w.n_groups_total))


def _inverse_rope(x_rot: np.ndarray, pos_first: int, base: float) -> np.ndarray:
    """R(-p) x for consecutive positions, through the oracle's forward RoPE: R(-p) x = conj(R(p) conj(x))."""
    half = x_rot.shape[-1] // 2
    y = np.array(x_rot, dtype=np.float32, copy=True)
    y[..., half:] *= -1.0
    z = oracle.rope(y, pos_first, base)
    z[..., half:] *= -1.0
    return z


def plant(w: W.Workload, q: np.ndarray, k: np.ndarray, depth: float, seed: int = 0, gain: float = 1.0,
          batch_item: int = 0) -> int:
    """Overwrite, in place, the keys of the needle group in every KV head of `batch_item`.  Returns g*."""
    g_star = needle_group(w, depth)
    G, C, D, gs = w.gqa, w.chunk, w.head_dim, w.group
    t0 = g_star * gs
    j_last = w.n_blocks - 1
    assert t0 // C < j_last - max(w.n_local, 1) and t0 // C >= w.n_sink, "needle must sit in the routed middle region"
    rng = np.random.Generator(np.random.Philox(key=[np.uint64(seed), np.uint64(97)]))
    rho = np.sqrt(D + 4.0) * gain
    for kh in range(w.n_kv_heads):
        q_rot = oracle.rope(q[batch_item, kh * G:(kh + 1) * G, j_last * C:], w.pos0 + j_last * C, w.rope_base)  # [G,C,D]
        q_bar = oracle.pool_queries(q_rot, C)[0]
        q_hat = q_bar / np.linalg.norm(q_bar)
        z = rng.standard_normal((gs, D))
        z -= np.outer(z @ q_hat, q_hat)
        z /= np.linalg.norm(z, axis=1, keepdims=True)
        k_rot = rho * (0.9 * q_hat[None, :] + np.sqrt(0.19) * z)
        k_raw = _inverse_rope(k_rot, w.pos0 + t0, w.rope_base).astype(np.float32)
        k[batch_item, kh, t0:t0 + gs] = W.bf16_round(k_raw) if w.dtype == "bf16" else k_raw
    return g_star
