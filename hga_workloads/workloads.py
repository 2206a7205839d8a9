"""Workload definitions and the seeded input generator (numpy only, no method arithmetic)."""
from __future__ import annotations

import dataclasses

import numpy as np

__all__ = ["Workload", "CONFIGS", "get", "generate", "bf16_round"]


@dataclasses.dataclass(frozen=True)
class Workload:
    """One synthetic HGA prefill problem (notation: SURVEY.md section 8 / PAPER.md section 3)."""

    name: str
    batch: int  # B
    seq: int  # N
    n_q_heads: int  # H_q
    n_kv_heads: int  # H_kv
    head_dim: int  # D
    dtype: str  # "f32" | "bf16"  (storage type of Q/K/V)
    rope_base: float
    chunk: int = 64  # C
    group: int = 16  # g_s
    n_sink: int = 1  # F
    n_local: int = 1  # L
    topk_chunks: int = 16  # K_c
    topk_groups: int = 32  # K_g
    dist: str = "clustered"  # "iid" | "clustered"
    n_clusters: int = 32
    cluster_scale: float = 2.0
    pos0: int = 0
    rope_pos_mod: int = 0  # N3: RoPE position index wrapped modulo this value; 0 = off
    route_max: bool = False  # N3 (R19): block score = max over per-query scores, not the pooled query
    n_hi_chunk: int = -1  # leading high-frequency RoPE pairs at chunk / group level (R1); -1 = default rule
    n_hi_group: int = -1
    n_valid: int = 0  # prompt tokens actually present (ragged tail); 0 = seq.  `seq` is then the cache capacity

    @property
    def n_tokens(self) -> int:
        return self.n_valid if self.n_valid > 0 else self.seq

    @property
    def n_blocks(self) -> int:
        return self.seq // self.chunk

    @property
    def n_groups_total(self) -> int:
        return self.seq // self.group

    @property
    def gqa(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    def replace(self, **kw) -> "Workload":
        return dataclasses.replace(self, **kw)


# BASELINE.json configs[0..4]; c2/c3 RoPE base is not stated there -> 1e4.
CONFIGS = {
    "c1": Workload("c1", 1, 1024, 4, 1, 64, "f32", 1.0e4, topk_chunks=4, topk_groups=8, dist="iid"),
    "c2": Workload("c2", 4, 8192, 8, 8, 64, "bf16", 1.0e4, topk_chunks=16, topk_groups=32),
    "c3": Workload("c3", 8, 12288, 8, 8, 64, "bf16", 1.0e4, topk_chunks=16, topk_groups=32),
    "c4": Workload("c4", 1, 32768, 32, 4, 128, "bf16", 1.0e6, topk_chunks=16, topk_groups=64),
    "c5": Workload("c5", 1, 65536, 32, 4, 128, "bf16", 1.0e6, topk_chunks=12, topk_groups=48),
    # the paper's own needle-test parameters: 65,599 prompt tokens across
    # 1,025 chunks (a ragged last chunk of 63 tokens), keep first 2 / keep last 8, K_c = 20, K_g = 32 (group refinement
    # keeps 32 of 80 candidate groups), Qwen3-30B-A3B head shape.  Attended: 32*16 + 11*64 = 1216 tokens = 1.85 %.
    "p5": Workload("p5", 1, 65600, 32, 4, 128, "bf16", 1.0e6, n_sink=2, n_local=8, topk_chunks=20, topk_groups=32,
                   n_valid=65599),
}


def get(name: str) -> Workload:
    return CONFIGS[name]


def bf16_round(x: np.ndarray) -> np.ndarray:
    """Round fp32 values to the nearest bf16 (ties to even); result stays in an fp32 array.

    Storage-format conversion only.  Inputs are finite by construction.
    """
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) & np.uint32(0xFFFF0000)
    return r.view(np.float32)


def _rng(seed: int, stream: int) -> np.random.Generator:
    # Philox is counter-based: (seed, stream) keys an independent, reproducible sequence.
    return np.random.Generator(np.random.Philox(key=[np.uint64(seed), np.uint64(stream)]))


def generate(w: Workload, seed: int = 0):
    """Return (q_raw, k_raw, v) as fp32 numpy arrays of shape [B,H,N,D] (pre-RoPE Q and K).

    * ``iid``: every element ~ N(0,1).
    * ``clustered``: per KV head 32 unit directions u_m; every 64-token chunk of every batch item
      draws one cluster id; K_raw = n + scale*u_id and Q_raw (all query heads of the KV group)
      = n + scale*u_id with n ~ N(0,1); V ~ N(0,1).  Planted before RoPE.
    For ``dtype == "bf16"`` the values are rounded to bf16 (still returned as fp32 arrays, so that the
    oracle and the GPU consume the same bits).
    """
    B, N, Hq, Hkv, D = w.batch, w.seq, w.n_q_heads, w.n_kv_heads, w.head_dim
    q = _rng(seed, 1).standard_normal((B, Hq, N, D), dtype=np.float32)
    k = _rng(seed, 2).standard_normal((B, Hkv, N, D), dtype=np.float32)
    v = _rng(seed, 3).standard_normal((B, Hkv, N, D), dtype=np.float32)
    if w.dist == "clustered":
        g = _rng(seed, 4)
        dirs = g.standard_normal((Hkv, w.n_clusters, D), dtype=np.float32)
        dirs /= np.linalg.norm(dirs, axis=-1, keepdims=True)
        ids = g.integers(0, w.n_clusters, size=(B, w.n_blocks))
        G = w.gqa
        for b in range(B):
            for kh in range(Hkv):
                shift = np.repeat(dirs[kh, ids[b]] * np.float32(w.cluster_scale), w.chunk, axis=0)  # [N,D]
                k[b, kh] += shift
                q[b, kh * G:(kh + 1) * G] += shift[None]
    elif w.dist != "iid":
        raise ValueError(f"unknown dist {w.dist!r}")
    if w.dtype == "bf16":
        q, k, v = bf16_round(q), bf16_round(k), bf16_round(v)
    elif w.dtype != "f32":
        raise ValueError(f"unknown dtype {w.dtype!r}")
    return q, k, v
