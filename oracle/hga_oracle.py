"""ctypes binding of oracle/hga_oracle.c (argument marshalling only; all arithmetic is in the C file).

TEST INFRASTRUCTURE ONLY.  Nothing here imports or calls the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hga_oracle.c")
_LIB = os.path.join(_HERE, "libhga_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("G", C.c_int32), ("N", C.c_int32), ("D", C.c_int32), ("C", C.c_int32), ("gs", C.c_int32),
        ("F", C.c_int32), ("L", C.c_int32), ("Kc", C.c_int32), ("Kg", C.c_int32),
        ("n_hi_chunk", C.c_int32), ("n_hi_group", C.c_int32), ("io_bf16", C.c_int32),
        ("pos0", C.c_int64), ("base", C.c_double), ("scale", C.c_double), ("pos_mod", C.c_int64),
        ("route_max", C.c_int32), ("pad_", C.c_int32),
    ]


@dataclasses.dataclass
class OracleParams:
    G: int
    N: int
    D: int
    C: int = 64
    gs: int = 16
    F: int = 1
    L: int = 1
    Kc: int = 16
    Kg: int = 32
    n_hi_chunk: int = -1
    n_hi_group: int = -1
    io_bf16: bool = False
    pos0: int = 0
    base: float = 1.0e4
    scale: float = 0.0
    pos_mod: int = 0  # N3: RoPE position index wrapped modulo pos_mod; 0 = off
    route_max: bool = False  # N3 (R4's alternative, R19): block score = max over the 64*G per-query scores

    def c_struct(self) -> _Params:
        return _Params(self.G, self.N, self.D, self.C, self.gs, self.F, self.L, self.Kc, self.Kg,
                       self.n_hi_chunk, self.n_hi_group, int(self.io_bf16), self.pos0, self.base, self.scale,
                       self.pos_mod, int(self.route_max), 0)


def params_from_workload(w) -> OracleParams:
    return OracleParams(G=w.n_q_heads // w.n_kv_heads, N=w.seq, D=w.head_dim, C=w.chunk, gs=w.group, F=w.n_sink,
                        L=w.n_local, Kc=w.topk_chunks, Kg=w.topk_groups, io_bf16=(w.dtype == "bf16"),
                        pos0=w.pos0, base=w.rope_base, pos_mod=getattr(w, "rope_pos_mod", 0),
                        n_hi_chunk=getattr(w, "n_hi_chunk", -1), n_hi_group=getattr(w, "n_hi_group", -1),
                        route_max=bool(getattr(w, "route_max", False)))


def _L():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.hga_oracle_theta.restype = C.c_double
        _lib.hga_oracle_theta.argtypes = [C.c_int, C.c_double, C.c_int]
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError(f"oracle {what} failed with code {rc} "
                         "(1=bad argument, 2=non-finite input, 3=bad group index)")


def max_threads() -> int:
    return int(_L().hga_oracle_max_threads())


def default_n_hi(D: int, base: float, span: int) -> int:
    return int(_L().hga_oracle_default_n_hi(C.c_int(D), C.c_double(base), C.c_int(span)))


def n_hi_rule(D: int, base: float, span: int, rule: int) -> int:
    """N3: # of leading high-frequency pairs under rule 0 (wavelength <= span), 1 (sweep >= pi), 2 (sweep >= 1 rad)."""
    n = int(_L().hga_oracle_n_hi_rule(C.c_int(D), C.c_double(base), C.c_int(span), C.c_int(rule)))
    if n < 0:
        raise ValueError("unknown n_hi rule")
    return n


def rope(x, pos_first: int, base: float, pos_mod: int = 0) -> np.ndarray:
    """x [..., n_rows, D] fp32, consecutive positions from pos_first along axis -2 (wrapped modulo pos_mod if > 0,
    PAPER.md:259-264) -> fp64."""
    x = _f32(x)
    D = x.shape[-1]
    n_rows = x.shape[-2]
    out = np.empty(x.shape, dtype=np.float64)
    xf = x.reshape(-1, n_rows, D)
    of = out.reshape(-1, n_rows, D)
    for i in range(xf.shape[0]):
        _check(_L().hga_oracle_rope_mod(_p(xf[i], C.c_float), C.c_int(n_rows), C.c_int(D), C.c_int64(pos_first),
                                        C.c_int64(pos_mod), C.c_double(base), _p(of[i], C.c_double)), "rope")
    return out


def round_io(x, io_bf16: bool) -> np.ndarray:
    out = _f64(x).copy()
    _L().hga_oracle_round_io(_p(out, C.c_double), C.c_size_t(out.size), C.c_int(int(io_bf16)))
    return out


def summaries(k_raw, span: int, n_hi: int, pos0: int, base: float, pos_mod: int = 0) -> np.ndarray:
    """k_raw [N,D] fp32 -> [N/span, D] fp64 mixed-RoPE summaries."""
    k_raw = _f32(k_raw)
    N, D = k_raw.shape
    out = np.empty((N // span, D), dtype=np.float64)
    _check(_L().hga_oracle_summaries_mod(_p(k_raw, C.c_float), C.c_int(N), C.c_int(D), C.c_int(span), C.c_int(n_hi),
                                         C.c_int64(pos0), C.c_int64(pos_mod), C.c_double(base),
                                         _p(out, C.c_double)), "summaries")
    return out


def pool_queries(q_rot, chunk: int) -> np.ndarray:
    """q_rot [G,N,D] fp64 -> [N/chunk, D]."""
    q_rot = _f64(q_rot)
    G, N, D = q_rot.shape
    out = np.empty((N // chunk, D), dtype=np.float64)
    _check(_L().hga_oracle_pool_queries(_p(q_rot, C.c_double), C.c_int(G), C.c_int(N), C.c_int(D), C.c_int(chunk),
                                        _p(out, C.c_double)), "pool_queries")
    return out


def route_chunks(qbar_j, S_c, j: int, F: int, L: int, Kc: int):
    """-> (idx [Kc] int32 ascending, -1 padded; scores [Kc]; count; all_scores [n_b] NaN off-candidate)."""
    qbar_j, S_c = _f64(qbar_j), _f64(S_c)
    n_b, D = S_c.shape
    idx = np.empty(max(Kc, 1), dtype=np.int32)
    sc = np.empty(max(Kc, 1), dtype=np.float64)
    alls = np.empty(n_b, dtype=np.float64)
    cnt = _L().hga_oracle_route_chunks(_p(qbar_j, C.c_double), _p(S_c, C.c_double), C.c_int(n_b), C.c_int(D),
                                       C.c_int(j), C.c_int(F), C.c_int(L), C.c_int(Kc), _p(idx, C.c_int),
                                       _p(sc, C.c_double), _p(alls, C.c_double))
    return idx[:Kc], sc[:Kc], int(cnt), alls


def route_groups(qbar_j, S_g, gpc: int, chunk_idx: Sequence[int], Kg: int):
    """chunk_idx: the selected chunks (no -1).  -> (idx [Kg], scores [Kg], count, cand_scores)."""
    qbar_j, S_g = _f64(qbar_j), _f64(S_g)
    D = S_g.shape[1]
    ci = _i32([c for c in chunk_idx if c >= 0])
    idx = np.empty(max(Kg, 1), dtype=np.int32)
    sc = np.empty(max(Kg, 1), dtype=np.float64)
    cand = np.empty(max(len(ci) * gpc, 1), dtype=np.float64)
    cnt = _L().hga_oracle_route_groups(_p(qbar_j, C.c_double), _p(S_g, C.c_double), C.c_int(D), C.c_int(gpc),
                                       _p(ci, C.c_int), C.c_int(len(ci)), C.c_int(Kg), _p(idx, C.c_int),
                                       _p(sc, C.c_double), _p(cand, C.c_double))
    return idx[:Kg], sc[:Kg], int(cnt), cand[:len(ci) * gpc]


def route_chunks_max(q_rows, S_c, j: int, F: int, L: int, Kc: int):
    """N3 (R4's alternative): score(c) = max over the rows of q_rows [n_rows, D] of q . S_c[c].  Returns as route_chunks."""
    q_rows, S_c = _f64(q_rows), _f64(S_c)
    n_b, D = S_c.shape
    q_rows = np.ascontiguousarray(q_rows.reshape(-1, D))
    idx = np.empty(max(Kc, 1), dtype=np.int32)
    sc = np.empty(max(Kc, 1), dtype=np.float64)
    alls = np.empty(n_b, dtype=np.float64)
    cnt = _L().hga_oracle_route_chunks_max(_p(q_rows, C.c_double), C.c_int(q_rows.shape[0]), _p(S_c, C.c_double),
                                           C.c_int(n_b), C.c_int(D), C.c_int(j), C.c_int(F), C.c_int(L), C.c_int(Kc),
                                           _p(idx, C.c_int), _p(sc, C.c_double), _p(alls, C.c_double))
    return idx[:Kc], sc[:Kc], int(cnt), alls


def route_groups_max(q_rows, S_g, gpc: int, chunk_idx: Sequence[int], Kg: int):
    """N3: score(g) = max over the rows of q_rows of q . S_g[g].  Returns as route_groups."""
    q_rows, S_g = _f64(q_rows), _f64(S_g)
    D = S_g.shape[1]
    q_rows = np.ascontiguousarray(q_rows.reshape(-1, D))
    ci = _i32([c for c in chunk_idx if c >= 0])
    idx = np.empty(max(Kg, 1), dtype=np.int32)
    sc = np.empty(max(Kg, 1), dtype=np.float64)
    cand = np.empty(max(len(ci) * gpc, 1), dtype=np.float64)
    cnt = _L().hga_oracle_route_groups_max(_p(q_rows, C.c_double), C.c_int(q_rows.shape[0]), _p(S_g, C.c_double),
                                           C.c_int(D), C.c_int(gpc), _p(ci, C.c_int), C.c_int(len(ci)), C.c_int(Kg),
                                           _p(idx, C.c_int), _p(sc, C.c_double), _p(cand, C.c_double))
    return idx[:Kg], sc[:Kg], int(cnt), cand[:len(ci) * gpc]


def key_set(j: int, chunk: int, gs: int, F: int, L: int, group_idx) -> np.ndarray:
    """Boolean mask over tokens [0, (j+1)*chunk): the union set of block j (before the causal cut)."""
    gi = _i32(group_idx)
    vis = np.zeros((j + 1) * chunk, dtype=np.uint8)
    _check(_L().hga_oracle_key_set(C.c_int(j), C.c_int(chunk), C.c_int(gs), C.c_int(F), C.c_int(L), _p(gi, C.c_int),
                                   C.c_int(gi.size), _p(vis, C.c_ubyte)), "key_set")
    return vis.astype(bool)


def attend_block(q_blk, k_rot, v, j: int, chunk: int, gs: int, F: int, L: int, group_idx, scale: float = 0.0):
    """q_blk [G,C,D], k_rot [N,D], v [N,D] (fp64, already storage-rounded) -> (out [G,C,D], lse [G,C], n_keys [C])."""
    q_blk, k_rot, v = _f64(q_blk), _f64(k_rot), _f64(v)
    G, Cc, D = q_blk.shape
    N = k_rot.shape[0]
    gi = _i32(group_idx)
    out = np.empty((G, Cc, D), dtype=np.float64)
    lse = np.empty((G, Cc), dtype=np.float64)
    nk = np.empty(Cc, dtype=np.int32)
    _check(_L().hga_oracle_attend_block(_p(q_blk, C.c_double), _p(k_rot, C.c_double), _p(v, C.c_double), C.c_int(G),
                                        C.c_int(N), C.c_int(D), C.c_int(chunk), C.c_int(gs), C.c_int(F), C.c_int(L),
                                        C.c_int(j), _p(gi, C.c_int), C.c_int(gi.size), C.c_double(scale),
                                        _p(out, C.c_double), _p(lse, C.c_double), _p(nk, C.c_int)), "attend_block")
    return out, lse, nk


def dense_block(q_blk, k_rot, v, j: int, chunk: int, scale: float = 0.0):
    """Eq. (1) for the rows of block j."""
    q_blk, k_rot, v = _f64(q_blk), _f64(k_rot), _f64(v)
    G, Cc, D = q_blk.shape
    N = k_rot.shape[0]
    out = np.empty((G, Cc, D), dtype=np.float64)
    lse = np.empty((G, Cc), dtype=np.float64)
    _check(_L().hga_oracle_dense_block(_p(q_blk, C.c_double), _p(k_rot, C.c_double), _p(v, C.c_double), C.c_int(G),
                                       C.c_int(N), C.c_int(D), C.c_int(chunk), C.c_int(j), C.c_double(scale),
                                       _p(out, C.c_double), _p(lse, C.c_double)), "dense_block")
    return out, lse


@dataclasses.dataclass
class SliceResult:
    blocks: np.ndarray  # [n_blocks] block ids
    k_rot: Optional[np.ndarray]  # [N,D] rotated keys after storage rounding
    chunk_sum: np.ndarray  # [n_b,D]
    group_sum: np.ndarray  # [n_g,D]
    q_pooled: np.ndarray  # [n_blocks,D]
    chunk_idx: np.ndarray  # [n_blocks,Kc]
    chunk_score: np.ndarray
    n_chunks: np.ndarray
    chunk_all_scores: np.ndarray  # [n_blocks,n_b], NaN where not a candidate
    group_idx: np.ndarray  # [n_blocks,Kg]
    group_score: np.ndarray
    n_groups: np.ndarray
    group_cand_scores: np.ndarray  # [n_blocks,Kc*C/gs], NaN padded
    out: Optional[np.ndarray]  # [n_blocks,G,C,D]
    lse: Optional[np.ndarray]  # [n_blocks,G,C]


def prefill_slice(p: OracleParams, q_raw, k_raw, v, blocks=None, attend: bool = True, want_k_rot: bool = True
                  ) -> SliceResult:
    """Steps O1..O6 for one (batch, kv-head) slice: q_raw [G,N,D], k_raw [N,D], v [N,D]."""
    q_raw, k_raw, v = _f32(q_raw), _f32(k_raw), _f32(v)
    G, N, D = q_raw.shape
    assert (G, N, D) == (p.G, p.N, p.D) and k_raw.shape == (N, D) and v.shape == (N, D)
    n_b, n_g, gpc = N // p.C, N // p.gs, p.C // p.gs
    blk = _i32(np.arange(n_b) if blocks is None else blocks)
    nb = blk.size
    Kc, Kg = max(p.Kc, 1), max(p.Kg, 1)
    r = SliceResult(
        blocks=blk,
        k_rot=np.empty((N, D)) if want_k_rot else None,
        chunk_sum=np.empty((n_b, D)), group_sum=np.empty((n_g, D)), q_pooled=np.empty((nb, D)),
        chunk_idx=np.empty((nb, Kc), dtype=np.int32), chunk_score=np.empty((nb, Kc)),
        n_chunks=np.empty(nb, dtype=np.int32), chunk_all_scores=np.empty((nb, n_b)),
        group_idx=np.empty((nb, Kg), dtype=np.int32), group_score=np.empty((nb, Kg)),
        n_groups=np.empty(nb, dtype=np.int32), group_cand_scores=np.empty((nb, Kc * gpc)),
        out=np.empty((nb, G, p.C, D)) if attend else None,
        lse=np.empty((nb, G, p.C)) if attend else None,
    )
    ps = p.c_struct()
    rc = _L().hga_oracle_slice(
        C.byref(ps), _p(q_raw, C.c_float), _p(k_raw, C.c_float), _p(v, C.c_float), _p(blk, C.c_int), C.c_int(nb),
        C.c_int(int(attend)), _p(r.k_rot, C.c_double), _p(r.chunk_sum, C.c_double), _p(r.group_sum, C.c_double),
        _p(r.q_pooled, C.c_double), _p(r.chunk_idx, C.c_int), _p(r.chunk_score, C.c_double), _p(r.n_chunks, C.c_int),
        _p(r.chunk_all_scores, C.c_double), _p(r.group_idx, C.c_int), _p(r.group_score, C.c_double),
        _p(r.n_groups, C.c_int), _p(r.group_cand_scores, C.c_double), _p(r.out, C.c_double), _p(r.lse, C.c_double))
    _check(rc, "prefill_slice")
    r.chunk_idx = r.chunk_idx[:, :p.Kc]
    r.chunk_score = r.chunk_score[:, :p.Kc]
    r.group_idx = r.group_idx[:, :p.Kg]
    r.group_score = r.group_score[:, :p.Kg]
    r.group_cand_scores = r.group_cand_scores[:, :p.Kc * gpc]
    return r


@dataclasses.dataclass
class StepResult:
    q_pooled: np.ndarray  # [D]
    chunk_idx: np.ndarray  # [Kc]
    chunk_score: np.ndarray
    n_chunks: int
    group_idx: np.ndarray  # [Kg]
    group_score: np.ndarray
    n_groups: int
    out: Optional[np.ndarray]  # [G,W,D]
    lse: Optional[np.ndarray]  # [G,W]


def step(p: OracleParams, q_win, k_hist, v_hist, t0: int, t1: int, attend: bool = True) -> StepResult:
    """One streaming step (hga_oracle_step, N1): window [t0, t1) of the active chunk; q_win [G, t1-t0, D] raw queries
    of the window, k_hist / v_hist [t1, D] -- ONLY tokens 0..t1-1 are handed over (p.N is ignored)."""
    q_win, k_hist, v_hist = _f32(q_win), _f32(k_hist), _f32(v_hist)
    G, W, D = q_win.shape
    assert (G, D) == (p.G, p.D) and W == t1 - t0 and k_hist.shape == (t1, D) and v_hist.shape == (t1, D)
    Kc, Kg = max(p.Kc, 1), max(p.Kg, 1)
    qp = np.empty(D)
    ci, cs, nc = np.empty(Kc, dtype=np.int32), np.empty(Kc), C.c_int(0)
    gi, gsc, ng = np.empty(Kg, dtype=np.int32), np.empty(Kg), C.c_int(0)
    out = np.empty((G, W, D)) if attend else None
    lse = np.empty((G, W)) if attend else None
    ps = p.c_struct()
    rc = _L().hga_oracle_step(C.byref(ps), _p(q_win, C.c_float), _p(k_hist, C.c_float), _p(v_hist, C.c_float),
                              C.c_int64(t0), C.c_int64(t1), _p(qp, C.c_double), _p(ci, C.c_int), _p(cs, C.c_double),
                              C.byref(nc), _p(gi, C.c_int), _p(gsc, C.c_double), C.byref(ng), _p(out, C.c_double),
                              _p(lse, C.c_double))
    _check(rc, "step")
    return StepResult(qp, ci[:p.Kc], cs[:p.Kc], nc.value, gi[:p.Kg], gsc[:p.Kg], ng.value, out, lse)


def prefill(p: OracleParams, q_raw, k_raw, v, blocks=None, attend: bool = True, want_k_rot: bool = False):
    """Whole tensors: q_raw [B,Hq,N,D], k_raw/v [B,Hkv,N,D].  Returns {(b, kv_head): SliceResult}."""
    B, Hq = q_raw.shape[:2]
    Hkv = k_raw.shape[1]
    assert Hq == Hkv * p.G
    res = {}
    for b in range(B):
        for kh in range(Hkv):
            res[(b, kh)] = prefill_slice(p, q_raw[b, kh * p.G:(kh + 1) * p.G], k_raw[b, kh], v[b, kh], blocks,
                                         attend, want_k_rot)
    return res
