"""Helpers shared by the GPU parity tests, smoke() and nothing else: run the CUDA path through the C ABI binding,
run the CPU oracle on the same seeded inputs, compare under the north star's rules.

Index sets: bit-exact, except that a swap is accepted iff the oracle's fp64 scores of the swapped items differ by
<= 1e-6 * max|score| over that selection's candidates (reading R15).
Outputs: max-abs <= 1e-4 (fp32 inputs) / 2e-2 (bf16 inputs, fp32 accumulation).
"""
from __future__ import annotations

import dataclasses

import numpy as np
import torch

import hga_workloads as W
import oracle
import paper_2606_30709_b200 as hga

TIE_REL = 1e-6
TOL_OUT = {"f32": 1e-4, "bf16": 2e-2}


def to_device(w: W.Workload, arrs, device="cuda"):
    dt = torch.bfloat16 if w.dtype == "bf16" else torch.float32
    return tuple(torch.from_numpy(a).to(device=device, dtype=dt) for a in arrs)  # bf16-valued fp32 -> bf16 is exact


@dataclasses.dataclass
class SetCheck:
    exact: int = 0
    tie_swaps: int = 0
    bad: int = 0
    skipped: int = 0


def compare_sets(gpu_idx, ora_idx, score_of, max_abs_score, chk: SetCheck) -> bool:
    """gpu_idx / ora_idx: 1-D int arrays (-1 padded).  score_of: dict/array lookup of the oracle's fp64 score.
    Returns True if the sets are identical."""
    g = set(int(x) for x in gpu_idx if x >= 0)
    o = set(int(x) for x in ora_idx if x >= 0)
    if g == o:
        chk.exact += 1
        return True
    only_g, only_o = g - o, o - g
    ok = len(only_g) == len(only_o)
    if ok:
        sc = [score_of(i) for i in (only_g | only_o)]
        ok = bool(np.all(np.isfinite(sc))) and (max(sc) - min(sc) <= TIE_REL * max_abs_score)
    if ok:
        chk.tie_swaps += 1
    else:
        chk.bad += 1
    return False


def check_lists_wellformed(idx: np.ndarray, cnt: np.ndarray):
    """ascending, distinct, -1 padded after `cnt` entries."""
    K = idx.shape[-1]
    flat = idx.reshape(-1, K)
    c = cnt.reshape(-1)
    pos = np.arange(K)[None, :]
    valid = pos < c[:, None]
    assert np.all(flat[~valid] == -1)
    assert np.all(flat[valid] >= 0)
    d = np.diff(flat, axis=1)
    assert np.all(d[valid[:, 1:]] > 0)


def run_gpu(w: W.Workload, q, k, v, attend_impl=hga.binding.ATTEND_AUTO, out_dtype=hga.binding.HGA_F32, **over):
    """Whole path through hga_prefill.  q,k,v: numpy fp32 arrays from hga_workloads."""
    p = hga.params_from_workload(w, out_dtype=out_dtype, attend_impl=attend_impl)
    if over:
        p = p.replace(**over)
    dq, dk, dv = to_device(w, (q, k, v))
    buf = hga.hga_prefill(p, dq, dk, dv)
    torch.cuda.synchronize()
    return p, buf


def check_against_oracle(w: W.Workload, q, k, v, p, buf, slices, blocks, check_intermediates=True, **over):
    """Compare the GPU buffers with the oracle on the given (b, kv) slices and block ids.  Returns a report dict."""
    op = oracle.params_from_workload(w)
    if over:
        op = dataclasses.replace(op, **{{"topk_chunks": "Kc", "topk_groups": "Kg", "n_sink": "F", "n_local": "L",
                                         "pos0": "pos0", "n_hi_chunk": "n_hi_chunk", "n_hi_group": "n_hi_group"}[a]: b
                                        for a, b in over.items()})
    G, C, D = op.G, op.C, op.D
    gpc = C // op.gs
    tol = TOL_OUT[w.dtype]
    cchk, gchk = SetCheck(), SetCheck()
    worst = dict(out=0.0, lse=0.0, pooled=0.0, chunk_sum=0.0, group_sum=0.0, k_rot=0.0, q_rot=0.0, score=0.0)
    blocks = np.asarray(blocks, dtype=np.int32)
    for (b, kh) in slices:
        r = oracle.prefill_slice(op, q[b, kh * G:(kh + 1) * G], k[b, kh], v[b, kh], blocks=blocks, attend=True)
        g_cidx = buf.chunk_idx[b, kh].cpu().numpy()
        g_gidx = buf.group_idx[b, kh].cpu().numpy()
        g_ncnt = buf.n_chunks[b, kh].cpu().numpy()
        g_gcnt = buf.n_groups[b, kh].cpu().numpy()
        if op.Kc > 0:
            check_lists_wellformed(g_cidx[:, :op.Kc], g_ncnt)
        if op.Kg > 0:
            check_lists_wellformed(g_gidx[:, :op.Kg], g_gcnt)
        if check_intermediates:
            kr = buf.k_rot[b, kh].float().cpu().numpy().astype(np.float64)
            worst["k_rot"] = max(worst["k_rot"], float(np.abs(kr - r.k_rot).max()))
            cs = buf.chunk_sum[b, kh].cpu().numpy().astype(np.float64)
            gs_ = buf.group_sum[b, kh].cpu().numpy().astype(np.float64)
            worst["chunk_sum"] = max(worst["chunk_sum"], float(np.abs(cs - r.chunk_sum).max()))
            worst["group_sum"] = max(worst["group_sum"], float(np.abs(gs_ - r.group_sum).max()))
            qp = buf.q_pooled[b, kh].cpu().numpy().astype(np.float64)[blocks]
            worst["pooled"] = max(worst["pooled"], float(np.abs(qp - r.q_pooled).max()))
            # rotated queries of the sampled blocks against O1 rounded to the I/O dtype (one storage rounding apart)
            for j in blocks[:: max(1, len(blocks) // 8)]:
                qo = oracle.round_io(oracle.rope(q[b, kh * G:(kh + 1) * G, j * C:(j + 1) * C], op.pos0 + j * C, op.base,
                                                 op.pos_mod), op.io_bf16)
                if buf.q_rot is not None:  # not materialised under FLAG_FUSE_Q_ROPE
                    qg = buf.q_rot[b, kh * G:(kh + 1) * G, j * C:(j + 1) * C].float().cpu().numpy().astype(np.float64)
                    worst["q_rot"] = max(worst["q_rot"], float(np.abs(qg - qo).max()))
        g_out = buf.out[b, kh * G:(kh + 1) * G].float().cpu().numpy().astype(np.float64)  # [G,N,D]
        g_lse = buf.lse[b, kh * G:(kh + 1) * G].cpu().numpy().astype(np.float64)
        kv64 = v[b, kh].astype(np.float64)
        for bi, j in enumerate(blocks):
            alls = r.chunk_all_scores[bi]
            n_cand = int(np.isfinite(alls).sum())
            assert g_ncnt[j] == r.n_chunks[bi] == min(op.Kc, n_cand)
            mx = float(np.nanmax(np.abs(alls))) if n_cand else 0.0
            same_c = compare_sets(g_cidx[j, :op.Kc], r.chunk_idx[bi], lambda c: alls[c], mx, cchk)
            if n_cand and op.Kc > 0 and r.n_chunks[bi] > 0:
                gsc = buf.chunk_score[b, kh, j].cpu().numpy()[: r.n_chunks[bi]]
                gi = g_cidx[j, : r.n_chunks[bi]]
                # error scale of a dot product of fp32-stored operands: eps * sum_d |q_d||s_d| <= eps * |q||s|
                # (Cauchy-Schwarz); a row whose few candidates all score near zero is not judged relative to itself
                mag = float(np.linalg.norm(r.q_pooled[bi]) * np.linalg.norm(r.chunk_sum[gi], axis=1).max())
                worst["score"] = max(worst["score"], float(np.abs(gsc - alls[gi]).max() / max(mx, mag, 1e-30)))
            same_g = False
            if op.Kg > 0:
                if same_c:
                    cand_ids = (r.chunk_idx[bi][: r.n_chunks[bi], None] * gpc + np.arange(gpc)[None]).reshape(-1)
                    cand_sc = dict(zip(cand_ids.tolist(), r.group_cand_scores[bi][: len(cand_ids)].tolist()))
                    gmx = max((abs(x) for x in cand_sc.values()), default=0.0)
                    assert g_gcnt[j] == r.n_groups[bi]
                    same_g = compare_sets(g_gidx[j, :op.Kg], r.group_idx[bi], lambda g_: cand_sc.get(g_, np.nan), gmx, gchk)
                else:
                    gchk.skipped += 1
            else:
                same_g = True
            # attention: against the oracle's own set when identical, else O6 re-run on the GPU's (tie-swapped) list
            if same_g:
                o_out, o_lse = r.out[bi], r.lse[bi]
            else:
                qb = oracle.round_io(oracle.rope(q[b, kh * G:(kh + 1) * G, j * C:(j + 1) * C], op.pos0 + j * C, op.base,
                                                 op.pos_mod),
                                     op.io_bf16)
                o_out, o_lse, _ = oracle.attend_block(qb, r.k_rot, kv64, int(j), C, op.gs, op.F, op.L, g_gidx[j, :max(op.Kg, 0)])
            worst["out"] = max(worst["out"], float(np.abs(g_out[:, j * C:(j + 1) * C] - o_out).max()))
            worst["lse"] = max(worst["lse"], float(np.abs(g_lse[:, j * C:(j + 1) * C] - o_lse).max()))
    rep = dict(worst=worst, chunk=dataclasses.asdict(cchk), group=dataclasses.asdict(gchk), tol=tol)
    return rep


def assert_report(rep, w: W.Workload, n_checked: int, score_tol: float = 1e-6):
    wst, tol = rep["worst"], rep["tol"]
    assert rep["chunk"]["bad"] == 0 and rep["group"]["bad"] == 0, rep
    # ties within 1e-6 relative must be rare
    assert rep["chunk"]["tie_swaps"] + rep["group"]["tie_swaps"] + rep["group"]["skipped"] <= max(1, n_checked // 50), rep
    assert wst["out"] <= tol, rep
    assert wst["lse"] <= (1e-4 if w.dtype == "f32" else 2e-2), rep
    assert wst["pooled"] <= 2e-6 and wst["chunk_sum"] <= 2e-6 and wst["group_sum"] <= 4e-6, rep
    assert wst["score"] <= score_tol, rep
    # rotated keys: one storage rounding apart at most (fp32: ~1e-6 abs; bf16: 1 ulp of values up to ~8 -> 2^-4)
    assert wst["k_rot"] <= (4e-6 if w.dtype == "f32" else 0.0625), rep
    assert wst["q_rot"] <= (4e-6 if w.dtype == "f32" else 0.0625), rep
