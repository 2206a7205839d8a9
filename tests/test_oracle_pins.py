"""Pins for the CPU oracle: the oracle is checked against things OTHER than itself --
library routines (transformers' Qwen3 RoPE, torch SDPA, torch bf16 casts), closed forms, brute force, values the
paper prints (tests/golden/paper_constants.txt) and invariants the method must have.  No GPU needed.
"""
import dataclasses
import math
import os

import numpy as np
import pytest
import torch

import hga_workloads as W
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def golden():
    vals = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if "=" in line:
                k, v = line.split("=")
                vals[k.strip()] = float(v)
    return vals


# ----------------------------------------------------------------------------------------------------------------
# Independent helpers (numpy / torch; none of this is shared with oracle/ or the CUDA path)
# ----------------------------------------------------------------------------------------------------------------
def rope_complex(x, pos, base):
    """RoPE as a complex rotation: (x[i] + 1j*x[i+D/2]) * exp(1j*p*theta_i), fp64."""
    x = np.asarray(x, dtype=np.float64)
    D = x.shape[-1]
    h = D // 2
    theta = 1.0 / np.power(float(base), np.arange(h, dtype=np.float64) * 2.0 / D)
    z = (x[..., :h] + 1j * x[..., h:]) * np.exp(1j * np.asarray(pos, dtype=np.float64)[..., None] * theta)
    return np.concatenate([z.real, z.imag], axis=-1)


def sdpa_causal(q, k, v):
    """torch's scaled_dot_product_attention, causal, fp64 -- the paper's dense baseline."""
    q, k, v = (torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)) for a in (q, k, v))
    return torch.nn.functional.scaled_dot_product_attention(q[None], k[None].expand(1, q.shape[0], -1, -1),
                                                            v[None].expand(1, q.shape[0], -1, -1),
                                                            is_causal=True)[0].numpy()


def nearest_bf16(x):
    """Nearest bf16 to each fp64 value by brute force over the three neighbouring bf16 bit patterns
    (ties -> even mantissa).  Independent of the oracle's frexp-based rounding."""
    x = np.asarray(x, dtype=np.float64)
    c = torch.from_numpy(x.astype(np.float32)).to(torch.bfloat16)
    bits = c.view(torch.int16).to(torch.int32)
    best, best_err, best_odd = None, None, None
    for d in (-1, 0, 1):
        b = (bits + d).to(torch.int16)
        cand = b.view(torch.bfloat16).to(torch.float64).numpy()
        err = np.abs(cand - x)
        odd = (b.to(torch.int32) & 1).numpy()
        if best is None:
            best, best_err, best_odd = cand.copy(), err, odd
        else:
            take = (err < best_err) | ((err == best_err) & (odd < best_odd))
            best = np.where(take, cand, best)
            best_odd = np.where(take, odd, best_odd)
            best_err = np.where(take, err, best_err)
    return best


def small_problem(seed=0, G=2, N=512, D=32, base=1.0e4, clustered=False):
    w = W.Workload("t", 1, N, G, 1, D, "f32", base, topk_chunks=3, topk_groups=5,
                   dist="clustered" if clustered else "iid", n_clusters=4)
    q, k, v = W.generate(w, seed)
    return w, q[0], k[0, 0], v[0, 0]


# ----------------------------------------------------------------------------------------------------------------
# O1 RoPE
# ----------------------------------------------------------------------------------------------------------------
def test_rope_matches_transformers_qwen3():
    """R6 convention = the Qwen3 family's: compare with transformers' own rotary code."""
    from transformers import Qwen3Config
    from transformers.models.qwen3.modeling_qwen3 import Qwen3RotaryEmbedding, apply_rotary_pos_emb

    for D, base in ((64, 1.0e4), (128, 1.0e6)):
        cfg = Qwen3Config(hidden_size=256, num_attention_heads=4, num_key_value_heads=1, head_dim=D,
                          max_position_embeddings=4096, rope_theta=base)
        if getattr(cfg, "rope_parameters", None) is not None:
            cfg.rope_parameters["rope_theta"] = base
        emb = Qwen3RotaryEmbedding(cfg)
        x = torch.randn(1, 2, 48, D, dtype=torch.float64, generator=torch.Generator().manual_seed(1))
        pos = torch.arange(5, 53)[None]
        cos, sin = emb(x, pos)
        ref, _ = apply_rotary_pos_emb(x, x, cos, sin)
        got = oracle.rope(x[0].numpy().astype(np.float32), 5, base)
        # transformers builds cos/sin in fp32 -> ~1e-6 agreement at these small positions
        assert np.abs(got - ref[0].numpy()).max() < 2e-5


def test_rope_complex_form_and_invariants():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((3, 40, 64)).astype(np.float32)
    got = oracle.rope(x, 1000, 1.0e4)
    ref = rope_complex(x, np.arange(1000, 1040)[None, :].repeat(3, 0), 1.0e4)
    assert np.abs(got - ref).max() < 1e-12
    # norm preserving, identity at position 0
    assert np.allclose(np.linalg.norm(got, axis=-1), np.linalg.norm(x.astype(np.float64), axis=-1), rtol=1e-13)
    assert np.array_equal(oracle.rope(x[:, :1], 0, 1.0e4), x[:, :1].astype(np.float64))
    # relative-position property: <R(p)q, R(t)k> depends on p - t only
    q = rng.standard_normal((1, 64)).astype(np.float32)
    k = rng.standard_normal((1, 64)).astype(np.float32)
    a = oracle.rope(q, 900, 1.0e4) @ oracle.rope(k, 100, 1.0e4).T
    b = oracle.rope(q, 50900, 1.0e4) @ oracle.rope(k, 50100, 1.0e4).T
    assert abs(a - b).max() < 1e-9


def test_round_io_matches_torch_casts():
    rng = np.random.default_rng(3)
    x = rng.standard_normal(20000) * np.exp(rng.uniform(-8, 8, 20000))
    # make some exact ties: value halfway between two bf16 numbers
    t = torch.tensor([1.0, 1.0 + 2.0 ** -7, 3.0], dtype=torch.float64)
    ties = (t + 2.0 ** -8 * torch.tensor([1.0, 1.0, 2.0], dtype=torch.float64)).numpy()
    x = np.concatenate([x, ties, -ties])
    got = oracle.round_io(x, True)
    # a double that is exactly representable in fp32 casts to bf16 with one rounding in torch
    xf = x.astype(np.float32).astype(np.float64)
    same = xf == x
    ref = torch.from_numpy(x.astype(np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    assert same.sum() >= 6 and np.array_equal(got[same], ref[same])
    # general doubles: result is a bf16 value and the nearest one
    back = torch.from_numpy(got.astype(np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(back, got)
    ulp = 2.0 ** (np.floor(np.log2(np.abs(x))) - 7)
    assert np.all(np.abs(got - x) <= 0.5 * ulp * (1 + 1e-12))
    assert np.array_equal(got, nearest_bf16(x))
    assert np.array_equal(oracle.round_io(x, False), x.astype(np.float32).astype(np.float64))


# ----------------------------------------------------------------------------------------------------------------
# O2 summaries (P11, P12, P14, P15 and a closed form)
# ----------------------------------------------------------------------------------------------------------------
def test_summary_all_high_is_mean_of_rotated_keys_P11():
    w, q, k, v = small_problem(1, N=256, D=32)
    for span in (64, 16):
        s = oracle.summaries(k, span, 16, 7, w.rope_base)  # n_hi = D/2
        kr = rope_complex(k, np.arange(7, 7 + 256), w.rope_base)
        assert np.abs(s - kr.reshape(-1, span, 32).mean(1)).max() < 1e-12
    # ... and then q.S_c is the mean of the chunk's q.k logits (closed form, linearity)
    qr = rope_complex(q[0], np.arange(7, 7 + 256), w.rope_base)
    s = oracle.summaries(k, 64, 16, 7, w.rope_base)
    logits = qr[200] @ kr.T
    assert np.abs(qr[200] @ s.T - logits.reshape(-1, 64).mean(1)).max() < 1e-11


def test_summary_all_low_is_rotated_mean_of_raw_keys_P12():
    w, q, k, v = small_problem(2, N=256, D=32)
    for span in (64, 16):
        s = oracle.summaries(k, span, 0, 11, w.rope_base)
        raw_mean = k.astype(np.float64).reshape(-1, span, 32).mean(1)
        p_mid = 11 + np.arange(256 // span) * span + (span - 1) / 2.0  # R2: centroid of the span's positions
        assert np.abs(s - rope_complex(raw_mean, p_mid, w.rope_base)).max() < 1e-12


def test_summary_mixed_rule_pairwise_split():
    """Pairs < n_hi follow the 'rotate then average' rule, the others 'average then rotate'."""
    w, q, k, v = small_problem(3, N=128, D=32)
    n_hi = 5
    s = oracle.summaries(k, 64, n_hi, 0, w.rope_base)
    hi = oracle.summaries(k, 64, 16, 0, w.rope_base)
    lo = oracle.summaries(k, 64, 0, 0, w.rope_base)
    cols_hi = np.r_[0:n_hi, 16:16 + n_hi]
    cols_lo = np.r_[n_hi:16, 16 + n_hi:32]
    assert np.array_equal(s[:, cols_hi], hi[:, cols_hi]) and np.array_equal(s[:, cols_lo], lo[:, cols_lo])
    # default rule R1: wavelength 2*pi/theta_i <= span
    for D, base, span in ((64, 1e4, 64), (64, 1e4, 16), (128, 1e6, 64), (128, 1e6, 16)):
        theta = base ** (-2.0 * np.arange(D // 2) / D)
        assert oracle.default_n_hi(D, base, span) == int(np.sum(2 * np.pi / theta <= span))
    assert np.array_equal(oracle.summaries(k, 64, -1, 0, w.rope_base),
                          oracle.summaries(k, 64, oracle.default_n_hi(32, w.rope_base, 64), 0, w.rope_base))


def test_summary_constant_key_closed_form():
    """k_t = (1, 0) on every pair: rotate-then-average gives the Dirichlet kernel
    e^{i p_mid th} * sin(S th/2) / (S sin(th/2)); average-then-rotate gives e^{i p_mid th}."""
    D, S, base, pos0 = 16, 64, 100.0, 321
    k = np.zeros((2 * S, D), dtype=np.float32)
    k[:, : D // 2] = 1.0
    theta = base ** (-2.0 * np.arange(D // 2) / D)
    for n_hi in (D // 2, 0):
        s = oracle.summaries(k, S, n_hi, pos0, base)
        for sp in range(2):
            p_mid = pos0 + sp * S + (S - 1) / 2.0
            amp = np.sin(S * theta / 2) / (S * np.sin(theta / 2)) if n_hi else np.ones_like(theta)
            z = amp * np.exp(1j * p_mid * theta)
            assert np.abs(s[sp, : D // 2] - z.real).max() < 1e-12
            assert np.abs(s[sp, D // 2:] - z.imag).max() < 1e-12


def test_summary_chunk_group_consistency_P14_P15():
    w, q, k, v = small_problem(4, N=256, D=32)
    n_hi, pos0, h = 6, 40, 16
    sc = oracle.summaries(k, 64, n_hi, pos0, w.rope_base)
    sg = oracle.summaries(k, 16, n_hi, pos0, w.rope_base)
    hi_cols = np.r_[0:n_hi, h:h + n_hi]
    # pairs high at both levels: chunk summary = mean of its 4 group summaries
    assert np.abs(sc[:, hi_cols] - sg.reshape(-1, 4, 32).mean(1)[:, hi_cols]).max() < 1e-12
    # pairs low at both levels: un-rotating each summary at its own middle gives raw means, which nest
    pm_c = pos0 + np.arange(4) * 64 + 31.5
    pm_g = pos0 + np.arange(16) * 16 + 7.5
    raw_c = rope_complex(sc, -pm_c, w.rope_base)
    raw_g = rope_complex(sg, -pm_g, w.rope_base)
    lo_cols = np.r_[n_hi:h, h + n_hi:32]
    assert np.abs(raw_c[:, lo_cols] - raw_g.reshape(-1, 4, 32).mean(1)[:, lo_cols]).max() < 1e-12
    # P15: the low-pair summary computed from ROTATED keys, (1/S) sum_t R(p_mid - p_t) k_rot_t
    kr = rope_complex(k, pos0 + np.arange(256), w.rope_base)
    for c in range(4):
        acc = np.zeros(32)
        for t in range(64):
            acc += rope_complex(kr[c * 64 + t], pm_c[c] - (pos0 + c * 64 + t), w.rope_base)
        assert np.abs(acc[lo_cols] / 64 - sc[c, lo_cols]).max() < 1e-12


# ----------------------------------------------------------------------------------------------------------------
# O3 pooled query, O4/O5 routing (P8, P9, P10, P16, P17)
# ----------------------------------------------------------------------------------------------------------------
def test_pooled_query_linearity_P17():
    w, q, k, v = small_problem(5, G=3, N=256, D=32)
    qr = rope_complex(q, np.arange(256)[None].repeat(3, 0), w.rope_base)
    qbar = oracle.pool_queries(qr, 64)
    s = oracle.summaries(k, 64, -1, 0, w.rope_base)
    per_query = np.einsum("gtd,cd->gtc", qr, s)  # every query's own score against every summary
    mean_of_scores = per_query.reshape(3, 4, 64, 4).transpose(1, 0, 2, 3).reshape(4, 192, 4).mean(1)
    assert np.abs(qbar @ s.T - mean_of_scores).max() < 1e-12
    assert np.abs(qbar - qr.reshape(3, 4, 64, 32).mean(axis=(0, 2))).max() < 1e-13


def brute_topk(scores, idxs, k):
    order = np.lexsort((idxs, -scores))  # score descending, then index ascending
    return np.sort(idxs[order[:k]])


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_topk_equals_bruteforce_sort_P8(seed):
    rng = np.random.default_rng(seed)
    n_b, D, F, L, Kc = 40, 8, 2, 3, 5
    S_c = rng.integers(-3, 4, size=(n_b, D)).astype(np.float64)  # small integers -> many exact score ties
    S_c[17] = S_c[9]
    S_c[30] = S_c[9]
    qbar = rng.integers(-2, 3, size=D).astype(np.float64)
    for j in range(n_b):
        idx, sc, cnt, alls = oracle.route_chunks(qbar, S_c, j, F, L, Kc)
        cand = np.arange(F, max(F, j - max(L, 1)))
        assert cnt == min(Kc, len(cand))
        want = brute_topk(S_c[cand] @ qbar, cand, Kc) if len(cand) else np.array([], dtype=int)
        assert np.array_equal(idx[:cnt], want) and np.all(idx[cnt:] == -1)
        assert np.array_equal(sc[:cnt], S_c[idx[:cnt]] @ qbar)
        assert np.array_equal(np.isfinite(alls), np.isin(np.arange(n_b), cand))
        # group level: brute force over the C/gs groups of the selected chunks
        gpc, Kg = 4, 7
        S_g = rng.integers(-3, 4, size=(n_b * gpc, D)).astype(np.float64)
        gidx, gsc, gcnt, cs = oracle.route_groups(qbar, S_g, gpc, idx[:cnt], Kg)
        gcand = (idx[:cnt, None] * gpc + np.arange(gpc)[None]).reshape(-1)
        assert gcnt == min(Kg, len(gcand))
        gwant = brute_topk(S_g[gcand] @ qbar, gcand, Kg) if len(gcand) else np.array([], dtype=int)
        assert np.array_equal(gidx[:gcnt], gwant) and np.all(gidx[gcnt:] == -1)


def test_routing_invariances_P9_P10_P16():
    w, q, k, v = small_problem(6, G=2, N=1024, D=32, clustered=True)
    p = oracle.OracleParams(G=2, N=1024, D=32, F=1, L=1, Kc=3, Kg=5, base=w.rope_base)
    r0 = oracle.prefill_slice(p, q, k, v, attend=False)
    # P9: scaling Q by a power of two changes no index set
    r1 = oracle.prefill_slice(p, q * np.float32(4.0), k, v, attend=False)
    assert np.array_equal(r0.chunk_idx, r1.chunk_idx) and np.array_equal(r0.group_idx, r1.group_idx)
    # P16: a global position shift leaves scores and index sets unchanged (RoPE is relative)
    p2 = oracle.OracleParams(**{**p.__dict__, "pos0": 4096})
    r2 = oracle.prefill_slice(p2, q, k, v, attend=False)
    assert np.array_equal(r0.chunk_idx, r2.chunk_idx) and np.array_equal(r0.group_idx, r2.group_idx)
    assert np.nanmax(np.abs(r0.chunk_all_scores - r2.chunk_all_scores)) < 1e-9
    # P10: K_g = (C/gs)*K_c opens every group of every selected chunk (the "exact-token variant")
    p3 = oracle.OracleParams(**{**p.__dict__, "Kg": 12})
    r3 = oracle.prefill_slice(p3, q, k, v, attend=False)
    for b in range(16):
        ch = r3.chunk_idx[b][r3.chunk_idx[b] >= 0]
        want = (ch[:, None] * 4 + np.arange(4)[None]).reshape(-1)
        assert np.array_equal(r3.group_idx[b][: r3.n_groups[b]], want)
    # selected chunks are middle chunks only; sets are ascending and distinct
    for b in range(16):
        ch = r0.chunk_idx[b][: r0.n_chunks[b]]
        assert np.all(ch >= p.F) and np.all(ch < b - 1) and np.all(np.diff(ch) > 0)
        assert r0.n_chunks[b] == min(p.Kc, max(0, b - 1 - p.F))


# ----------------------------------------------------------------------------------------------------------------
# union set (P6, P7) and the numbers the paper prints
# ----------------------------------------------------------------------------------------------------------------
def test_union_set_contains_sink_local_current_and_paper_sizes_P6_P7():
    g = golden()
    C, gs = int(g["chunk_size"]), int(g["group_size"])
    F, L = int(g["needle_keep_first"]), int(g["needle_keep_last"])
    Kc, Kg = int(g["needle_topk_chunks"]), int(g["needle_topk_groups"])
    n_tok = int(g["needle_prompt_tokens"])
    n_chunks = -(-n_tok // C)
    assert n_chunks == int(g["needle_chunks"])
    j = n_chunks - 1
    rng = np.random.default_rng(0)
    # any K_g distinct middle groups (middle = chunks F .. j-L-1)
    groups = rng.choice(np.arange(F * 4, (j - L) * 4), size=Kg, replace=False)
    vis = oracle.key_set(j, C, gs, F, L, groups)
    assert vis[: F * C].all() and vis[(j - L) * C: j * C].all() and vis[j * C:].all()  # P6
    for gi in groups:
        assert vis[gi * gs:(gi + 1) * gs].all()
    assert vis.sum() == Kg * gs + (F + L + 1) * C == 1216  # P7
    assert round(100.0 * vis.sum() / n_tok, 1) == g["needle_sparsity_percent"]  # "approximately 1.9%"
    # the Qwen3 exact-token budget: K_c = 16 whole chunks -> 1024 routed tokens
    chunks16 = rng.choice(np.arange(2, j - 8), size=16, replace=False)
    groups16 = (chunks16[:, None] * 4 + np.arange(4)[None]).reshape(-1)
    vis16 = oracle.key_set(j, C, gs, 2, 8, groups16)
    assert vis16.sum() - (2 + 8 + 1) * C == int(g["qwen3_routed_budget_tokens"])
    # early blocks: sink and local overlap -> union, never double counted (R13)
    assert oracle.key_set(1, C, gs, 2, 8, []).sum() == 2 * C
    assert oracle.key_set(0, C, gs, 2, 8, []).sum() == C
    # -1 padding is ignored; future / current / duplicate / negative groups are rejected
    assert oracle.key_set(5, C, gs, 1, 1, [-1, 8, -1]).sum() == 3 * C + gs
    for bad in ([20], [24], [8, 8], [-2]):
        with pytest.raises(ValueError):
            oracle.key_set(5, C, gs, 1, 1, bad)


# ----------------------------------------------------------------------------------------------------------------
# O6 attention (P1..P5)
# ----------------------------------------------------------------------------------------------------------------
def test_full_coverage_equals_dense_causal_sdpa_P1():
    """PAPER.md:281 / Table 7: full chunk coverage must reproduce dense causal SDPA (< 1e-6)."""
    tol = golden()["full_coverage_max_abs"]
    for seed, (G, N, D, base) in enumerate([(2, 512, 32, 1.0e4), (4, 1024, 64, 1.0e4)]):
        w, q, k, v = small_problem(seed, G=G, N=N, D=D, base=base)
        p = oracle.OracleParams(G=G, N=N, D=D, F=1, L=1, Kc=N // 64, Kg=N // 16, base=base)
        r = oracle.prefill_slice(p, q, k, v)
        pos = np.arange(N)
        ref = sdpa_causal(rope_complex(q, pos[None].repeat(G, 0), base), rope_complex(k, pos, base), v)
        got = r.out.transpose(1, 0, 2, 3).reshape(G, N, D)
        assert np.abs(got - ref).max() < tol
        # the oracle's own Eq. (1) helper agrees with torch SDPA too
        kr = oracle.round_io(oracle.rope(k, 0, base), False)
        qb = oracle.round_io(oracle.rope(q[:, 128:192], 128, base), False)
        d_out, _ = oracle.dense_block(qb, kr, v.astype(np.float64), 2, 64)
        assert np.abs(d_out - ref[:, 128:192]).max() < tol


def test_early_blocks_equal_dense_for_any_budget_P2():
    w, q, k, v = small_problem(7, G=2, N=512, D=32)
    pos = np.arange(512)
    ref = sdpa_causal(rope_complex(q, pos[None].repeat(2, 0), w.rope_base), rope_complex(k, pos, w.rope_base), v)
    for F, L in ((1, 1), (2, 3), (0, 0)):
        p = oracle.OracleParams(G=2, N=512, D=32, F=F, L=L, Kc=0, Kg=0, base=w.rope_base)
        r = oracle.prefill_slice(p, q, k, v)
        n_dense = F + max(L, 1) + 1  # blocks 0 .. F+L_eff see every earlier token
        got = r.out.transpose(1, 0, 2, 3).reshape(2, 512, 32)
        assert np.abs(got[:, : n_dense * 64] - ref[:, : n_dense * 64]).max() < 1e-6
        assert np.abs(got[:, n_dense * 64:] - ref[:, n_dense * 64:]).max() > 1e-4  # later blocks really are sparse


def test_softmax_rows_sum_to_one_and_lse_P3():
    w, q, k, v = small_problem(8, G=2, N=512, D=32)
    p = oracle.OracleParams(G=2, N=512, D=32, Kc=2, Kg=3, base=w.rope_base)
    ones = np.ones_like(v)
    r = oracle.prefill_slice(p, q, k, ones)
    assert np.abs(r.out - 1.0).max() < 1e-14  # sum_j softmax_j * 1 == 1
    assert np.isfinite(r.lse).all()
    # lse against torch.logsumexp over the block's visible set
    j = 6
    vis = oracle.key_set(j, 64, 16, 1, 1, r.group_idx[j])
    kr = rope_complex(k, np.arange(512), w.rope_base).astype(np.float32).astype(np.float64)
    qr = rope_complex(q[1, j * 64: j * 64 + 64], np.arange(j * 64, j * 64 + 64), w.rope_base)
    qr = qr.astype(np.float32).astype(np.float64)
    for row in (0, 17, 63):
        keys = np.nonzero(vis[: j * 64 + row + 1])[0]
        logits = torch.from_numpy(qr[row] @ kr[keys].T / math.sqrt(32))
        assert abs(float(torch.logsumexp(logits, 0)) - r.lse[j, 1, row]) < 1e-12


def test_attention_against_direct_softmax_on_visible_set():
    """O6 on a sparse set, checked row by row with torch.softmax over the explicitly enumerated key set."""
    w, q, k, v = small_problem(9, G=2, N=512, D=32, clustered=True)
    p = oracle.OracleParams(G=2, N=512, D=32, Kc=2, Kg=3, base=w.rope_base, io_bf16=True)
    r = oracle.prefill_slice(p, q, k, v)
    to_bf16 = nearest_bf16
    kr = to_bf16(rope_complex(k, np.arange(512), w.rope_base))
    for j in (0, 1, 3, 7):
        vis = oracle.key_set(j, 64, 16, 1, 1, r.group_idx[j])
        for h in range(2):
            qr = to_bf16(rope_complex(q[h, j * 64: j * 64 + 64], np.arange(j * 64, j * 64 + 64), w.rope_base))
            for row in (0, 31, 63):
                keys = np.nonzero(vis[: j * 64 + row + 1])[0]
                pw = torch.softmax(torch.from_numpy(qr[row] @ kr[keys].T / math.sqrt(32)), 0).numpy()
                assert np.abs(pw @ v[keys].astype(np.float64) - r.out[j, h, row]).max() < 1e-12


def test_index_list_permutation_invariance_P4():
    w, q, k, v = small_problem(10, G=1, N=512, D=32)
    kr = oracle.rope(k, 0, w.rope_base)
    qb = oracle.rope(q[:, 448:512], 448, w.rope_base)
    groups = np.array([5, 9, 10, 17, 22, -1, -1], dtype=np.int32)
    a, la, na = oracle.attend_block(qb, kr, v, 7, 64, 16, 1, 1, groups)
    b, lb, nb = oracle.attend_block(qb, kr, v, 7, 64, 16, 1, 1, groups[::-1].copy())
    assert np.abs(a - b).max() < 1e-15 and np.array_equal(na, nb)
    assert np.array_equal(na, 5 * 16 + 2 * 64 + np.arange(1, 65))  # row r sees r+1 current tokens (causal)


def test_causality_P5():
    """Perturbing tokens after position t changes neither output row t nor any index set of earlier blocks."""
    w, q, k, v = small_problem(11, G=2, N=512, D=32)
    p = oracle.OracleParams(G=2, N=512, D=32, Kc=2, Kg=3, base=w.rope_base)
    r0 = oracle.prefill_slice(p, q, k, v)
    t = 300  # inside block 4
    q2, k2, v2 = q.copy(), k.copy(), v.copy()
    q2[:, t + 1:] += 1.0
    k2[t + 1:] -= 2.0
    v2[t + 1:] *= 3.0
    r1 = oracle.prefill_slice(p, q2, k2, v2)
    jb, row = divmod(t, 64)
    assert np.array_equal(r0.out[:jb], r1.out[:jb])
    assert np.array_equal(r0.out[jb, :, : row + 1], r1.out[jb, :, : row + 1])
    assert not np.array_equal(r0.out[jb, :, row + 1:], r1.out[jb, :, row + 1:])
    assert np.array_equal(r0.chunk_idx[:jb], r1.chunk_idx[:jb]) and np.array_equal(r0.group_idx[:jb], r1.group_idx[:jb])


def test_bad_inputs_are_rejected():
    w, q, k, v = small_problem(12, G=1, N=128, D=32)
    p = oracle.OracleParams(G=1, N=128, D=32, base=w.rope_base)
    k2 = k.copy()
    k2[3, 3] = np.nan
    with pytest.raises(ValueError):
        oracle.prefill_slice(p, q, k2, v)
    with pytest.raises(ValueError):  # R12: partial last chunk is not a closed chunk
        oracle.prefill_slice(oracle.OracleParams(G=1, N=100, D=32), q[:, :100], k[:100], v[:100])


def test_config1_tiny_cpu_checkable():
    """BASELINE.json configs[0]: runs in seconds; top-k = all chunks equals dense causal attention."""
    w = W.get("c1")
    q, k, v = W.generate(w, 0)
    p = oracle.params_from_workload(w)
    r = oracle.prefill_slice(p, q[0], k[0, 0], v[0, 0])
    assert r.out.shape == (16, 4, 64, 64)
    assert np.all(r.n_chunks == np.minimum(4, np.maximum(0, np.arange(16) - 2)))
    assert np.all(r.n_groups == np.minimum(8, 4 * r.n_chunks))
    p_all = oracle.OracleParams(**{**p.__dict__, "Kc": 16, "Kg": 64})
    r_all = oracle.prefill_slice(p_all, q[0], k[0, 0], v[0, 0])
    pos = np.arange(1024)
    ref = sdpa_causal(rope_complex(q[0], pos[None].repeat(4, 0), 1e4), rope_complex(k[0, 0], pos, 1e4), v[0, 0])
    assert np.abs(r_all.out.transpose(1, 0, 2, 3).reshape(4, 1024, 64) - ref).max() < 1e-6


# ----------------------------------------------------------------------------------------------------------------
# N1 streaming step (chunk-by-chunk prefill, decode, ragged tail): Table 7 :291-292
# ----------------------------------------------------------------------------------------------------------------
def test_step_decode_full_coverage_equals_dense_recompute():
    """Table 7 "HA decode vs full recompute": token-by-token steps with full coverage reproduce the dense causal row;
    the step is handed only tokens 0..t, so the future cannot leak."""
    tol = golden()["full_coverage_max_abs"]
    w, q, k, v = small_problem(21, G=2, N=320, D=32)
    pos = np.arange(320)
    ref = sdpa_causal(rope_complex(q, pos[None].repeat(2, 0), w.rope_base), rope_complex(k, pos, w.rope_base), v)
    p = oracle.OracleParams(G=2, N=320, D=32, F=1, L=1, Kc=5, Kg=20, base=w.rope_base)
    for t in (0, 1, 63, 64, 65, 127, 200, 255, 256, 300, 319):
        r = oracle.step(p, q[:, t:t + 1], k[:t + 1], v[:t + 1], t, t + 1)
        assert r.out.shape == (2, 1, 32)
        assert np.abs(r.out[:, 0] - ref[:, t]).max() < tol
    # ragged prompt tail: window [256, 300) of the unfinished chunk 4, full coverage
    r = oracle.step(p, q[:, 256:300], k[:300], v[:300], 256, 300)
    assert np.abs(r.out - ref[:, 256:300]).max() < tol


def test_step_sparse_window_against_direct_computation():
    """A sparse step checked end to end against numpy/torch written here: pooled query = mean over the window's rows
    and heads (R17), brute-force sort over the closed middle chunks and over the kept chunks' groups, softmax over
    the explicitly enumerated key set.  Summaries come from oracle.summaries (pinned by P11-P15)."""
    base, G, N, D, F, L, Kc, Kg = 1.0e4, 2, 640, 32, 1, 2, 3, 5
    w, q, k, v = small_problem(22, G=G, N=N, D=D, clustered=True)
    p = oracle.OracleParams(G=G, N=N, D=D, F=F, L=L, Kc=Kc, Kg=Kg, base=base, io_bf16=True)
    kr_all = rope_complex(k, np.arange(N), base)
    for (t0, t1) in ((576, 640), (600, 601), (639, 640), (448, 470), (130, 131), (64, 128)):
        j = t0 // 64
        r = oracle.step(p, q[:, t0:t1], k[:t1], v[:t1], t0, t1)
        qr = rope_complex(q[:, t0:t1], np.arange(t0, t1)[None].repeat(G, 0), base)
        qbar = qr.reshape(-1, D).mean(0)
        assert np.abs(qbar - r.q_pooled).max() < 1e-13
        S_c = oracle.summaries(k[: j * 64], 64, oracle.default_n_hi(D, base, 64), 0, base) if j else np.zeros((0, D))
        S_g = oracle.summaries(k[: j * 64], 16, oracle.default_n_hi(D, base, 16), 0, base) if j else np.zeros((0, D))
        cand = list(range(F, j - L))
        order = sorted(cand, key=lambda c: (-float(S_c[c] @ qbar), c))[:Kc]
        assert sorted(order) == [c for c in r.chunk_idx if c >= 0] and r.n_chunks == len(order)
        gc = [4 * c + u for c in sorted(order) for u in range(4)]
        gorder = sorted(sorted(gc, key=lambda g: (-float(S_g[g] @ qbar), g))[:Kg])
        assert gorder == [g for g in r.group_idx if g >= 0] and r.n_groups == len(gorder)
        # union set: sink chunks, local chunks, opened groups, current chunk up to the query
        chunks = set(range(min(F, j))) | set(range(max(0, j - L), j))
        base_keys = sorted({u for c in chunks for u in range(c * 64, c * 64 + 64)} |
                           {u for g in gorder for u in range(g * 16, g * 16 + 16)})
        kr, qrb = nearest_bf16(kr_all[:t1]), nearest_bf16(qr)
        for h in range(G):
            for row in sorted({0, (t1 - t0) // 2, t1 - t0 - 1}):
                keys = np.array(base_keys + list(range(j * 64, t0 + row + 1)), dtype=np.int64)
                pw = torch.softmax(torch.from_numpy(qrb[h, row] @ kr[keys].T / math.sqrt(D)), 0).numpy()
                assert np.abs(pw @ v[keys].astype(np.float64) - r.out[h, row]).max() < 1e-12


def test_step_chunk_by_chunk_equals_vectorised_prefill():
    """"vectorized prefill and chunk-by-chunk decode must agree up to floating-point noise" -- in the
    oracle both run the same arithmetic in the same order, so whole-block steps agree exactly."""
    w, q, k, v = small_problem(23, G=2, N=512, D=32, clustered=True)
    p = oracle.OracleParams(G=2, N=512, D=32, Kc=2, Kg=5, base=w.rope_base, io_bf16=True)
    full = oracle.prefill_slice(p, q, k, v)
    for j in range(8):
        r = oracle.step(p, q[:, j * 64:(j + 1) * 64], k[:(j + 1) * 64], v[:(j + 1) * 64], j * 64, (j + 1) * 64)
        assert np.array_equal(r.chunk_idx, full.chunk_idx[j]) and np.array_equal(r.group_idx, full.group_idx[j])
        assert np.array_equal(r.out, full.out[j]) and np.array_equal(r.lse, full.lse[j])
        assert np.array_equal(r.q_pooled, full.q_pooled[j])
    with pytest.raises(ValueError):
        oracle.step(p, q[:, 60:70], k[:70], v[:70], 60, 70)  # a step never spans two chunks


def test_c5_needle_group_is_routed_by_the_oracle():
    """BASELINE.json configs[4]: the planted 16-token needle group (cosine 0.9 with the final block's pooled rotated
    query) must appear in the routed set of the final block, at 10 / 50 / 90 % depth.  Stand-in for PAPER.md:214-231."""
    import needle

    w = W.get("c5")
    q, k, v = W.generate(w, 0)
    op = oracle.params_from_workload(w)
    G = w.gqa
    for depth in needle.DEPTHS:
        kk = k.copy()
        g_star = needle.plant(w, q, kk, depth)
        assert g_star == int(depth * w.n_groups_total) and (g_star * 16) // 64 not in (0, w.n_blocks - 2, w.n_blocks - 1)
        # cosine of the planted rotated keys with the pooled rotated query of the final block is 0.9 (before rounding)
        kh = 1
        kr = oracle.rope(kk[0, kh, g_star * 16:(g_star + 1) * 16], g_star * 16, w.rope_base)
        qb = oracle.pool_queries(oracle.rope(q[0, kh * G:(kh + 1) * G, -64:], w.seq - 64, w.rope_base), 64)[0]
        cos = kr @ qb / (np.linalg.norm(kr, axis=1) * np.linalg.norm(qb))
        assert np.all(np.abs(cos - 0.9) < 5e-3)
        r = oracle.prefill_slice(op, q[0, kh * G:(kh + 1) * G], kk[0, kh], v[0, kh], blocks=[w.n_blocks - 1],
                                 attend=False, want_k_rot=False)
        assert g_star // 4 in r.chunk_idx[0] and g_star in r.group_idx[0]
        # without the needle the same group is NOT routed (the planted signal, not chance, selects it)
        r0 = oracle.prefill_slice(op, q[0, kh * G:(kh + 1) * G], k[0, kh], v[0, kh], blocks=[w.n_blocks - 1],
                                  attend=False, want_k_rot=False)
        assert g_star not in r0.group_idx[0]


# ----------------------------------------------------------------------------------------------------------------
# N3 variants: wrapped RoPE position index and alternative high-frequency thresholds (R1)
# ----------------------------------------------------------------------------------------------------------------
def test_rope_position_wrap_matches_complex_rotation_at_wrapped_positions():
    M = int(golden()["rope_wrap_modulus"])
    assert M == 65536
    rng = np.random.default_rng(3)
    x = rng.standard_normal((192, 32)).astype(np.float32)
    # rows straddle the wrap: positions M-64 .. M+127 become M-64 .. M-1, 0 .. 127
    got = oracle.rope(x, M - 64, 1.0e4, pos_mod=M)
    pos = (np.arange(M - 64, M + 128) % M)
    assert np.abs(got - rope_complex(x, pos, 1.0e4)).max() < 1e-9
    # after the wrap the rotation is the un-wrapped rotation of position p - M (periodicity of the index, not of RoPE)
    assert np.array_equal(got[64:], oracle.rope(x[64:], 0, 1.0e4))
    # a modulus no position reaches changes nothing, bit for bit
    assert np.array_equal(oracle.rope(x, 100, 1.0e4, pos_mod=M), oracle.rope(x, 100, 1.0e4))
    # and wrapping is NOT the identity: the pair with theta = 1 (i = 0) differs at position M vs 0 unless M*1 = 2*pi*k
    assert np.abs(got[64:] - oracle.rope(x[64:], M, 1.0e4)).max() > 1e-2


def test_summaries_under_position_wrap():
    w, q, k, v = small_problem(4, N=256, D=32)
    M = 128  # spans 0,1 sit at positions 64..127, spans 2,3 wrap to 0..127 (pos0 = 64)
    pos = (64 + np.arange(256)) % M
    for span in (64, 16):
        # all pairs high: mean of the keys rotated at their wrapped positions (P11 under the wrap)
        s = oracle.summaries(k, span, 16, 64, w.rope_base, pos_mod=M)
        assert np.abs(s - rope_complex(k, pos, w.rope_base).reshape(-1, span, 32).mean(1)).max() < 1e-12
        # all pairs low: raw mean rotated at the wrapped start + (S-1)/2 (P12 under the wrap, reading R18)
        s = oracle.summaries(k, span, 0, 64, w.rope_base, pos_mod=M)
        p_mid = pos.reshape(-1, span)[:, 0] + (span - 1) / 2.0
        raw_mean = k.astype(np.float64).reshape(-1, span, 32).mean(1)
        assert np.abs(s - rope_complex(raw_mean, p_mid, w.rope_base)).max() < 1e-12
    # a span may not straddle a wrap: modulus or pos0 off the span grid is rejected
    with pytest.raises(Exception):
        oracle.summaries(k, 64, 4, 0, w.rope_base, pos_mod=96)
    with pytest.raises(Exception):
        oracle.summaries(k, 64, 4, 32, w.rope_base, pos_mod=128)


def test_prefill_under_position_wrap_is_a_global_shift_and_leaves_routing_unchanged():
    w, q, k, v = small_problem(8, G=2, N=512, D=32, clustered=True)
    base = dict(G=2, N=512, D=32, F=1, L=1, Kc=3, Kg=5, base=w.rope_base)
    r_plain = oracle.prefill_slice(oracle.OracleParams(**base), q, k, v)
    # a sequence that starts exactly at the modulus is position-for-position the sequence that starts at 0
    r_wrap = oracle.prefill_slice(oracle.OracleParams(**base, pos0=1024, pos_mod=1024), q, k, v)
    assert np.array_equal(r_plain.chunk_idx, r_wrap.chunk_idx) and np.array_equal(r_plain.group_idx, r_wrap.group_idx)
    assert np.array_equal(r_plain.out, r_wrap.out)
    # a modulus beyond the last position is inert
    r_big = oracle.prefill_slice(oracle.OracleParams(**base, pos_mod=65536), q, k, v)
    assert np.array_equal(r_plain.out, r_big.out) and np.array_equal(r_plain.group_idx, r_big.group_idx)
    # a wrap in the middle of the sequence changes the logits (positions 256.. alias 0..) but the routing algorithm
    # is "unchanged": same budgets, same visibility windows, still exact softmax over the union set
    pw = oracle.OracleParams(**base, pos_mod=256)
    r_mid = oracle.prefill_slice(pw, q, k, v)
    assert np.array_equal(r_mid.n_chunks, r_plain.n_chunks) and np.array_equal(r_mid.n_groups, r_plain.n_groups)
    assert np.abs(r_mid.out - r_plain.out).max() > 1e-3
    # ... checked against a direct computation: rotate at wrapped positions, softmax over the oracle's own key set
    pos = np.arange(512) % 256
    qr = rope_complex(q, pos, w.rope_base)
    kr = rope_complex(k, pos, w.rope_base)
    j = 7
    keys = oracle.key_set(j, 64, 16, 1, 1, r_mid.group_idx[j])
    for t in (j * 64, j * 64 + 37, j * 64 + 63):
        vis = np.flatnonzero(keys & (np.arange(keys.size) <= t))  # union set, causal cut inside the block
        lg = (qr[1, t] @ kr[vis].T) / math.sqrt(32)
        pr = np.exp(lg - lg.max())
        ref = (pr / pr.sum()) @ v[vis].astype(np.float64)
        assert np.abs(r_mid.out[j, 1, t - j * 64] - ref).max() < 1e-5  # Q_rot/K_rot are stored as fp32 (R7)


def test_n_hi_rules_closed_form():
    # theta_i = base^(-2i/D) decreases with i, so each rule keeps pairs i <= (D/2) ln(S/c) / ln(base):
    # c = 2*pi (wavelength <= span), pi (half a turn), 1 (one radian)
    for D, base in ((64, 1.0e4), (128, 1.0e6), (32, 100.0)):
        for span in (64, 16):
            for rule, c in ((0, 2 * math.pi), (1, math.pi), (2, 1.0)):
                x = (D / 2) * math.log(span / c) / math.log(base)
                want = min(D // 2, max(0, math.floor(x) + 1)) if x >= 0 else 0
                assert oracle.n_hi_rule(D, base, span, rule) == want, (D, base, span, rule)
            assert oracle.n_hi_rule(D, base, span, 0) == oracle.default_n_hi(D, base, span)
    # the counts SURVEY.md 8(c) R1 lists for the two model shapes (chunk / group)
    assert [oracle.n_hi_rule(64, 1e4, s, r) for r in range(3) for s in (64, 16)] == [9, 4, 11, 6, 15, 10]
    assert [oracle.n_hi_rule(128, 1e6, s, r) for r in range(3) for s in (64, 16)] == [11, 5, 14, 8, 20, 13]
    with pytest.raises(ValueError):
        oracle.n_hi_rule(64, 1e4, 64, 3)


# ---------------------------------------------------------------------------------------------------------------
# N3: R4's alternative -- a block's score of a candidate is the MAX over its 64*G per-query scores (PAPER.md:33, 45,
# 97 leave the reduction open; reading R19: per-query scores use the rotated queries as stored)
# ---------------------------------------------------------------------------------------------------------------
def _max_mode_inputs(seed, n_b=24, D=32, rows=48):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((rows, D)), rng.standard_normal((n_b, D)), rng.standard_normal((n_b * 4, D))


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_max_mode_equals_bruteforce_on_tiny_inputs(seed):
    """score(c) = max_r q_r . S[c] written out with numpy, then a full lexsort (score desc, index asc) -- the
    definition, not the oracle's routine; constructed exact ties included."""
    q_rows, S_c, S_g = _max_mode_inputs(seed)
    S_c[7] = S_c[5]   # exact ties between candidates
    S_c[11] = S_c[5]
    F, L, Kc, Kg, gpc = 1, 2, 6, 9, 4
    for j in (0, 1, 3, 4, 9, 23):
        idx, sc, cnt, alls = oracle.route_chunks_max(q_rows, S_c, j, F, L, Kc)
        cand = np.arange(F, max(F, j - max(L, 1)))
        full = (q_rows @ S_c.T).max(axis=0)
        order = cand[np.lexsort((cand, -full[cand]))][:Kc]
        assert cnt == len(order) and np.array_equal(idx[:cnt], np.sort(order)) and np.all(idx[cnt:] == -1)
        assert np.allclose(alls[cand], full[cand], rtol=1e-13, atol=1e-13) and np.isnan(np.delete(alls, cand)).all()
        if cnt:
            gc = (np.sort(order)[:, None] * gpc + np.arange(gpc)[None]).reshape(-1)
            gfull = (q_rows @ S_g.T).max(axis=0)
            gorder = gc[np.lexsort((gc, -gfull[gc]))][:Kg]
            gidx, gsc, gcnt, gcand = oracle.route_groups_max(q_rows, S_g, gpc, idx[:cnt], Kg)
            assert gcnt == len(gorder) and np.array_equal(gidx[:gcnt], np.sort(gorder))
            assert np.allclose(gcand, gfull[gc], rtol=1e-13, atol=1e-13)


def test_max_mode_reduces_to_mean_mode_when_all_queries_are_equal_and_dominates_it():
    q_rows, S_c, S_g = _max_mode_inputs(5)
    one = np.repeat(q_rows[:1], 48, axis=0)
    for j in (6, 15, 23):
        a = oracle.route_chunks_max(one, S_c, j, 1, 1, 5)
        b = oracle.route_chunks(one[0], S_c, j, 1, 1, 5)
        assert np.array_equal(a[0], b[0]) and a[2] == b[2] and np.allclose(a[1], b[1], rtol=1e-14)
        ga = oracle.route_groups_max(one, S_g, 4, a[0][:a[2]], 7)
        gb = oracle.route_groups(one[0], S_g, 4, b[0][:b[2]], 7)
        assert np.array_equal(ga[0], gb[0]) and np.allclose(ga[3], gb[3], rtol=1e-14)
        # max over queries >= mean over queries = pooled-query score (P17 linearity), candidate by candidate
        mx = oracle.route_chunks_max(q_rows, S_c, j, 1, 1, 5)[3]
        mean = oracle.route_chunks(q_rows.mean(axis=0), S_c, j, 1, 1, 5)[3]
        cand = ~np.isnan(mx)
        assert np.array_equal(cand, ~np.isnan(mean)) and np.all(mx[cand] >= mean[cand] - 1e-12)


def test_max_mode_invariances():
    """Row order of the block does not matter; scaling every query by alpha > 0 keeps the sets; a single dominant query
    decides the selection alone."""
    q_rows, S_c, _ = _max_mode_inputs(9)
    base = oracle.route_chunks_max(q_rows, S_c, 20, 1, 1, 6)
    perm = np.random.default_rng(1).permutation(len(q_rows))
    assert np.array_equal(oracle.route_chunks_max(q_rows[perm], S_c, 20, 1, 1, 6)[0], base[0])
    assert np.array_equal(oracle.route_chunks_max(3.5 * q_rows, S_c, 20, 1, 1, 6)[0], base[0])
    big = q_rows.copy()
    big[17] = 100.0 * S_c[9]   # one query aligned with candidate 9: its score dwarfs every other
    idx = oracle.route_chunks_max(big, S_c, 20, 1, 1, 1)[0]
    assert idx[0] == 9
    alone = oracle.route_chunks(big[17], S_c, 20, 1, 1, 6)[0]     # the mean rule applied to that single query
    assert 9 in alone


def test_max_mode_prefill_slice_causality_and_attention_on_its_own_sets():
    """Whole-slice run with route_max: (a) index sets equal route_*_max applied to the stored rotated queries (R19);
    (b) sets of earlier blocks ignore later tokens; (c) O6 is the exact softmax over the resulting union
    set (same attention code as the mean rule, checked through dense_block on full coverage)."""
    w = W.Workload("mx", 1, 1024, 4, 2, 64, "bf16", 1e4, topk_chunks=3, topk_groups=7, n_clusters=4)
    q, k, v = W.generate(w, 3)
    op = dataclasses.replace(oracle.params_from_workload(w), route_max=True)
    r = oracle.prefill_slice(op, q[0, :2], k[0, 0], v[0, 0])
    rm = oracle.prefill_slice(dataclasses.replace(op, route_max=False), q[0, :2], k[0, 0], v[0, 0])
    assert not np.array_equal(r.chunk_idx, rm.chunk_idx)  # the two rules do differ on this input
    for j in (5, 9, 15):
        qb = oracle.round_io(oracle.rope(q[0, :2, j * 64:(j + 1) * 64], j * 64, w.rope_base), True)
        idx, sc, cnt, alls = oracle.route_chunks_max(qb, r.chunk_sum, j, 1, 1, 3)
        assert np.array_equal(idx, r.chunk_idx[j]) and cnt == r.n_chunks[j]
        gidx = oracle.route_groups_max(qb, r.group_sum, 4, idx[:cnt], 7)[0]
        assert np.array_equal(gidx, r.group_idx[j])
        o, l, _ = oracle.attend_block(qb, r.k_rot, v[0, 0].astype(np.float64), j, 64, 16, 1, 1, r.group_idx[j])
        assert np.abs(o - r.out[j]).max() < 1e-12
    k2, q2 = k.copy(), q.copy()
    k2[0, 0, 640:] += 1.0
    q2[0, :2, 640:] -= 0.5
    r2 = oracle.prefill_slice(op, q2[0, :2], k2[0, 0], v[0, 0])
    assert np.array_equal(r2.chunk_idx[:10], r.chunk_idx[:10]) and np.array_equal(r2.group_idx[:10], r.group_idx[:10])
    assert np.abs(r2.out[:10] - r.out[:10]).max() == 0.0
    # full coverage under the max rule is still dense causal attention (Eq. (1))
    opd = dataclasses.replace(op, Kc=16, Kg=64)
    rd = oracle.prefill_slice(opd, q[0, :2], k[0, 0], v[0, 0], blocks=[15])
    qb = oracle.round_io(oracle.rope(q[0, :2, 960:1024], 960, w.rope_base), True)
    ref, _ = oracle.dense_block(qb, rd.k_rot, v[0, 0].astype(np.float64), 15, 64)
    assert np.abs(rd.out[0] - ref).max() < 1e-10
