"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI binding, against the CPU oracle on the same
seeded inputs.  Element-by-element at sizes the oracle finishes in seconds; sampled blocks at BASELINE.json's full
sizes in the launch configuration bench.py times.
"""
import dataclasses

import numpy as np
import pytest
import torch

import hga_workloads as W
import oracle
import paper_2606_30709_b200 as hga
from paper_2606_30709_b200.binding import (ATTEND_AUTO, ATTEND_SIMT, ATTEND_TCGEN05, ATTEND_TCGEN05_ITEM,
                                             ATTEND_TCGEN05_PAIR, HGA_BF16, HGA_F32)

import parity

pytestmark = pytest.mark.gpu


def _all_slices(w):
    return [(b, kh) for b in range(w.batch) for kh in range(w.n_kv_heads)]


def _sample_blocks(n_b, n, seed):
    """first blocks (dense regime, partial budgets), a ragged middle sample, and the last block."""
    rng = np.random.default_rng(seed)
    fixed = [0, 1, 2, 3, 4, 5, n_b // 2, n_b - 2, n_b - 1]
    extra = rng.choice(np.arange(6, n_b - 2), size=max(0, n - len(fixed)), replace=False).tolist() if n_b > 16 else []
    return sorted(set(j for j in fixed + extra if 0 <= j < n_b))


# ---------------------------------------------------------------------------------------------------------------
# config 1: tiny, fp32, every element, three seeds; SIMT fp32 kernel (the 1e-4 path)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_c1_full_parity_fp32(seed):
    w = W.get("c1")
    q, k, v = W.generate(w, seed)
    p, buf = parity.run_gpu(w, q, k, v)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks)
    assert rep["worst"]["out"] <= 1e-4


def test_c1_topk_all_equals_dense_causal():
    """BASELINE.json configs[0]: 'also run with top-k = all chunks, which must equal dense causal attention'."""
    w = W.get("c1")
    q, k, v = W.generate(w, 0)
    p, buf = parity.run_gpu(w, q, k, v, topk_chunks=16, topk_groups=64)
    op = dataclasses.replace(oracle.params_from_workload(w), Kc=16, Kg=64)
    kr = oracle.round_io(oracle.rope(k[0, 0], 0, w.rope_base), False)
    got = buf.out[0].cpu().numpy().astype(np.float64)
    for j in range(w.n_blocks):
        qb = oracle.round_io(oracle.rope(q[0, :, j * 64:(j + 1) * 64], j * 64, w.rope_base), False)
        ref, _ = oracle.dense_block(qb, kr, v[0, 0].astype(np.float64), j, 64)
        assert np.abs(got[:, j * 64:(j + 1) * 64] - ref).max() <= 1e-4
    # and against torch SDPA on the GPU's own rotated tensors (secondary sanity check, not the oracle)
    v_dev = torch.from_numpy(v).cuda().expand(-1, 4, -1, -1)
    ref2 = torch.nn.functional.scaled_dot_product_attention(buf.q_rot, buf.k_rot.expand(-1, 4, -1, -1), v_dev,
                                                            is_causal=True)
    assert (buf.out - ref2).abs().max().item() <= 1e-4


# ---------------------------------------------------------------------------------------------------------------
# small bf16 problems covering ragged tails, G in {1, 2, 3, 8}, D in {64, 128}, both attend kernels
# ---------------------------------------------------------------------------------------------------------------
SMALL = [
    # name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L
    ("d64_g1", 2, 1024, 4, 4, 64, 1e4, 4, 9, 1, 1),
    ("d128_g8", 1, 2048, 16, 2, 128, 1e6, 6, 24, 1, 1),
    ("d128_g3", 1, 1536, 6, 2, 128, 1e6, 5, 7, 2, 3),
    ("d64_g2_nolocal", 1, 1024, 4, 2, 64, 1e4, 3, 5, 0, 0),
    ("d128_g2_pos0", 1, 1024, 4, 2, 128, 1e6, 4, 16, 1, 2),
    ("d64_g1_kc40", 1, 4096, 2, 2, 64, 1e4, 40, 50, 1, 1),   # K_c > 32: the generic selection kernel
    ("d64_g2_kg_lt", 1, 2048, 4, 2, 64, 1e4, 20, 33, 1, 1),  # 80 group candidates, non-trivial top-33
    # split mode of the persistent S4 kernel (G <= 2): even / odd key-tile counts, a 64-key partial tail, two stages
    ("d64_g1_two_tiles", 1, 1024, 2, 2, 64, 1e4, 2, 4, 1, 1),     # 256 keys = 2 tiles
    ("d128_g1_three_tiles", 1, 1024, 2, 2, 128, 1e6, 2, 8, 1, 1),  # 320 keys = 2.5 tiles, D 128 (two K/V stages)
    ("d64_g2_five_tiles", 1, 2048, 4, 2, 64, 1e4, 8, 28, 0, 1),   # 576 keys = 4.5 tiles, no sink
]


@pytest.mark.parametrize("impl", [ATTEND_SIMT, ATTEND_TCGEN05, ATTEND_TCGEN05_ITEM])
@pytest.mark.parametrize("cfg", SMALL, ids=[c[0] for c in SMALL])
def test_small_bf16_full_parity(cfg, impl):
    name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L = cfg
    w = W.Workload(name, B, N, Hq, Hkv, D, "bf16", base, n_sink=F, n_local=L, topk_chunks=Kc, topk_groups=Kg,
                   n_clusters=8, pos0=(40000 if "pos0" in name else 0))
    q, k, v = W.generate(w, 7)
    p, buf = parity.run_gpu(w, q, k, v, attend_impl=impl)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks * B * Hkv)


# N3 variants: wrapped RoPE position index and the alternative high-frequency
# thresholds -- S0..S3 feel them, S4 only through the rotated tensors and the index lists
VARIANTS = [
    # name, D, base, pos0, rope_pos_mod, n_hi rule
    ("wrap_mid_sequence", 128, 1e6, 0, 1024, 0),      # positions 1024.. alias 0..
    ("wrap_pos0_offset", 64, 1e4, 65536 - 512, 65536, 0),  # the paper's modulus, crossed at token 512
    ("wrap_inert", 64, 1e4, 0, 65536, 0),
    ("n_hi_half_turn", 128, 1e6, 0, 0, 1),
    ("n_hi_one_radian_wrap", 64, 1e4, 128, 2048, 2),
]


@pytest.mark.parametrize("cfg", VARIANTS, ids=[c[0] for c in VARIANTS])
def test_variants_position_wrap_and_n_hi_rules(cfg):
    name, D, base, pos0, mod, rule = cfg
    n_hi_c = hga.hga_n_hi_rule(D, base, 64, rule) if rule else -1
    n_hi_g = hga.hga_n_hi_rule(D, base, 16, rule) if rule else -1
    if rule:
        assert (n_hi_c, n_hi_g) == (oracle.n_hi_rule(D, base, 64, rule), oracle.n_hi_rule(D, base, 16, rule))
    w = W.Workload(name, 1, 2048, 4, 2, D, "bf16", base, topk_chunks=5, topk_groups=11, n_clusters=8, pos0=pos0,
                   rope_pos_mod=mod, n_hi_chunk=n_hi_c, n_hi_group=n_hi_g)
    q, k, v = W.generate(w, 13)
    p, buf = parity.run_gpu(w, q, k, v)
    assert p.rope_pos_mod == mod and p.n_hi_chunk == n_hi_c
    rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks * 2)
    if name == "wrap_inert":  # bit-identical to the run without the modulus
        p0, buf0 = parity.run_gpu(dataclasses.replace(w, rope_pos_mod=0), q, k, v)
        assert torch.equal(buf.out, buf0.out) and torch.equal(buf.group_idx, buf0.group_idx)
    if name == "wrap_mid_sequence":  # and the wrap is not a no-op
        p0, buf0 = parity.run_gpu(dataclasses.replace(w, rope_pos_mod=0), q, k, v)
        assert not torch.equal(buf.k_rot, buf0.k_rot)


@pytest.mark.parametrize("impl", [ATTEND_SIMT, ATTEND_TCGEN05, ATTEND_TCGEN05_ITEM])
def test_bf16_full_coverage_equals_dense(impl):
    """full chunk coverage must reproduce dense causal attention (bf16 bar: 2e-2)."""
    w = W.Workload("dense", 1, 1024, 8, 2, 128, "bf16", 1e6, topk_chunks=16, topk_groups=64, n_clusters=4)
    q, k, v = W.generate(w, 3)
    p, buf = parity.run_gpu(w, q, k, v, attend_impl=impl)
    kr = oracle.round_io(oracle.rope(k[0], 0, w.rope_base), True)
    got = buf.out[0].cpu().numpy().astype(np.float64)
    for kh in range(2):
        for j in (0, 1, 7, 15):
            qb = oracle.round_io(oracle.rope(q[0, kh * 4:(kh + 1) * 4, j * 64:(j + 1) * 64], j * 64, w.rope_base), True)
            ref, _ = oracle.dense_block(qb, kr[kh], v[0, kh].astype(np.float64), j, 64)
            assert np.abs(got[kh * 4:(kh + 1) * 4, j * 64:(j + 1) * 64] - ref).max() <= 2e-2


@pytest.mark.parametrize("impl", [ATTEND_SIMT, ATTEND_TCGEN05, ATTEND_TCGEN05_ITEM])
def test_attend_isolated_caller_supplied_lists(impl):
    """S4 alone: oracle-rotated Q/K and arbitrary (unsorted, padded, window-overlapping) group lists."""
    w = W.Workload("iso", 1, 1024, 4, 2, 128, "bf16", 1e6, topk_chunks=4, topk_groups=12, n_clusters=4)
    q, k, v = W.generate(w, 11)
    rng = np.random.default_rng(5)
    G, C = 2, 64
    q_rot = np.stack([oracle.round_io(oracle.rope(q[0, h], 0, w.rope_base), True) for h in range(4)])[None]
    k_rot = np.stack([oracle.round_io(oracle.rope(k[0, h], 0, w.rope_base), True) for h in range(2)])[None]
    gidx = -np.ones((1, 2, 16, 12), dtype=np.int32)
    for kh in range(2):
        for j in range(16):
            n_avail = 4 * j
            take = min(n_avail, int(rng.integers(0, 11)))
            if take:
                sel = rng.choice(n_avail, size=take, replace=False)  # may fall inside sink/local windows: set union
                slots = rng.choice(12, size=take, replace=False)     # -1 holes anywhere, unsorted
                gidx[0, kh, j, slots] = sel
    p = hga.params_from_workload(w, attend_impl=impl)
    dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dt)
    out, lse = hga.hga_attend(p, dev(q_rot.astype(np.float32), torch.bfloat16), dev(k_rot.astype(np.float32), torch.bfloat16),
                              dev(v, torch.bfloat16), dev(gidx, torch.int32))
    torch.cuda.synchronize()
    out, lse = out.cpu().numpy(), lse.cpu().numpy()
    for kh in range(2):
        for j in range(16):
            ref, rl, _ = oracle.attend_block(q_rot[0, kh * G:(kh + 1) * G, j * C:(j + 1) * C], k_rot[0, kh],
                                             v[0, kh].astype(np.float64), j, C, 16, 1, 1, gidx[0, kh, j])
            assert np.abs(out[0, kh * G:(kh + 1) * G, j * C:(j + 1) * C] - ref).max() <= 2e-2
            assert np.abs(lse[0, kh * G:(kh + 1) * G, j * C:(j + 1) * C] - rl).max() <= 2e-2


@pytest.mark.parametrize("heads", [(4, 2), (8, 1), (3, 1), (2, 2)], ids=["g2", "g8", "g3", "g1"])
def test_bf16_output_dtype(heads):
    w = W.Workload("bf16out", 1, 512, heads[0], heads[1], 64, "bf16", 1e4, topk_chunks=2, topk_groups=4, n_clusters=4)
    q, k, v = W.generate(w, 2)
    p, buf = parity.run_gpu(w, q, k, v, out_dtype=HGA_F32)
    p2, buf2 = parity.run_gpu(w, q, k, v, out_dtype=HGA_BF16)
    assert buf2.out.dtype == torch.bfloat16
    assert (buf2.out.float() - buf.out).abs().max().item() <= 2.0 ** -6  # one bf16 rounding of |o| < 4


def test_determinism_and_in_place_rope():
    w = W.Workload("det", 1, 1024, 4, 2, 128, "bf16", 1e6, topk_chunks=4, topk_groups=12, n_clusters=4)
    q, k, v = W.generate(w, 4)
    p, a = parity.run_gpu(w, q, k, v)
    _, b = parity.run_gpu(w, q, k, v)
    for name in ("q_rot", "k_rot", "q_pooled", "chunk_sum", "group_sum", "chunk_idx", "group_idx", "out", "lse"):
        assert torch.equal(getattr(a, name), getattr(b, name)), name
    dq, dk, dv = parity.to_device(w, (q, k, v))
    q2, pooled = hga.hga_rope(p, dq, x_rot=dq)  # in place
    assert torch.equal(q2, a.q_rot) and torch.equal(pooled, a.q_pooled)


def test_error_codes_on_device_calls():
    w = W.Workload("err", 1, 512, 4, 2, 64, "bf16", 1e4)
    p = hga.params_from_workload(w)
    x = torch.zeros((1, 4, 512, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(hga.HgaError) as e:
        hga.hga_rope(p, x[:, :, :, :], x_rot=x, pooled=torch.zeros(17, device="cuda")[1:])  # misaligned pooled
    assert e.value.code == 1
    qp = torch.zeros((1, 2, 8, 64), device="cuda")
    gs = torch.zeros((1, 2, 32, 64), device="cuda")
    with pytest.raises(hga.HgaError) as e:
        hga.hga_route(p, qp, qp, gs, workspace=torch.zeros(16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == 3


# ---------------------------------------------------------------------------------------------------------------
# BASELINE.json configs 2..5 at FULL size, in the launch configuration bench.py times; sampled blocks
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n_slices,n_blocks", [("c2", 3, 14), ("c3", 2, 14), ("c4", 2, 14), ("c5", 2, 12)])
def test_full_size_sampled_parity(name, n_slices, n_blocks):
    w = W.get(name)
    q, k, v = W.generate(w, 0)
    p, buf = parity.run_gpu(w, q, k, v)
    rng = np.random.default_rng(1)
    alls = _all_slices(w)
    slices = [alls[i] for i in rng.choice(len(alls), size=n_slices, replace=False)]
    blocks = _sample_blocks(w.n_blocks, n_blocks, 2)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, slices, blocks)
    parity.assert_report(rep, w, len(slices) * len(blocks))
    # property that holds at any size: every list is well formed and counts follow the budget rule
    n_chunks = buf.n_chunks.cpu().numpy()
    j = np.arange(w.n_blocks)
    want = np.minimum(w.topk_chunks, np.maximum(0, j - max(w.n_local, 1) - w.n_sink))
    assert np.array_equal(n_chunks, np.broadcast_to(want, n_chunks.shape))
    assert np.array_equal(buf.n_groups.cpu().numpy(), np.minimum(w.topk_groups, 4 * n_chunks))
    assert torch.isfinite(buf.out).all() and torch.isfinite(buf.lse).all()


# ---------------------------------------------------------------------------------------------------------------
# BASELINE.json configs[4]: planted needle at 10 / 50 / 90 % depth must be in the routed set of the final block
# ---------------------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def c5_inputs():
    w = W.get("c5")
    return w, W.generate(w, 0)


@pytest.mark.parametrize("depth", [0.10, 0.50, 0.90])
def test_c5_needle_group_is_routed(c5_inputs, depth):
    import needle

    w, (q, k, v) = c5_inputs
    kk = k.copy()
    g_star = needle.plant(w, q, kk, depth)
    p, buf = parity.run_gpu(w, q, kk, v)
    last = w.n_blocks - 1
    gidx = buf.group_idx[0, :, last].cpu().numpy()
    cidx = buf.chunk_idx[0, :, last].cpu().numpy()
    op = oracle.params_from_workload(w)
    G = w.gqa
    for kh in range(w.n_kv_heads):
        r = oracle.prefill_slice(op, q[0, kh * G:(kh + 1) * G], kk[0, kh], v[0, kh], blocks=[last], attend=False,
                                 want_k_rot=False)
        assert g_star in r.group_idx[0]                      # the oracle routes it ...
        assert g_star in gidx[kh] and g_star // 4 in cidx[kh]  # ... and so does the GPU
    # and the whole final block (sets, scores, attention output) matches the oracle on the planted input
    rep = parity.check_against_oracle(w, q, kk, v, p, buf, [(0, 0), (0, 3)], [last - 1, last])
    parity.assert_report(rep, w, 4)


# ---------------------------------------------------------------------------------------------------------------
# the persistent S4 kernel across MANY items per CTA: every block of every slice against the oracle.  The grid is one
# CTA per SM (148), so n_items >= 4 x 148 makes every CTA walk at least four items through the phase bits, the
# double-buffered key lists and the pre-issued next-item Q K^T.  items = B * Hkv * n_b * ceil(ceil(G/2)/2).
# ---------------------------------------------------------------------------------------------------------------
MULTI_ITEM = [
    # name,            B, N,    Hq, Hkv, D,   base, Kc, Kg, F, L   -> items (per-CTA items at 148 CTAs)
    ("mi_g8_d128",     2, 8192, 32, 4, 128, 1e6, 6, 24, 1, 1),   # 2*4*128*2 = 2048 (13.8): <128, split 0, pad 0>
    ("mi_g1_d64",      4, 4096, 8, 8, 64, 1e4, 8, 20, 1, 1),     # 4*8*64    = 2048 (13.8): <64, split 1, pad 1>
    ("mi_g3_d64",      2, 8192, 12, 4, 64, 1e4, 8, 20, 1, 1),    # 2*4*128   = 1024 (6.9):  <64, split 0, pad 1>
    ("mi_g2_d128",     2, 8192, 8, 4, 128, 1e6, 6, 24, 1, 2),    # 2*4*128   = 1024 (6.9):  <128, split 1, pad 1>
    ("mi_g4_d64",      2, 8192, 16, 4, 64, 1e4, 6, 24, 2, 1),    # 2*4*128   = 1024 (6.9):  <64, split 0, pad 0>
    # the paper's SmallLM head layout at its own head_dim (hidden 384, 6 query / 2 KV heads -> D 64,
    # G 3) at its speed-test length (12,288 tokens)
    ("smalllm_6_2",    2, 12288, 6, 2, 64, 1e4, 16, 32, 1, 1),   # 2*2*192   = 768  (5.2):  <64, split 0, pad 1>
]


@pytest.mark.parametrize("cfg", MULTI_ITEM, ids=[c[0] for c in MULTI_ITEM])
def test_persistent_kernel_many_items_all_blocks(cfg):
    name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L = cfg
    w = W.Workload(name, B, N, Hq, Hkv, D, "bf16", base, n_sink=F, n_local=L, topk_chunks=Kc, topk_groups=Kg)
    G = Hq // Hkv
    n_items = B * Hkv * w.n_blocks * (((G + 1) // 2 + 1) // 2)
    assert n_items >= 4 * 148
    q, k, v = W.generate(w, 21)
    p, buf = parity.run_gpu(w, q, k, v, attend_impl=ATTEND_TCGEN05)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks * B * Hkv)
    assert torch.isfinite(buf.out).all() and torch.isfinite(buf.lse).all()
    if G == 8 and D == 128:  # the CTA-pair kernel: 1,024 units on 74 pairs = 13.8 units per pair
        p2, buf2 = parity.run_gpu(w, q, k, v, attend_impl=ATTEND_TCGEN05_PAIR)
        rep = parity.check_against_oracle(w, q, k, v, p2, buf2, _all_slices(w), np.arange(w.n_blocks))
        parity.assert_report(rep, w, w.n_blocks * B * Hkv)
        assert torch.isfinite(buf2.out).all() and torch.isfinite(buf2.lse).all()


@pytest.mark.parametrize("name,slc", [("c4", (0, 2)), ("c5", (0, 1))])
def test_full_size_whole_slice_parity(name, slc):
    """BASELINE.json configs[3], [4] at full size in the bench's launch configuration: one whole (batch, kv head)
    slice -- all 512 / 1,024 query blocks x 8 heads, index sets + out + LSE -- against the oracle (c5: 8,192 items
    on 148 CTAs = 55 items per CTA; the slice is 2,048 of them)."""
    w = W.get(name)
    q, k, v = W.generate(w, 0)
    p, buf = parity.run_gpu(w, q, k, v)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [slc], np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks)


# ---------------------------------------------------------------------------------------------------------------
# the CTA-pair S4 kernel (tcgen05.mma.cta_group::2; bf16, D 128, G 8): every block against the oracle.  The last key
# tile of a unit holds np = n_pieces % 8 sixteen-key pieces, split ceil(np/2) / floor(np/2) between the two CTAs:
# the cases cover np = 1..7 and 0 (full), the windows F/L in {0..3}, 32-token groups, and bf16 output.
# ---------------------------------------------------------------------------------------------------------------
PAIR = [
    # name,        B, N,    Hq, Hkv, Kc, Kg, F, L, group   steady-state pieces = 4*(F + max(L,1) + 1) + Kg*group/16
    ("np4",        1, 2048, 16, 2, 6, 24, 1, 1, 16),   # 36 -> 4 full tiles + 4 pieces
    ("np1",        1, 2048, 16, 2, 6, 21, 1, 1, 16),   # 33 -> np 1: the peer CTA holds no key of the last tile
    ("np2",        1, 2048, 8, 1, 6, 22, 1, 1, 16),    # 34
    ("np3",        1, 2048, 8, 1, 6, 23, 1, 1, 16),    # 35
    ("np5",        1, 2048, 8, 1, 8, 25, 1, 1, 16),    # 37
    ("np6_f0l0",   1, 2048, 8, 1, 8, 30, 0, 0, 16),    # 8 + 30 = 38
    ("np7_f2l3",   1, 2048, 8, 1, 8, 31, 2, 3, 16),    # 24 + 31 = 55 -> 6 tiles + 7
    ("np0_gs32",   2, 2048, 8, 1, 6, 10, 1, 1, 32),    # 12 + 20 = 32 -> exactly 4 tiles
    ("tiny_lists", 1, 1024, 16, 2, 1, 2, 1, 1, 16),    # 14 pieces: 2 tiles
]


@pytest.mark.parametrize("out_dtype", [HGA_F32, HGA_BF16], ids=["f32out", "bf16out"])
@pytest.mark.parametrize("cfg", PAIR, ids=[c[0] for c in PAIR])
def test_pair_kernel_full_parity(cfg, out_dtype):
    name, B, N, Hq, Hkv, Kc, Kg, F, L, gs = cfg
    w = W.Workload("pair_" + name, B, N, Hq, Hkv, 128, "bf16", 1e6, group=gs, n_sink=F, n_local=L, topk_chunks=Kc,
                   topk_groups=Kg, n_clusters=8)
    q, k, v = W.generate(w, 17)
    p, buf = parity.run_gpu(w, q, k, v, attend_impl=ATTEND_TCGEN05_PAIR, out_dtype=out_dtype)
    if out_dtype == HGA_F32:
        rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), np.arange(w.n_blocks))
        parity.assert_report(rep, w, w.n_blocks * B * Hkv)
    # the same arithmetic in the same order as the single-CTA kernel (same MMA shapes per row, same softmax code)
    p1, buf1 = parity.run_gpu(w, q, k, v, attend_impl=ATTEND_TCGEN05, out_dtype=out_dtype)
    assert (buf.out.float() - buf1.out.float()).abs().max().item() <= (2e-2 if out_dtype == HGA_F32 else 2.0 ** -6)
    assert (buf.lse - buf1.lse).abs().max().item() <= 2e-2


def test_pair_kernel_rejects_other_shapes():
    w = W.Workload("pair_bad", 1, 512, 4, 2, 128, "bf16", 1e6, topk_chunks=2, topk_groups=4)
    p = hga.params_from_workload(w, attend_impl=ATTEND_TCGEN05_PAIR)
    x = torch.zeros((1, 4, 512, 128), dtype=torch.bfloat16, device="cuda")
    kv = torch.zeros((1, 2, 512, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(hga.HgaError) as e:
        hga.hga_attend(p, x, kv, kv, torch.full((1, 2, 8, 4), -1, dtype=torch.int32, device="cuda"))
    assert e.value.code == 2


# ---------------------------------------------------------------------------------------------------------------
# N3: R4's alternative, max over the block's per-query scores (reading R19) -- the whole path
# with hga_params.route_mode = HGA_ROUTE_MAX against the oracle's route_max switch, every block
# ---------------------------------------------------------------------------------------------------------------
ROUTE_MAX = [
    # name, B, N, Hq, Hkv, D, dtype, base, Kc, Kg, F, L
    ("mx_d64_g2", 1, 2048, 4, 2, 64, "bf16", 1e4, 5, 11, 1, 1),
    ("mx_d128_g8", 1, 2048, 16, 2, 128, "bf16", 1e6, 6, 24, 1, 1),
    ("mx_d128_g3_f2l3", 2, 1536, 6, 2, 128, "bf16", 1e6, 5, 7, 2, 3),
    ("mx_f32", 1, 1024, 4, 1, 64, "f32", 1e4, 4, 8, 1, 1),
    ("mx_kc40", 1, 4096, 2, 2, 64, "bf16", 1e4, 40, 50, 1, 1),   # 160 group candidates: three candidate tiles
]


@pytest.mark.parametrize("cfg", ROUTE_MAX, ids=[c[0] for c in ROUTE_MAX])
def test_route_max_mode_full_parity(cfg):
    name, B, N, Hq, Hkv, D, dt, base, Kc, Kg, F, L = cfg
    w = W.Workload(name, B, N, Hq, Hkv, D, dt, base, n_sink=F, n_local=L, topk_chunks=Kc, topk_groups=Kg, n_clusters=8,
                   dist="iid" if dt == "f32" else "clustered", route_max=True)
    q, k, v = W.generate(w, 31)
    p, buf = parity.run_gpu(w, q, k, v)
    assert p.route_mode == hga.binding.ROUTE_MAX
    rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks * B * Hkv)
    # the rule is not a no-op: the pooled-query rule picks other sets on the same input
    p0, buf0 = parity.run_gpu(dataclasses.replace(w, route_max=False), q, k, v)
    assert not torch.equal(buf.chunk_idx, buf0.chunk_idx)
    # stand-alone call == what hga_prefill did; hga_route refuses the mode
    lib = hga.load_library()
    import ctypes as C
    cp = p.c()
    ci, gi = torch.empty_like(buf.chunk_idx), torch.empty_like(buf.group_idx)
    nc, ng = torch.empty_like(buf.n_chunks), torch.empty_like(buf.n_groups)
    st = torch.cuda.current_stream().cuda_stream
    rc = lib.hga_route_max(C.byref(cp), buf.q_rot.data_ptr(), buf.chunk_sum.data_ptr(), buf.group_sum.data_ptr(),
                           ci.data_ptr(), None, nc.data_ptr(), gi.data_ptr(), None, ng.data_ptr(), buf.workspace.data_ptr(),
                           buf.workspace.numel(), st)
    torch.cuda.synchronize()
    assert rc == 0 and torch.equal(ci, buf.chunk_idx) and torch.equal(gi, buf.group_idx) and torch.equal(ng, buf.n_groups)
    rc = lib.hga_route(C.byref(cp), buf.q_pooled.data_ptr(), buf.chunk_sum.data_ptr(), buf.group_sum.data_ptr(),
                       ci.data_ptr(), None, nc.data_ptr(), gi.data_ptr(), None, ng.data_ptr(), buf.workspace.data_ptr(),
                       buf.workspace.numel(), st)
    assert rc == 1


# The tensor-core prefilter of the max rule (bf16, more than 128 blocks): approximate scores by a bf16 tcgen05 contraction,
# exact fp64 re-scoring of every candidate within the error bound of the K_c-th best.  Against the oracle on sampled
# blocks, and bit-identical to the fp64-only mode (HGA_ROUTE_MAX_FP64) on every block.
ROUTE_MAX_TC = [
    # name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L, dist
    ("mxtc_d64_g2", 1, 16384, 4, 2, 64, 1e4, 5, 11, 1, 1, "clustered"),
    ("mxtc_d128_g8", 1, 16384, 8, 1, 128, 1e6, 12, 48, 1, 1, "clustered"),
    ("mxtc_d128_g3_f2l3", 2, 12288, 6, 2, 128, 1e6, 7, 9, 2, 3, "clustered"),
    ("mxtc_d64_g6_iid", 1, 16384, 6, 1, 64, 1e4, 16, 64, 1, 1, "iid"),
    ("mxtc_d128_g5_kc40", 1, 16384, 5, 1, 128, 1e4, 40, 50, 1, 2, "clustered"),
    ("mxtc_d128_g1", 1, 24576, 2, 2, 128, 1e6, 8, 16, 1, 1, "iid"),
]


def _route_outputs(buf):
    return [buf.chunk_idx, buf.chunk_score, buf.n_chunks, buf.group_idx, buf.group_score, buf.n_groups]


@pytest.mark.parametrize("cfg", ROUTE_MAX_TC, ids=[c[0] for c in ROUTE_MAX_TC])
def test_route_max_tensor_core_prefilter(cfg):
    name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L, dist = cfg
    w = W.Workload(name, B, N, Hq, Hkv, D, "bf16", base, n_sink=F, n_local=L, topk_chunks=Kc, topk_groups=Kg, n_clusters=8,
                   dist=dist, route_max=True)
    q, k, v = W.generate(w, 37)
    p, buf = parity.run_gpu(w, q, k, v)
    assert p.route_mode == hga.binding.ROUTE_MAX
    p2, buf2 = parity.run_gpu(w, q, k, v, route_mode=hga.binding.ROUTE_MAX_FP64)
    for a, b in zip(_route_outputs(buf), _route_outputs(buf2)):
        assert torch.equal(a, b)
    assert torch.equal(buf.out, buf2.out)
    blocks = _sample_blocks(w.n_blocks, 10, 4)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [(B - 1, Hkv - 1)], blocks)
    parity.assert_report(rep, w, len(blocks))


def test_route_max_tensor_core_prefilter_ties_fall_back():
    """Every chunk summary identical (keys periodic in the chunk length, RoPE positions wrapped at the chunk length): all
    candidates tie exactly, the band of possible winners overflows its list and the unit is recomputed by the dense fp64
    path -- the lowest indices win (R8), as in the fp64-only mode and the oracle."""
    w = W.Workload("mxtc_ties", 1, 16384, 4, 2, 64, "bf16", 1e4, topk_chunks=6, topk_groups=12, n_clusters=8, route_max=True,
                   rope_pos_mod=64)
    q, k, v = W.generate(w, 5)
    k = np.ascontiguousarray(np.tile(k[:, :, :64], (1, 1, w.n_blocks, 1)))
    p, buf = parity.run_gpu(w, q, k, v)
    p2, buf2 = parity.run_gpu(w, q, k, v, route_mode=hga.binding.ROUTE_MAX_FP64)
    for a, b in zip(_route_outputs(buf), _route_outputs(buf2)):
        assert torch.equal(a, b)
    ci = buf.chunk_idx[0, 0].cpu().numpy()
    j = w.n_blocks - 1
    assert list(ci[j, :6]) == [1, 2, 3, 4, 5, 6]  # F = 1: candidates start at chunk 1; all tied -> lowest indices
    blocks = _sample_blocks(w.n_blocks, 6, 2)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [(0, 1)], blocks)
    parity.assert_report(rep, w, len(blocks))


def test_route_max_tensor_core_prefilter_many_tied_queries():
    """Blocks whose queries are all zero: every (candidate, query) pair scores exactly 0, so every query row is within the
    error bound of the best and the exact re-scoring takes its list path (more than four rows per candidate); the other
    blocks take the usual path.  Same result as the fp64-only mode and the oracle (all candidates tie -> lowest indices)."""
    w = W.Workload("mxtc_zero_q", 1, 16384, 8, 1, 128, "bf16", 1e6, topk_chunks=6, topk_groups=12, n_clusters=8, route_max=True)
    q, k, v = W.generate(w, 9)
    zero_blocks = [3, 100, 101, 130, 200, 255]   # below and above the 128-candidate limit of the band list
    for j in zero_blocks:
        q[:, :, 64 * j:64 * (j + 1)] = 0.0
    p, buf = parity.run_gpu(w, q, k, v)
    p2, buf2 = parity.run_gpu(w, q, k, v, route_mode=hga.binding.ROUTE_MAX_FP64)
    for a, b in zip(_route_outputs(buf), _route_outputs(buf2)):
        assert torch.equal(a, b)
    ci = buf.chunk_idx[0, 0].cpu().numpy()
    assert list(ci[200, :6]) == [1, 2, 3, 4, 5, 6] and list(ci[100, :6]) == [1, 2, 3, 4, 5, 6]
    blocks = np.array(sorted(set(zero_blocks) | {50, 150, 254}))
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [(0, 0)], blocks)
    parity.assert_report(rep, w, len(blocks))


# ---------------------------------------------------------------------------------------------------------------
# N2: HGA_FLAG_FUSE_Q_ROPE -- q_rot is never written; S0 only pools, S4 reads q_raw and rotates its query tiles in
# shared memory.  Against the oracle on every block, and against the unfused path (same lists bit for bit; outputs equal
# up to the rare one-step bf16 difference of a rotated query, far inside the output tolerance).
# ---------------------------------------------------------------------------------------------------------------
FUSED = [
    # name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L, pos0, pos_mod
    ("fz_d128_g8", 1, 2048, 16, 2, 128, 1e6, 6, 24, 1, 1, 0, 0),
    ("fz_d128_g3_f2l3", 2, 1536, 6, 2, 128, 1e6, 5, 7, 2, 3, 0, 0),       # odd G: a padding head in the last tile
    ("fz_d64_g2", 1, 2048, 4, 2, 64, 1e4, 5, 11, 1, 1, 0, 0),             # split mode: one query tile on both warpgroups
    ("fz_d64_g1", 2, 1024, 4, 4, 64, 1e4, 4, 8, 1, 1, 0, 0),              # split + padding
    ("fz_d64_g6", 1, 2048, 6, 1, 64, 1e4, 6, 12, 1, 2, 0, 0),
    ("fz_d128_g4_pos0", 1, 2048, 8, 2, 128, 1e6, 6, 24, 1, 1, 40000 * 64, 0),
    ("fz_d128_g2_wrap", 1, 4096, 4, 2, 128, 1e4, 6, 24, 1, 1, 0, 2048),   # positions wrap in mid-sequence
    ("fz_smalllm_12k", 1, 12288, 6, 2, 64, 1e4, 16, 32, 1, 1, 0, 0),      # >= 4 items per persistent CTA
]


@pytest.mark.parametrize("cfg", FUSED, ids=[c[0] for c in FUSED])
def test_fused_q_rope_full_parity(cfg):
    name, B, N, Hq, Hkv, D, base, Kc, Kg, F, L, pos0, pos_mod = cfg
    w = W.Workload(name, B, N, Hq, Hkv, D, "bf16", base, n_sink=F, n_local=L, topk_chunks=Kc, topk_groups=Kg, n_clusters=8,
                   pos0=pos0, rope_pos_mod=pos_mod)
    q, k, v = W.generate(w, 41)
    p, buf = parity.run_gpu(w, q, k, v, flags=hga.binding.FLAG_FUSE_Q_ROPE)
    assert buf.q_rot is None
    blocks = np.arange(w.n_blocks) if N <= 4096 else _sample_blocks(w.n_blocks, 24, 4)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, _all_slices(w), blocks)
    parity.assert_report(rep, w, len(blocks) * B * Hkv)
    p0, buf0 = parity.run_gpu(w, q, k, v)
    for a, b in zip(_route_outputs(buf), _route_outputs(buf0)):
        assert torch.equal(a, b)
    assert torch.equal(buf.k_rot, buf0.k_rot) and torch.equal(buf.q_pooled, buf0.q_pooled)
    diff = (buf.out - buf0.out).abs()
    assert float(diff.max()) <= 5e-3, float(diff.max())
    assert float((diff > 0).float().mean()) < 0.2      # most rows see exactly the same rotated queries


def test_fused_q_rope_c5_whole_slice_and_rejections():
    """BASELINE.json configs[4] at full size through the fused path: one whole (batch, kv head) slice against the oracle;
    then the argument checks of the flag."""
    w = W.get("c5")
    q, k, v = W.generate(w, 0)
    p, buf = parity.run_gpu(w, q, k, v, flags=hga.binding.FLAG_FUSE_Q_ROPE)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [(0, 2)], np.arange(w.n_blocks))
    parity.assert_report(rep, w, w.n_blocks)
    assert torch.isfinite(buf.out).all()
    dq, dk, dv = parity.to_device(w, (q, k, v))
    for bad in (dict(route_mode=hga.binding.ROUTE_MAX), dict(attend_impl=ATTEND_SIMT), dict(attend_impl=ATTEND_TCGEN05_ITEM)):
        with pytest.raises(RuntimeError, match="UNSUPPORTED"):
            hga.hga_prefill(p.replace(**bad), dq, dk, dv)
    with pytest.raises(RuntimeError, match="INVALID_ARG"):
        hga.hga_prefill(p.replace(flags=2), dq, dk, dv)


@pytest.mark.parametrize("name", ["c4", "c2"])
def test_route_without_score_outputs_gives_the_same_lists(name):
    """chunk_score / group_score / n_chunks / n_groups are optional outputs (hga.h).  Without group_score, and with K_g keeping
    every group of the kept chunks (c4: K_g = 4 K_c), select_fast_kernel skips the group scoring altogether; the lists must
    not change.  c2 (K_g < 4 K_c) still scores."""
    import ctypes as C
    w = W.get(name)
    q, k, v = W.generate(w, 0)
    p, buf = parity.run_gpu(w, q, k, v)
    lib, cp = hga.load_library(), p.c()
    ci, gi = torch.full_like(buf.chunk_idx, -7), torch.full_like(buf.group_idx, -7)
    rc = lib.hga_route(C.byref(cp), buf.q_pooled.data_ptr(), buf.chunk_sum.data_ptr(), buf.group_sum.data_ptr(), ci.data_ptr(),
                       None, None, gi.data_ptr(), None, None, buf.workspace.data_ptr(), buf.workspace.numel(),
                       torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == 0
    assert torch.equal(ci, buf.chunk_idx) and torch.equal(gi, buf.group_idx)


def test_route_exact_ties_take_the_lowest_indices():
    """Pooled-query rule with every chunk summary identical (keys periodic in the chunk length, RoPE positions wrapped at the
    chunk length): all candidates of a block tie exactly -- also on the fp64 tensor-core instruction, which treats identical
    columns identically -- and the lowest indices win (R8), in the register-resident top-K (16 candidates per lane at 512
    blocks), the shared-memory form (8 per lane at 256 blocks) and the generic kernel (K_c > 32)."""
    for n_blocks, Kc, Kg in ((512, 6, 12), (256, 6, 12), (256, 40, 50)):
        w = W.Workload("ties_mean", 1, 64 * n_blocks, 4, 2, 64, "bf16", 1e4, topk_chunks=Kc, topk_groups=Kg, n_clusters=8,
                       rope_pos_mod=64)
        q, k, v = W.generate(w, 5)
        k = np.ascontiguousarray(np.tile(k[:, :, :64], (1, 1, w.n_blocks, 1)))
        p, buf = parity.run_gpu(w, q, k, v)
        ci = buf.chunk_idx[0, 1].cpu().numpy()
        assert list(ci[n_blocks - 1, :Kc]) == list(range(1, Kc + 1))   # F = 1: candidates start at chunk 1
        assert list(ci[100, :Kc]) == list(range(1, Kc + 1))
        blocks = _sample_blocks(w.n_blocks, 6, 2)
        rep = parity.check_against_oracle(w, q, k, v, p, buf, [(0, 1)], blocks)
        parity.assert_report(rep, w, len(blocks))


def test_route_in_slabs_beyond_1024_blocks():
    """131,072 tokens = 2,048 blocks: S2 + S3 run in two slabs of 1,024 query blocks over one half-size workspace
    (hga_workspace_bytes grows linearly past 1,024 blocks).  Sampled blocks of both slabs, and the blocks around the slab
    boundary, against the oracle; the whole path (outputs included)."""
    w = W.Workload("slab_128k", 1, 131072, 2, 1, 64, "bf16", 1.0e4, topk_chunks=6, topk_groups=12, n_clusters=8)
    q, k, v = W.generate(w, 11)
    p, buf = parity.run_gpu(w, q, k, v)
    assert hga.hga_workspace_bytes(p) == 1024 * 2048 * 4
    blocks = np.array([0, 1, 2, 500, 1022, 1023, 1024, 1025, 1500, 2046, 2047])
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [(0, 0)], blocks)
    parity.assert_report(rep, w, len(blocks))
    nch = buf.n_chunks[0, 0].cpu().numpy()
    assert (nch[8:] == 6).all()          # every later block got its full budget, in both slabs
    assert torch.isfinite(buf.out).all()


def test_route_max_mode_c5_full_size_sampled():
    """The max rule at BASELINE.json configs[4] (64K, Qwen3 head shape): sampled blocks of two slices against the oracle."""
    w = dataclasses.replace(W.get("c5"), route_max=True)
    q, k, v = W.generate(w, 0)
    p, buf = parity.run_gpu(w, q, k, v)
    blocks = _sample_blocks(w.n_blocks, 12, 4)
    rep = parity.check_against_oracle(w, q, k, v, p, buf, [(0, 0), (0, 3)], blocks)
    parity.assert_report(rep, w, 2 * len(blocks))
    assert torch.isfinite(buf.out).all()
