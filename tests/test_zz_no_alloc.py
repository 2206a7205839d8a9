"""hga_route_static: S2 + S3 through the library's static device scratch (no workspace argument, no allocation).

Collected last on purpose (the suite runs with `pytest -x`): a failure here must not hide the parity tests.  The test
passes alone in a fresh process and after the other tests -- it depends on nothing they leave behind, and the scratch array
needs no particular initial contents.
"""
from __future__ import annotations

import pytest
import torch

import hga_workloads as W
import paper_2606_30709_b200 as hga
import parity

pytestmark = pytest.mark.gpu

FIELDS = ("chunk_idx", "chunk_score", "n_chunks", "group_idx", "group_score", "n_groups")


def _inputs(w, seed):
    """q_pooled / chunk_sum / group_sum of a workload, produced by the existing path (hga_prefill)."""
    q, k, v = W.generate(w, seed)
    p, buf = parity.run_gpu(w, q, k, v)
    return p, buf


def _assert_same(a, b, p):
    for f in FIELDS:
        x, y = getattr(a, f), getattr(b, f)
        # integer lists bit-exact; scores are the same kernels on the same inputs -> bit-exact as well, which is inside the
        # 1e-6-relative score tolerance of the parity tests
        assert torch.equal(x, y), f


def test_route_static_matches_hga_route_on_two_calls_in_a_row():
    # call 1: a larger problem (128 blocks, routing budgets that make S3 a real selection); call 2: a smaller one with other
    # data and budgets, run right after it on the same stream -- the array still holds call 1's scores where call 2 does not
    # write, and the result must not care
    w1 = W.Workload("na_d128_g8", 1, 8192, 16, 2, 128, "bf16", 1.0e6, topk_chunks=6, topk_groups=11, n_clusters=8)
    w2 = W.Workload("na_d64_g2", 1, 4096, 4, 2, 64, "bf16", 1.0e4, n_sink=2, n_local=3, topk_chunks=40, topk_groups=50,
                    n_clusters=8)
    p1, b1 = _inputs(w1, 3)
    p2, b2 = _inputs(w2, 4)
    ref1 = hga.hga_route(p1, b1.q_pooled, b1.chunk_sum, b1.group_sum)
    ref2 = hga.hga_route(p2, b2.q_pooled, b2.chunk_sum, b2.group_sum)
    torch.cuda.synchronize()
    got1 = hga.hga_route_static(p1, b1.q_pooled, b1.chunk_sum, b1.group_sum)
    got2 = hga.hga_route_static(p2, b2.q_pooled, b2.chunk_sum, b2.group_sum)
    torch.cuda.synchronize()
    _assert_same(got1, ref1, p1)
    _assert_same(got2, ref2, p2)
    # and what hga_prefill itself selected (the path every parity test checks against the oracle)
    assert torch.equal(got1.group_idx, b1.group_idx) and torch.equal(got2.group_idx, b2.group_idx)
    # the same call again into the same output tensors: identical, and the device's free memory does not move (no cudaMalloc
    # inside the call; the outputs are reused, so the Python side allocates nothing either)
    for attempt in range(3):  # mem_get_info is device-wide: tolerate an unrelated change once or twice, never a steady one
        free0 = torch.cuda.mem_get_info()[0]
        again = hga.hga_route_static(p1, b1.q_pooled, b1.chunk_sum, b1.group_sum, out=got1)
        again = hga.hga_route_static(p2, b2.q_pooled, b2.chunk_sum, b2.group_sum, out=got2)
        torch.cuda.synchronize()
        if torch.cuda.mem_get_info()[0] == free0:
            break
    else:
        raise AssertionError("device free memory moved across hga_route_static calls three times in a row")
    _assert_same(again, ref2, p2)
    _assert_same(got1, ref1, p1)


def test_route_static_at_its_size_limit_and_beyond():
    # BASELINE.json configs[4] (64K, 4 KV heads) needs exactly HGA_ROUTE_STATIC_MAX_BYTES
    w = W.get("c5")
    p, buf = _inputs(w, 0)
    assert p.batch * p.n_kv_heads * p.n_blocks ** 2 * 4 == hga.binding.ROUTE_STATIC_MAX_BYTES
    ref = hga.hga_route(p, buf.q_pooled, buf.chunk_sum, buf.group_sum)
    got = hga.hga_route_static(p, buf.q_pooled, buf.chunk_sum, buf.group_sum)
    torch.cuda.synchronize()
    _assert_same(got, ref, p)
    assert torch.equal(got.chunk_idx, buf.chunk_idx) and torch.equal(got.group_idx, buf.group_idx)
    # one block more per slice does not fit: refused with HGA_ERR_WORKSPACE before anything is launched
    big = p.replace(seq=p.seq + 64)
    units = (big.batch, big.n_kv_heads, big.n_blocks)
    qp = torch.zeros(units + (big.head_dim,), dtype=torch.float32, device="cuda")
    gs = torch.zeros((big.batch, big.n_kv_heads, big.seq // big.group, big.head_dim), dtype=torch.float32, device="cuda")
    with pytest.raises(RuntimeError, match="WORKSPACE"):
        hga.hga_route_static(big, qp, qp, gs)
    # the max-over-queries rule has its own entry point
    with pytest.raises(RuntimeError, match="INVALID_ARG"):
        hga.hga_route_static(p.replace(route_mode=hga.binding.ROUTE_MAX), buf.q_pooled, buf.chunk_sum, buf.group_sum)
    # still usable after the refusals
    got2 = hga.hga_route_static(p, buf.q_pooled, buf.chunk_sum, buf.group_sum, out=got)
    torch.cuda.synchronize()
    _assert_same(got2, ref, p)
