"""Host-side checks of the C-ABI library (no GPU, no compute calls): libhga.so loads, exports every symbol that
include/hga.h declares, and its host-arithmetic entry points (validation, sizes, pair-count rules) behave as the
header says.
"""
import ctypes as C
import os
import re

import pytest

import hga_workloads as W
import paper_2606_30709_b200 as hga

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hga.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)  # drop comments
    return sorted(set(re.findall(r"HGA_API\s+[^;(]*?\b(hga_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    names = declared_symbols()
    # the boundary SURVEY.md 8(b) lists, plus what this build added around it
    for must in ("hga_status_string", "hga_workspace_bytes", "hga_rope", "hga_build_summaries", "hga_route",
                 "hga_attend", "hga_prefill", "hga_prefill_window", "hga_host_prefill", "hga_n_hi_rule"):
        assert must in names
    lib = C.CDLL(hga.lib_path())
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing


def test_version_and_status_strings():
    lib = hga.load_library()
    assert hga.hga_version() >= 100
    lib.hga_status_string.restype = C.c_char_p
    seen = {lib.hga_status_string(i) for i in range(5)}
    assert len(seen) == 5 and all(s for s in seen)  # five distinct, non-empty messages
    assert lib.hga_status_string(12345)  # unknown codes still give a string


def test_validate_accepts_the_baseline_configs_and_rejects_bad_shapes():
    for name in ("c1", "c2", "c3", "c4", "c5"):
        assert hga.hga_validate(hga.params_from_workload(W.get(name))) == 0
    ok = hga.params_from_workload(W.get("c2"))
    bad = [ok.replace(seq=ok.seq + 1),            # only closed chunks
           ok.replace(n_q_heads=7),               # GQA: H_q % H_kv
           ok.replace(group=24),                  # group must divide the chunk
           ok.replace(topk_chunks=-1), ok.replace(n_sink=-1),
           ok.replace(n_hi_chunk=ok.head_dim),    # more pairs than D/2
           ok.replace(rope_base=0.0), ok.replace(softmax_scale=-1.0), ok.replace(pos0=-5),
           ok.replace(io_dtype=7), ok.replace(head_dim=0)]
    for p in bad:
        assert hga.hga_validate(p) != 0, p
    assert hga.hga_validate(ok.replace(head_dim=96)) == 2  # HGA_ERR_UNSUPPORTED: the kernels cover D in {64, 128}


def test_position_wrap_argument_checks():
    """rope_pos_mod and pos0 must be multiples of the chunk so that no span straddles a wrap."""
    ok = hga.params_from_workload(W.get("c2"))
    assert hga.hga_validate(ok.replace(rope_pos_mod=65536)) == 0
    assert hga.hga_validate(ok.replace(rope_pos_mod=128, pos0=64 * 5)) == 0
    for p in (ok.replace(rope_pos_mod=-1), ok.replace(rope_pos_mod=100), ok.replace(rope_pos_mod=128, pos0=32)):
        assert hga.hga_validate(p) == 1  # HGA_ERR_INVALID_ARG


def test_workspace_and_host_byte_counts():
    for name in ("c1", "c4", "c5"):
        w = W.get(name)
        p = hga.params_from_workload(w)
        n_b = w.seq // 64
        assert hga.hga_workspace_bytes(p) >= w.batch * w.n_kv_heads * n_b * n_b * 4  # the chunk-score matrix
    # beyond 1024 blocks the route stage runs in slabs of 1024 query blocks: the workspace grows linearly, not quadratically
    big = hga.params_from_workload(W.get("c5").replace(seq=16 * 65536))
    assert hga.hga_workspace_bytes(big) == 1 * 4 * 1024 * (16 * 1024) * 4
    for name in ("c5",):
        w = W.get(name)
        p = hga.params_from_workload(w)
        e = 2 if w.dtype == "bf16" else 4
        h2d, d2h = C.c_size_t(0), C.c_size_t(0)
        assert hga.load_library().hga_host_bytes(C.byref(p.c()), 0, 0, C.byref(h2d), C.byref(d2h)) == 0
        assert h2d.value == w.batch * w.seq * w.head_dim * e * (w.n_q_heads + 2 * w.n_kv_heads)
        assert d2h.value == w.batch * w.seq * w.head_dim * w.n_q_heads * 4  # fp32 out
    n = C.c_size_t(0)
    assert hga.load_library().hga_workspace_bytes(None, C.byref(n)) != 0


def test_n_hi_rules_host_arithmetic():
    # counts for the two model shapes (chunk, group) under the three thresholds: SURVEY.md 8(c) R1
    assert [hga.hga_n_hi_rule(64, 1e4, s, r) for r in range(3) for s in (64, 16)] == [9, 4, 11, 6, 15, 10]
    assert [hga.hga_n_hi_rule(128, 1e6, s, r) for r in range(3) for s in (64, 16)] == [11, 5, 14, 8, 20, 13]
    assert hga.hga_n_hi_rule(64, 1e4, 64, 0) == hga.hga_default_n_hi(64, 1e4, 64)
    assert hga.hga_n_hi_rule(64, 1e4, 64, 3) == -1 and hga.hga_n_hi_rule(63, 1e4, 64, 0) == -1


def test_compute_calls_fail_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    w = W.get("c1")
    p = hga.params_from_workload(w)
    with pytest.raises(Exception):
        hga.PrefillBuffers.allocate(p, "cuda")
