"""Seeded synthetic workloads for HGA prefill (inputs only).

This module is the single source of input bits for BOTH the CPU oracle (``oracle/``) and the
CUDA path (``paper_2606_30709_b200/``).  It holds none of the method's arithmetic: no RoPE, no
summaries, no routing, no attention -- only random-number draws, the planted cluster structure
BASELINE.json's configs describe, and the fp32 -> bf16 storage rounding.

The five configs are BASELINE.json ``configs[0..4]`` (named c1..c5 as in SURVEY.md 8(d)).  They stand
in for the paper's FineWeb / needle / Qwen3 workloads, which are not
available offline; shapes and routing parameters are taken from those passages.
"""
from .workloads import (  # noqa: F401
    CONFIGS,
    Workload,
    bf16_round,
    generate,
    get,
)
