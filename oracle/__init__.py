"""CPU oracle for HGA prefill -- TEST INFRASTRUCTURE ONLY (see oracle/hga_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It never imports paper_2606_30709_b200 and shares no code with it.
"""
from .hga_oracle import (  # noqa: F401
    OracleParams,
    SliceResult,
    StepResult,
    attend_block,
    build,
    default_n_hi,
    dense_block,
    key_set,
    max_threads,
    n_hi_rule,
    params_from_workload,
    pool_queries,
    prefill,
    prefill_slice,
    rope,
    round_io,
    route_chunks,
    route_chunks_max,
    route_groups_max,
    route_groups,
    step,
    summaries,
)
