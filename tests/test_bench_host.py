"""Host-side logic of bench.py on CPU (-m "not gpu"): the N>1 path over `gloo` with world_size 2, the reference arm's
JSON contract, and the algorithmic-work accounting the roofline uses."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import hga_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank times its own replica; the job's step time is the max over ranks
        my_ms = 10.0 + 5.0 * rank
        ms = bench.reduce_max_over_ranks(my_ms, dist, "cpu")
        # replicas run on distinct seeded inputs (no data-path collective)
        w = W.get("c1").replace(seq=128)
        q, _, _ = W.generate(w, bench.rank_seed(rank))
        digest = torch.tensor([float(np.abs(q).sum())], dtype=torch.float64)
        both = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(both, digest)
        ret[rank] = (ms, bench.job_tokens_per_s(world, w.batch * w.seq, ms), [float(t.item()) for t in both])
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_max_over_ranks_and_weak_scaling_value():
    world, port = 2, _free_port()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    assert set(ret.keys()) == {0, 1}
    for r in range(world):
        ms, value, digests = ret[r]
        assert ms == 15.0                                   # max over ranks, same on every rank
        assert value == pytest.approx(2 * 128 / 15e-3)      # whole-job tokens/s = world * per-rank tokens / max time
        assert digests[0] != digests[1]                     # different seeds per rank
    assert ret[0][2] == ret[1][2]


def test_reference_arm_under_torchrun_rank0_prints_others_exit_0():
    """`bench.py --impl reference` launched like the driver launches N>1: rank 0 alone prints ONE JSON line."""
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--workload", "c1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["unit"] == bench.UNIT
    assert d["value"] > 0 and d["higher_is_better"] is True and d["n_gpus"] == 2
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("c1")


def test_algorithmic_work_matches_survey_figures():
    """steady-state attended tokens and the per-stage byte/FLOP figures at c4 / c5."""
    w5, w4 = W.get("c5"), W.get("c4")
    a5, a4 = bench.algorithmic_work(w5), bench.algorithmic_work(w4)
    assert a5["tokens"] == 65536 and a4["tokens"] == 32768
    assert a5["s0_bytes"] == pytest.approx(1076e6, rel=2e-3) and a5["s1_bytes"] == pytest.approx(145e6, rel=5e-3)
    # S4 FLOPs: 4*D*(64*G)*T per (block, kv head), T -> 960 (c5) / 1216 (c4) in steady state
    assert a5["s4_flops"] == pytest.approx(1.024e12, rel=0.01)
    assert a4["s4_flops"] == pytest.approx(0.641e12, rel=0.01)
    last = 4 * 128 * (64 * 8) * (48 * 16 + 3 * 64)
    assert last == 4 * 128 * 512 * 960
    # compulsory S4 DRAM bytes (c5 1208 MB with bf16 output; fp32 output adds another |Q|): Q + O + K + V
    assert a5["s4_bytes"] == 537e6 * 0 + (65536 * 32 * 128) * (2 + 4) + 2 * (65536 * 4 * 128) * 2
    assert a5["s4_bytes_gathered"] > 2 * a5["s4_bytes"]  # the per-block re-gathers are L2 traffic, not DRAM
    # useful FLOPs exclude the masked half of the causal chunk: 63/128 of one 64-key chunk per block
    assert a5["s4_flops_useful"] == a5["s4_flops"] - 4 * 128 * 32 * 1024 * (64 * 63 // 2)


def test_peaks_loader_falls_back_to_the_profiling_guide_numbers(tmp_path, monkeypatch):
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    peaks, src = bench.load_peaks()
    assert src == "fallback" and peaks["hbm_gbs"] == 6650.0 and peaks["bf16_tflops"] == 1590.0
