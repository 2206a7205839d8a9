#!/usr/bin/env python
"""bench.py -- HGA routed prefill attention, tokens/s per layer (BASELINE.json `metric`).

A "step" is one pass of the whole hot path (S0 RoPE+pool -> S1 summaries -> S2/S3 route -> S4 gather attention) over
one batch of seeded synthetic input of the chosen workload (default c5: Qwen3-30B-A3B attention shape, 64K prefill).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5] [--impl ours|reference]

Prints ONE JSON line (rank 0).  See the module-level keys in `main()`; the contract is in the task statement:
value = whole-job tokens/s with inputs resident in HBM; e2e = same metric through the host-buffer C-ABI call
(H2D + S0..S4 + D2H inside the timed region); roofline = dominant kernel (S4) against MEASURED_PEAKS.json;
cpu_baseline = the CPU oracle, as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "routed prefill attention tokens/s per layer"
UNIT = "tokens/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return {k: float(d[k]) for k in FALLBACK_PEAKS}, "measured"
    except Exception:
        return dict(FALLBACK_PEAKS), "fallback"


# ---------------------------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.idx = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# algorithmic work per step
# ---------------------------------------------------------------------------------------------------------------
def algorithmic_work(w):
    """Bytes / FLOPs each stage must move / execute for one step of workload `w`."""
    B, N, Hq, Hkv, D = w.batch, w.seq, w.n_q_heads, w.n_kv_heads, w.head_dim
    e = 2 if w.dtype == "bf16" else 4
    n_b, n_g, G = w.n_blocks, w.seq // w.group, w.gqa
    gpc = w.chunk // w.group
    L_eff = max(w.n_local, 1)
    q_elems, kv_elems = B * Hq * N * D, B * Hkv * N * D
    units = B * Hkv * n_b
    s0 = 2 * q_elems * e + units * D * 4
    s1 = 2 * kv_elems * e + units * D * 4 + B * Hkv * n_g * D * 4
    # per block j: attended tokens
    keys_total, cand_pairs, routed_groups = 0, 0, 0
    for j in range(n_b):
        sink = min(w.n_sink, j)
        loc_lo = max(max(0, j - L_eff), sink)
        n_cand = max(0, j - L_eff - w.n_sink)
        n_c = min(w.topk_chunks, n_cand)
        n_gr = min(w.topk_groups, n_c * gpc)
        keys_total += (sink + (j - loc_lo) + 1) * w.chunk + n_gr * w.group
        cand_pairs += n_cand
        routed_groups += n_c * gpc
    keys_total *= B * Hkv
    s2_flops = 2 * B * Hkv * cand_pairs * D
    s2_bytes = 2 * units * D * 4 + B * Hkv * cand_pairs * 4 * 2 + units * (w.topk_chunks + w.topk_groups) * 4 * 2
    s3_bytes = B * Hkv * routed_groups * D * 4
    s4_flops = 4 * D * (w.chunk * G) * keys_total          # QK^T + PV, executed tiles (causal chunk counted whole)
    out_e = 4
    s4_bytes = q_elems * e + q_elems * out_e + 2 * keys_total * D * e   # Q + O + gathered K,V per unit
    return dict(s0_bytes=s0, s1_bytes=s1, s2_bytes=s2_bytes + s3_bytes, s2_flops=s2_flops, s4_flops=s4_flops,
                s4_bytes=s4_bytes, tokens=B * N, launches_per_step=4)


# ---------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample_rate(w, q, k, v, n_blocks_sample: int):
    """Time the oracle on one (b, kv) slice and `n_blocks_sample` evenly spaced query blocks.  Returns
    (tokens_per_s, seconds, description).  A token counts as processed when all H_q heads of it are done, so one
    KV slice of G heads contributes 1/H_kv of a token per row."""
    import numpy as np

    import oracle

    op = oracle.params_from_workload(w)
    blocks = np.unique(np.linspace(0, w.n_blocks - 1, n_blocks_sample).astype(np.int32))
    G = w.gqa
    t0 = time.time()
    oracle.prefill_slice(op, q[0, :G], k[0, 0], v[0, 0], blocks=blocks, attend=True, want_k_rot=False)
    dt = time.time() - t0
    tokens_equiv = len(blocks) * w.chunk / w.n_kv_heads
    desc = (f"oracle (fp64 C, OpenMP) on slice (b=0, kv=0): RoPE+summaries of the whole {w.seq}-token slice, then routing+"
            f"attention for {len(blocks)} of {w.n_blocks} query blocks x {G} heads = {tokens_equiv:.0f} layer-token equivalents")
    return tokens_equiv / dt, dt, desc


def run_reference(args, w):
    import numpy as np

    import hga_workloads as W
    import oracle

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    oracle.build()
    q, k, v = W.generate(w, 0)
    n_s = max(8, args.ref_blocks // max(1, args.steps + args.warmup))  # whole run stays within minutes
    for _ in range(args.warmup):
        oracle_sample_rate(w, q, k, v, max(2, n_s // 4))
    rates, secs = [], []
    desc = ""
    for _ in range(args.steps):
        r, dt, desc = oracle_sample_rate(w, q, k, v, n_s)
        rates.append(r)
        secs.append(dt)
    value = float(np.sum([r * s for r, s in zip(rates, secs)]) / np.sum(secs))
    cores = oracle.max_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, args),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def reduce_max_over_ranks(x: float, dist, device) -> float:
    """Timing rule: a multi-GPU number is the MAX over ranks (device-timed).  `dist` is torch.distributed or None."""
    if dist is None:
        return float(x)
    import torch

    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_tokens_per_s(world: int, tokens_per_rank: int, ms_per_step: float) -> float:
    """Whole-job throughput of `world` independent replicas (weak scaling, no data-path collective)."""
    return world * tokens_per_rank / (ms_per_step * 1e-3)


def rank_seed(rank: int) -> int:
    """Every rank runs its own replica of the workload on its own seeded inputs."""
    return int(rank)


def workload_config(w, args):
    return {"workload": f"{w.name}: B{w.batch} N{w.seq} Hq{w.n_q_heads}/Hkv{w.n_kv_heads} D{w.head_dim} {w.dtype} "
                        f"rope_base {w.rope_base:g}, C{w.chunk} g{w.group} F{w.n_sink} L{w.n_local} Kc{w.topk_chunks} "
                        f"Kg{w.topk_groups}, {w.dist} synthetic Q/K (seed 0)",
            "global_batch": w.batch, "seq_len": w.seq,
            "l2": "per-step working set (Q, Q_rot, K, V, out) exceeds the 126 MB L2; no explicit flush",
            "parallelism": f"replicas x{args.gpus} (no collective: units (batch, kv head) are independent)"}


# ---------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------
def run_ours(args, w):
    import numpy as np
    import torch

    import hga_workloads as W
    import paper_2606_30709_b200 as hga

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hga.load_library()
    peaks, peak_src = load_peaks()

    q, k, v = W.generate(w, rank_seed(rank))  # weak scaling: every rank runs its own replica of the workload
    dt_io = torch.bfloat16 if w.dtype == "bf16" else torch.float32
    hq, hk, hv = (torch.from_numpy(a).to(dt_io).pin_memory() for a in (q, k, v))
    dq, dk, dv = (t.cuda(non_blocking=True) for t in (hq, hk, hv))
    p = hga.params_from_workload(w)
    buf = hga.PrefillBuffers.allocate(p)
    work = algorithmic_work(w)
    torch.cuda.synchronize()

    def step(ev=None):
        """one pass of the hot path through the C ABI; optional per-stage events"""
        if ev is not None:
            ev[0].record()
        hga.hga_rope(p, dq, buf.q_rot, buf.q_pooled)
        if ev is not None:
            ev[1].record()
        hga.hga_build_summaries(p, dk, buf.k_rot, buf.chunk_sum, buf.group_sum)
        if ev is not None:
            ev[2].record()
        lib_route(p, buf)
        if ev is not None:
            ev[3].record()
        hga.hga_attend(p, buf.q_rot, buf.k_rot, dv, buf.group_idx, buf.out, buf.lse)
        if ev is not None:
            ev[4].record()

    import ctypes as C

    lib = hga.load_library()
    cp = p.c()

    def lib_route(p_, b_):
        rc = lib.hga_route(C.byref(cp), b_.q_pooled.data_ptr(), b_.chunk_sum.data_ptr(), b_.group_sum.data_ptr(),
                           b_.chunk_idx.data_ptr(), b_.chunk_score.data_ptr(), b_.n_chunks.data_ptr(),
                           b_.group_idx.data_ptr(), b_.group_score.data_ptr(), b_.n_groups.data_ptr(),
                           b_.workspace.data_ptr(), b_.workspace.numel(), torch.cuda.current_stream().cuda_stream)
        if rc != 0:
            raise hga.HgaError(rc, "hga_route")

    def whole_step():
        """the user's call: S0..S4 through ONE C-ABI call (hga_prefill: S0+S1 fused launch, route, attend)"""
        hga.hga_prefill(p, dq, dk, dv, buf)

    for _ in range(max(args.warmup, 3)):
        whole_step()
    torch.cuda.synchronize()

    K = args.steps
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t_wall0 = time.time()
    start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    start.record()
    for i in range(K):
        whole_step()
    end.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t_wall1 = time.time()
    total_ms = start.elapsed_time(end)
    # ---- per-stage breakdown --------------------------------------------------------------------------------------
    # (a) inside the real call sequence: hga_prefill_profile records CUDA events on the launching stream between the
    #     three launch groups of hga_prefill {S0+S1 fused, S2+S3, S4}; (b) S0 and S1 alone, as separate C-ABI calls.
    Ks = max(K, 10)
    flow_ms = np.zeros(3)
    hga.hga_prefill_profile(p, dq, dk, dv, buf)
    for i in range(Ks):
        flow_ms += np.asarray(hga.hga_prefill_profile(p, dq, dk, dv, buf))
    flow_ms /= Ks
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(Ks)]
    for _ in range(2):
        step()
    torch.cuda.synchronize()
    for i in range(Ks):
        step(evs[i])
    torch.cuda.synchronize()
    clocks = sampler.stop(t_wall0, time.time()) if rank == 0 else None
    stage_ms = np.zeros(4)
    for i in range(Ks):
        for s in range(4):
            stage_ms[s] += evs[i][s].elapsed_time(evs[i][s + 1])
    stage_ms /= Ks
    sep_s4_ms = float(stage_ms[3])
    stage_ms[2], stage_ms[3] = flow_ms[1], flow_ms[2]  # route and S4 as they run inside hga_prefill
    total_ms = reduce_max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / K
    value = job_tokens_per_s(world, work["tokens"], ms_per_step)

    # ---- e2e: host buffers through hga_host_prefill (H2D + S0..S4 + D2H inside the timed region) ---------------
    plan = hga.HostPlan(p)
    out_host = torch.empty((w.batch, w.n_q_heads, w.seq, w.head_dim), dtype=p.torch_out).pin_memory()
    for _ in range(2):
        plan.prefill(hq, hk, hv, out_host)
    Ke = max(3, min(K, 10))
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        plan.prefill(hq, hk, hv, out_host)   # returns after the plan's stream has drained
    e2e_s = (time.perf_counter() - t0) / Ke
    e2e_s = reduce_max_over_ranks(e2e_s, dist, "cuda")
    e2e_value = job_tokens_per_s(world, work["tokens"], e2e_s * 1e3)
    # cheap end-to-end sanity: the host path and the device path agree bit for bit
    same = bool(torch.equal(out_host.cuda(), buf.out))
    plan.close()

    # ---- N1 streaming steps at the end of the context (hga_prefill_window on the filled cache): the last 64-token
    #      chunk as one prefill step, and one single-token decode step.  Idempotent: they rewrite what is there.
    def time_window(t_begin, t_end, reps=20):
        for _ in range(3):
            hga.hga_prefill_window(p, dq, dk, dv, buf, t_begin, t_end)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            hga.hga_prefill_window(p, dq, dk, dv, buf, t_begin, t_end)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    streaming = {"context": w.seq, "chunk_step_ms": time_window(w.seq - w.chunk, w.seq),
                 "decode_step_ms": time_window(w.seq - 1, w.seq),
                 "what": "hga_prefill_window over the last chunk [N-64, N) and over the last token [N-1, N) of the "
                         "filled cache, all batch items and heads; CUDA events, mean of 20 calls (launch-bound)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (S4) and per-stage fractions -------------------------------------------
    s4_s = stage_ms[3] * 1e-3
    tensor_peak = peaks["bf16_tflops_sustained"]  # S4 is timed inside a long step -> sustained figure
    hbm = peaks["hbm_gbs"]
    s4_tflops = work["s4_flops"] / s4_s / 1e12
    s4_t_tensor = work["s4_flops"] / (tensor_peak * 1e12)
    s4_t_hbm = work["s4_bytes"] / (hbm * 1e9)
    bound = "tensor" if s4_t_tensor >= s4_t_hbm else "hbm"
    if bound == "tensor":
        roof = {"bound": "tensor", "achieved": s4_tflops, "peak": tensor_peak, "unit": "TFLOP/s",
                "frac": s4_tflops / tensor_peak}
    else:
        gbs = work["s4_bytes"] / s4_s / 1e9
        roof = {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm}
    roof.update({"traffic": None, "kernel": "attend_tc2_kernel (S4 gather attention)", "peak_source": peak_src,
                 "peak_kind": "bf16_tflops_sustained" if bound == "tensor" else "hbm_gbs",
                 "algorithmic_flops": work["s4_flops"], "algorithmic_bytes": work["s4_bytes"],
                 "kernel_ms": stage_ms[3], "share_of_step": stage_ms[3] / ms_per_step,
                 "timing": "CUDA events recorded by hga_prefill_profile on the launching stream around the S4 launch "
                           "inside the S0..S4 sequence, mean of %d steps" % Ks,
                 "kernel_ms_as_separate_call": sep_s4_ms})
    traffic_file = os.path.join(ROOT, "profiles", f"s4_dram_bytes_{w.name}.json")
    if os.path.exists(traffic_file):
        try:
            roof["traffic"] = json.load(open(traffic_file))["dram_bytes_per_launch"]
        except Exception:
            pass
    stages = {}
    for name, ms, nbytes in (("S0_rope_pool", stage_ms[0], work["s0_bytes"]), ("S1_summaries", stage_ms[1], work["s1_bytes"]),
                             ("S2S3_route", stage_ms[2], work["s2_bytes"])):
        gbs = nbytes / (ms * 1e-3) / 1e9
        stages[name] = {"ms": float(ms), "bound": "hbm", "achieved_GBs": gbs, "frac": gbs / hbm, "bytes": nbytes}
    stages["S0S1_fused"] = {"ms": float(flow_ms[0]), "bound": "hbm", "bytes": work["s0_bytes"] + work["s1_bytes"],
                            "achieved_GBs": (work["s0_bytes"] + work["s1_bytes"]) / (flow_ms[0] * 1e-3) / 1e9,
                            "frac": (work["s0_bytes"] + work["s1_bytes"]) / (flow_ms[0] * 1e-3) / 1e9 / hbm}
    stages["S4_attend"] = {"ms": float(stage_ms[3]), "bound": bound, "achieved_TFLOPs": s4_tflops,
                           "frac_tensor": s4_tflops / tensor_peak,
                           "frac_tensor_burst": s4_tflops / peaks["bf16_tflops"],
                           "achieved_GBs": work["s4_bytes"] / s4_s / 1e9}
    stages["sum_of_flow_stages_ms"] = float(flow_ms.sum())
    roofline_floor_ms = 1e3 * (work["s0_bytes"] / (hbm * 1e9) + work["s1_bytes"] / (hbm * 1e9) +
                               max(s4_t_tensor, s4_t_hbm))

    # ---- cpu baseline (oracle, bounded sample) -------------------------------------------------------------------
    cpu = None
    if not args.no_cpu_baseline:
        import oracle

        oracle.build()
        rate, secs, desc = oracle_sample_rate(w, q, k, v, args.ref_blocks)
        cpu = {"value": rate, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle", "sample": desc,
               "seconds": secs}

    h2d = plan.h2d_bytes
    d2h = plan.d2h_bytes
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic",
        "config": workload_config(w, args),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_s * 1e3, "matches_device_path": same},
        "gpu_launches": work["launches_per_step"] * K,
        "roofline": roof,
        "cpu_baseline": cpu,
        "stages": stages,
        "streaming": streaming,
        "roofline_floor_ms": roofline_floor_ms,
        "frac_of_roofline_floor": roofline_floor_ms / ms_per_step,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5", help="c1..c5 (BASELINE.json configs[0..4]); default c5 = 64K Qwen3 shape")
    ap.add_argument("--ref-blocks", type=int, default=2048,
                    help="query blocks in the oracle's bounded sample (cpu_baseline: one sample of min(this, n_blocks); "
                         "--impl reference: spread over the steps)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    import hga_workloads as W

    w = W.get(args.workload)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
