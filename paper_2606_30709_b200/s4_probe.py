"""Developer probe for the S4 kernels: times hga_attend ALONE (CUDA events, median / min of N calls) on a BASELINE
workload after one hga_prefill has produced the routed lists, and -- for a library built with -DHGA_S4_TRACE --
dumps the clock64 timeline of two work items of CTA 0 (softmax warpgroups and the MMA issuer).

    python -m paper_2606_30709_b200.s4_probe --workload c5 [--impl 2] [--lib path/to/libhga_variant.so] [--trace]
    python -m paper_2606_30709_b200.s4_probe --workload c5 --route-max     (N3 max rule: both route modes timed and compared;
                                                                            per-phase cycles with a -DHGA_ROUTE_TRACE build)

Kernel experiments are compile-time knobs (HGA_S4_DIAG bit mask: 1 no softmax arithmetic, 2 no MMAs, 4 no MUFU,
8 no K/V TMA; HGA_S4_EMU_PERIOD / _COUNT; HGA_S4_TRACE), set through HGA_NVCC_EXTRA:

    HGA_NVCC_EXTRA=-DHGA_S4_DIAG=9 python -m paper_2606_30709_b200.build --force
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import os


def route_max_probe(B, w, dq, dk, dv, reps):
    import torch

    lib = B.load_library()
    res = {}
    for mode in (B.ROUTE_MAX, B.ROUTE_MAX_FP64):
        p = B.params_from_workload(w).replace(route_mode=mode)
        buf = B.hga_prefill(p, dq, dk, dv)
        cp, st = p.c(), torch.cuda.current_stream().cuda_stream
        nbytes = buf.workspace.numel() * buf.workspace.element_size()

        def call():
            rc = lib.hga_route_max(C.byref(cp), buf.q_rot.data_ptr(), buf.chunk_sum.data_ptr(), buf.group_sum.data_ptr(),
                                   buf.chunk_idx.data_ptr(), buf.chunk_score.data_ptr(), buf.n_chunks.data_ptr(),
                                   buf.group_idx.data_ptr(), buf.group_score.data_ptr(), buf.n_groups.data_ptr(),
                                   buf.workspace.data_ptr(), nbytes, st)
            assert rc == 0, rc

        call()
        torch.cuda.synchronize()
        n = reps if mode == B.ROUTE_MAX else max(2, reps // 10)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            call()
        e1.record()
        torch.cuda.synchronize()
        res[mode] = (e0.elapsed_time(e1) / n, [t.clone() for t in (buf.chunk_idx, buf.chunk_score, buf.n_chunks, buf.group_idx,
                                                                   buf.group_score, buf.n_groups, buf.out)])
    same = all(torch.equal(a, b) for a, b in zip(res[B.ROUTE_MAX][1], res[B.ROUTE_MAX_FP64][1]))
    print(json.dumps({"workload": w.name, "route_max_ms": res[B.ROUTE_MAX][0], "route_max_fp64_ms": res[B.ROUTE_MAX_FP64][0],
                      "bit_identical": same, "workspace_MB": nbytes / 1e6}))
    if hasattr(lib, "hga_debug_route_trace"):
        arr = (C.c_ulonglong * 32)()
        lib.hga_debug_route_trace(arr)
        n = max(int(arr[15]), 1)
        names = ["setup + Q TMA issue", "stage candidate rows", "Q wait + q_max", "MMA", "row max", "sweep", "fp64 re-score", "dealloc"]
        print("score_max_listed_kernel, CTAs", n, "| mean cycles per CTA:", {k: round(arr[i] / n) for i, k in enumerate(names)})


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lib", default=None, help="alternative libhga.so (a build with experiment knobs)")
    ap.add_argument("--workload", default="c5")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--impl", type=int, default=0, help="hga_attend_impl (0 auto, 2 persistent, 4 CTA pair)")
    ap.add_argument("--trace", action="store_true", help="print the HGA_S4_TRACE timeline (needs a trace build)")
    ap.add_argument("--out-bf16", action="store_true", help="bf16 output rows instead of fp32")
    ap.add_argument("--route-max", action="store_true", help="time hga_route_max under HGA_ROUTE_MAX and HGA_ROUTE_MAX_FP64")
    args = ap.parse_args()
    import numpy as np
    import torch

    from . import binding as B
    if args.lib:
        B._LIB_PATH = os.path.abspath(args.lib)
    import hga_workloads as W

    w = W.get(args.workload)
    q, k, v = W.generate(w, 0)
    dt = torch.bfloat16 if w.dtype == "bf16" else torch.float32
    dq, dk, dv = (torch.from_numpy(a).to(dt).cuda() for a in (q, k, v))
    if args.route_max:
        return route_max_probe(B, w, dq, dk, dv, args.reps)
    p = B.params_from_workload(w, attend_impl=args.impl, out_dtype=B.HGA_BF16 if args.out_bf16 else B.HGA_F32)
    buf = B.PrefillBuffers.allocate(p)
    for _ in range(3):
        B.hga_prefill(p, dq, dk, dv, buf)
    torch.cuda.synchronize()
    ms = []
    for _ in range(args.reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        B.hga_attend(p, buf.q_rot, buf.k_rot, dv, buf.group_idx, buf.out, buf.lse)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    flow = np.mean([B.hga_prefill_profile(p, dq, dk, dv, buf) for _ in range(10)], axis=0)
    print(json.dumps({"workload": w.name, "impl": args.impl, "s4_ms_median": float(np.median(ms)), "s4_ms_min": float(np.min(ms)),
                      "prefill_stage_ms": [float(x) for x in flow]}))
    if args.trace:
        out = (C.c_longlong * 4096)()
        rc = B.load_library().hga_debug_trace(out)
        a = np.array(out[:], dtype=np.int64)
        t0 = a[a > 0].min()
        sm, mm = a[:256].reshape(2, 8, 2, 8), a[1024:1280].reshape(2, 8, 2, 8)
        print("rc", rc, "| item tile t | softmax: S ready, ld done, max done, P(0..63) handed, P(64..127) handed | "
              "MMA issuer: P_a seen, PV_a issued, P_b seen, PV_b + next QK issued   (cycles)")
        for kk in range(2):
            for i in range(8):
                for t in range(2):
                    print(kk, i, t, "|", " ".join("%6d" % x for x in (sm[kk, i, t, :5] - t0)), "|",
                          " ".join("%6d" % x for x in (mm[kk, i, t, :4] - t0)))


if __name__ == "__main__":
    main()
