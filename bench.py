#!/usr/bin/env python
"""bench.py — AMP-PCG time-to-tolerance / iterations per second on one B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--impl ours|reference]

One "step" = one whole solve (every row of SURVEY.md §8(a): set-up, then per iteration the fused
z/(r,z), p, SpMV/(p,Ap), x/r/||r|| kernels with device-side precision switching) of the seeded
synthetic system `--workload` (default c2 = BASELINE.json configs[1], 3-D Poisson 128^3, tol 1e-10)
from x0 = 0, with A resident in HBM.  `value` = PCG iterations per second over all ranks
(N > 1: independent replicas, one per GPU, no data-path collective: "weak" scaling).
Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "amp_pcg_iterations_per_s"
UNIT = "iterations/s"
SMI_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the SpMV kernel from the committed ncu --set full
# captures (profiles/r01c_*.md name the commands); None where no capture exists for that workload
NCU_TRAFFIC = {
    ("c2", "fp32mat_fp16vec"): 64.82e6 + 2.17e6,   # profiles/r01c_c2_ncu_full.csv, k_spmv in phase (FP16, FP32)
    ("c4", "fp32mat_fp16vec"): 907.34e6 + 28.23e6,  # profiles/r01c_c4_ncu_full.csv
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--size", type=int, default=None, help="override grid edge / rows (debug only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--policy", default="amp_fp64_delay", choices=["amp_fp64_delay", "amp_fp16_linear"])
    ap.add_argument("--loop", default="auto", choices=["auto", "stream", "graph", "persistent"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profile-iters", type=int, default=0,
                    help="profiling aid for ncu: run ONE solve of this many iterations with plain stream launches "
                         "(u_r forced to FP32 from k=ell so the low-precision kernels appear) and exit; prints no bench line")
    ap.add_argument("--profile-policy", default="amp_fp16_linear", choices=["pcg_fp64", "amp_fp16_linear", "amp_fp64_delay", "amp_fp16_linear_lagged"])
    ap.add_argument("--ref-iters", type=int, default=100, help="--impl reference: iterations per step (bounded sample)")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={SMI_QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *exc):
        self.result = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        for line in out.splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if sm:
            self.result = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                           "samples": len(sm)}


def reduce_over_ranks(dist, vmax, vsum, device):
    """Whole-job aggregation of one timed region: element-wise MAX over ranks of `vmax` (device times: the job is as
    slow as its slowest rank) and SUM over ranks of `vsum` (work done: iterations, launches).  dist = None: one rank."""
    if dist is None:
        return [float(v) for v in vmax], [float(v) for v in vsum]
    import torch

    tm = torch.tensor([float(v) for v in vmax], dtype=torch.float64, device=device)
    ts = torch.tensor([float(v) for v in vsum], dtype=torch.float64, device=device)
    dist.all_reduce(tm, op=dist.ReduceOp.MAX)
    dist.all_reduce(ts, op=dist.ReduceOp.SUM)
    return tm.tolist(), ts.tolist()


def policy_kwargs(name: str):
    return {"amp_fp64_delay": dict(amp=1, u0=0, eta_rule=0), "amp_fp16_linear": dict(amp=1, u0=2, eta_rule=1)}[name]


# --------------------------------------------------------------------------------------------
def run_reference(args, rank: int, world: int):
    """--impl reference: the CPU oracle as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle as O
    from workloads import make_config

    s = make_config(args.workload, args.size)
    kw = policy_kwargs(args.policy)
    pol = O.make_policy(**kw)
    cap = min(args.ref_iters, s.maxit)
    times, its = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, cap, pol)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt); its += r.iters
    total = sum(times)
    val = its / total
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / max(len(times), 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 (f32/f16 storage emulated by rounding)", "data": "synthetic",
        "config": {"workload": s.name, "n": s.n, "nnz": s.nnz, "tol": s.tol, "policy": args.policy,
                   "sample": f"first {cap} iterations of the solve per step"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                         "sample": f"{args.steps} x first {cap} iterations of AMP-PCG on {s.name}"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, rank: int, local_rank: int, world: int):
    import numpy as np
    import torch

    import paper_2505_04155_b200 as A
    from workloads import make_config

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_

        dist = dist_
        dist.init_process_group("nccl", device_id=dev)

    s = make_config(args.workload, args.size)
    rp, ci, va, b = (torch.from_numpy(a).to(dev) for a in (s.rowptr, s.colidx, s.vals, s.b))
    t0 = time.perf_counter()
    h = A.AmpPcg(rp, ci, va, A.PRECOND_JACOBI)
    torch.cuda.synchronize()
    create_s = time.perf_counter() - t0
    if args.profile_iters > 0:
        kwp = {"pcg_fp64": dict(amp=0), "amp_fp16_linear": dict(u0=A.FP16, eta_rule=A.ETA_LINEAR, eps32=1e-30),
               "amp_fp16_linear_lagged": dict(u0=A.FP16, eta_rule=A.ETA_LINEAR, eps32=1e-30, scale_mode=A.SCALE_LAGGED),
               "amp_fp64_delay": dict()}[args.profile_policy]
        lp = A.LOOP_STREAM if args.loop == "auto" else {"stream": A.LOOP_STREAM, "graph": A.LOOP_GRAPH, "persistent": A.LOOP_PERSISTENT}[args.loop]
        xp = torch.zeros(s.n, dtype=torch.float64, device=dev)
        stp = h.solve(b, xp, s.tol, args.profile_iters, A.Policy.default(x0_zero=1, loop_mode=lp, **kwp))
        print("profile run:", stp.asdict(), file=sys.stderr)
        h.close()
        return
    loop = {"auto": A.LOOP_AUTO, "stream": A.LOOP_STREAM, "graph": A.LOOP_GRAPH, "persistent": A.LOOP_PERSISTENT}[args.loop]
    kw = policy_kwargs(args.policy)
    pol = A.Policy.default(x0_zero=1, loop_mode=loop, **kw)
    pol_fp64 = A.Policy.default(x0_zero=1, loop_mode=loop, amp=0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # 256 MiB > 126 MB L2
    x = torch.zeros(s.n, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_solves(policy, count, host=False, bh=None, xh=None):
        """count solves, each bracketed by CUDA events on the solve stream, L2 flushed before each."""
        ms, its, launches, last = [], 0, 0, None
        for _ in range(count):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            if host:
                st = h.solve_host(bh, xh, s.tol, s.maxit, policy)
            else:
                st = h.solve(b, x, s.tol, s.maxit, policy)
            e1.record(stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1)); its += st.iters; launches += h.last_launch_count(); last = st
        return ms, its, launches, last

    # ---- warm-up, then EXACTLY K timed steps between barriers ----
    timed_solves(pol, args.warmup)
    barrier()
    with ClockSampler(local_rank) as clk:
        ms, its, launches, st = timed_solves(pol, args.steps)
    barrier()
    total_ms = sum(ms)
    (total_ms_max,), (its_all, launches_all) = reduce_over_ranks(dist, [total_ms], [its, launches], dev)
    launches_all = int(launches_all)
    value = its_all / (total_ms_max * 1e-3)

    # ---- end-to-end through the host-buffer entry point (H2D of b, solve, D2H of x inside) ----
    bh = torch.from_numpy(s.b).pin_memory()
    xh = torch.zeros(s.n, dtype=torch.float64).pin_memory()
    timed_solves(pol, 1, host=True, bh=bh, xh=xh)
    barrier()
    ms_e, its_e, _, _ = timed_solves(pol, args.steps, host=True, bh=bh, xh=xh)
    barrier()
    (tot_e,), (its_e,) = reduce_over_ranks(dist, [sum(ms_e)], [its_e], dev)
    e2e_value = its_e / (tot_e * 1e-3)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- this library's own FP64 PCG on the same system (north_star: AMP must beat it) ----
    timed_solves(pol_fp64, 1)
    ms64, its64, _, st64 = timed_solves(pol_fp64, max(2, min(args.steps, 3)))
    t_amp = statistics.median(ms) * 1e-3
    t_fp64 = statistics.median(ms64) * 1e-3
    # ---- the lagged variant (AMP_SCALE_LAGGED, reading R17): same policy, three kernels per iteration ----
    lagged = None
    if True:
        pol_lag = A.Policy.default(x0_zero=1, loop_mode=loop, scale_mode=A.SCALE_LAGGED, **kw)
        timed_solves(pol_lag, 1)
        ms_l, _, _, st_l = timed_solves(pol_lag, max(2, min(args.steps, 3)))
        t_lag = statistics.median(ms_l) * 1e-3
        lagged = {"time_to_tol_s": t_lag, "iters": st_l.iters, "iterations_per_s": st_l.iters / t_lag,
                  "switch_iters": {"ur32": st_l.it_ur32, "uz32": st_l.it_uz32, "uz16": st_l.it_uz16},
                  "relres_updated": st_l.relres_updated, "speedup_vs_own_fp64": t_fp64 / t_lag}

    # ---- roofline of the dominant kernel (SpMV) timed alone with CUDA events ----
    peak, peak_src = peaks()
    m = s.nnz / s.n
    reps = 20
    npad = (s.n + 7) // 8 * 8
    roof = {}
    for tag, matp, pt, sA, sz in (("fp32mat_fp16vec", A.FP32, torch.float16, 4, 2), ("fp64mat_fp64vec", A.FP64, torch.float64, 8, 8)):
        pvec = torch.zeros(npad, dtype=pt, device=dev)
        pvec[: s.n] = torch.from_numpy(np.cos(np.arange(s.n) * 0.37)).to(dev).to(pt)
        q = torch.empty(s.n, dtype=torch.float32 if matp == A.FP32 else torch.float64, device=dev)
        for _ in range(3):
            h.spmv(pvec, matp, out=q)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            h.spmv(pvec, matp, out=q)
        e1.record(stream); e1.synchronize()
        dur_ms = e0.elapsed_time(e1) / reps
        # bytes this handle's matrix format must move per launch (amp_pcg_spmv_bytes):
        # stored values + the index data actually read + p once + q once
        alg_bytes = h.spmv_bytes(matp, A.FP16 if pt == torch.float16 else A.FP64)
        csr_bytes = s.n * (m * (sA + 4) + 4 + sz + sA)  # the same mat-vec in plain CSR
        roof[tag] = {"bound": "hbm", "achieved": alg_bytes / dur_ms * 1e-6, "peak": peak, "unit": "GB/s",
                     "frac": alg_bytes / dur_ms * 1e-6 / peak, "traffic": NCU_TRAFFIC.get((s.name.split("@")[0], tag)),
                     "kernel": "k_spmv_any (phase_spmv)",
                     "us_per_launch": dur_ms * 1e3, "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src,
                     "csr_equivalent_bytes_per_launch": csr_bytes, "csr_equivalent_gbs": csr_bytes / dur_ms * 1e-6}
    roofline = dict(roof["fp32mat_fp16vec"])
    roofline["fp64"] = {k: roof["fp64mat_fp64vec"][k] for k in ("achieved", "frac", "us_per_launch", "algorithmic_bytes_per_launch",
                                                                "traffic", "csr_equivalent_gbs")}
    loop_gbs = st.algorithmic_bytes / (statistics.median(ms) * 1e-3) * 1e-9
    loop64_gbs = st64.algorithmic_bytes / (statistics.median(ms64) * 1e-3) * 1e-9
    roofline["whole_loop"] = {"amp_gbs": loop_gbs, "amp_frac": loop_gbs / peak, "amp_frac_of_8TBs": loop_gbs / 8000.0,
                              "fp64_gbs": loop64_gbs, "fp64_frac": loop64_gbs / peak}

    # ---- CPU oracle on the host cores (reported baseline, not the target) ----
    cpu = None
    if not args.no_cpu_baseline:
        import oracle as O

        cap = min(150, s.maxit)
        tt0 = time.perf_counter()
        r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, cap, O.make_policy(**kw))
        dt = time.perf_counter() - tt0
        cpu = {"value": r.iters / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
               "sample": f"first {r.iters} iterations of the same AMP-PCG solve on {s.name} ({dt:.1f} s, OpenMP, all cores)"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64 (r,q,A: f64->f32; z,p storage: f64->f32->f16; x, dots f64)", "data": "synthetic",
        "config": {"workload": s.name, "n": s.n, "nnz": s.nnz, "tol": s.tol, "maxit": s.maxit, "policy": args.policy,
                   "precond": "jacobi", "x0": "zero", "loop": {0: "auto", 1: "stream", 2: "graph", 3: "persistent"}[st.loop_mode],
                   "l2": "L2 flushed (256 MiB write) before every timed solve; working set > 126 MB L2",
                   "replicas": world},
        "time_to_tol_s": t_amp, "iters": st.iters, "switch_iters": {"ur32": st.it_ur32, "uz32": st.it_uz32, "uz16": st.it_uz16},
        "relres_updated": st.relres_updated,
        "fp64_pcg": {"time_to_tol_s": t_fp64, "iters": st64.iters, "iterations_per_s": st64.iters / t_fp64},
        "amp_speedup_vs_own_fp64": t_fp64 / t_amp,
        "lagged_scale_variant": lagged,
        "paper_speedup_context": "1.63x on A100 SXM 40GB, matrix-free FEM (PAPER.md:506) - other hardware and operator",
        "create_s": create_s,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * s.n, "d2h_bytes_per_step": 8 * s.n,
                "ms_per_step": tot_e / args.steps, "api": "amp_pcg_solve_host (pinned host b, x)"},
        "gpu_launches": launches_all,
        "clocks": clk.result,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    h.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
