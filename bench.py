#!/usr/bin/env python
"""bench.py — AMP-PCG time-to-tolerance / iterations per second on one B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4] [--impl ours|reference]

One "step" = one whole solve (every row of SURVEY.md §8(a): set-up, then per iteration the fused
z/(r,z), p, SpMV/(p,Ap), x/r/||r|| kernels with device-side precision switching) of the seeded
synthetic system `--workload` from x0 = 0, with A resident in HBM.  Default workload: c4 =
BASELINE.json configs[3], the 27-point FE Laplacian 200^3 (n = 8 M, nnz = 213.8 M), the LARGEST
single-GPU configuration (BASELINE.json's metric names no configuration).  `value` = PCG iterations per
second over all ranks (N > 1: independent replicas, one per GPU, no data-path collective: "weak").
`roofline` is measured on the kernels the loop itself runs: one extra solve with the stream-driven loop and a CUDA
event between every two kernels (amp_policy_t.profile_kernels); each kernel's time is the average over all its
launches in the dominant precision phase (u_z, u_r) = (FP16, FP32); the per-iteration working set of c4 (1.3 GB)
is ten times the L2, so every launch starts cold.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import ctypes
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
DTYPE = "f64 (r,q,A: f64->f32; z,p storage: f64->f32->f16; x, dots f64)"
POLICIES = {
    "amp_fp64_delay": dict(amp=1, u0=0, eta_rule=0),                                          # paper: AMP-PCG(FP64), (4.9)+(4.10)
    "amp_fp16_linear": dict(amp=1, u0=2, eta_rule=1),                                         # paper: AMP-PCG(FP16), (4.11)
    # theta-split of (3.10) (reading R12): switch u_r at eta_k <= theta tol ||b||, stop at
    # ||r_k|| <= (1 - theta) tol ||b||  =>  ||b - A x|| <= ||zeta|| + ||r|| <~ tol ||b||: the policies that meet north_star's
    # "true relative residual <= tol".  theta = 0.3 is the headline: smallest summed (and geometric-mean) time to tolerance over
    # c2, c3, c4 among theta in {0.1 .. 0.5}, all of which reach true relres <= tol in the oracle at full size
    # (tests/golden/oracle_full_size.json) and on the GPU (profiles/r03_theta_sweep.txt)
    "amp_fp64_delay_strict": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.1, stop_safety=0.9),
    "amp_fp64_delay_strict_t03": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.3, stop_safety=0.7),
    "amp_fp64_delay_strict_t05": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.5, stop_safety=0.5),
    "amp_fp16_linear_strict_t03": dict(amp=1, u0=2, eta_rule=1, eta_safety=0.3, stop_safety=0.7),
    # omega = sqrt(n)/||r_k|| (PAPER.md:34, :223 allow other scaling factors; reading R10): on c3 it takes the FP16
    # stores of z, p out of the subnormal range (oracle, full size: 90 % -> 0.2 % subnormal; 928 -> 901 iterations, FP64: 898)
    "amp_fp64_delay_rms": dict(amp=1, u0=0, eta_rule=0, scale_mode=1),
}


HEADLINE_POLICY = "amp_fp64_delay_strict_t03"
PAPER_POLICY = "amp_fp64_delay"  # Algorithm 4.1 with (4.10) and line 18 as printed: true relres <~ 2 tol


def policy_label(name: str) -> str:
    kw = POLICIES[name]
    if "eta_safety" in kw:
        return (f"{name} (Alg 4.1, theta-split of (3.10): u_r switch at eta_k <= {kw['eta_safety']} tol||b||, stop at "
                f"||r_k|| <= {kw['stop_safety']} tol||b||; criterion: true relres <= tol)")
    return f"{name} (Alg 4.1 as printed: switch at eta_k <= tol||b||, stop at ||r_k|| <= tol||b||; the paper promises true relres <~ 2 tol)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--size", type=int, default=None, help="override grid edge / rows (debug only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--policy", default=HEADLINE_POLICY, choices=sorted(POLICIES))
    ap.add_argument("--loop", default="auto", choices=["auto", "stream", "graph", "persistent"])
    ap.add_argument("--spmv-kernel", default="auto", choices=["auto", "direct", "pipelined"])
    ap.add_argument("--vec-kernel", default="auto", choices=["auto", "direct", "staged"])
    ap.add_argument("--fuse", default="auto", choices=["auto", "off", "on"], help="fused vector kernel (create option fuse_vec)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--others", default="c2,c3,c1,c5",
                    help="comma list of further workloads to report under 'other_workloads' (value / time_to_tol / speed-up "
                         "only; '' = none); a workload is skipped once --time-budget seconds have passed")
    ap.add_argument("--time-budget", type=float, default=100.0,
                    help="seconds after which the optional legs (other workloads) are skipped, so that the default run ends "
                         "within a few minutes")
    ap.add_argument("--cheb-degrees", default="2,3", help="degrees of the Chebyshev-Jacobi preconditioner to time beside "
                                                           "the Jacobi headline ('' = none)")
    ap.add_argument("--profile-iters", type=int, default=0,
                    help="profiling aid for ncu: run ONE solve of this many iterations with plain stream launches "
                         "(u_r forced to FP32 from k=ell so the low-precision kernels appear) and exit; prints no bench line")
    ap.add_argument("--profile-policy", default="amp_fp16_linear",
                    choices=["pcg_fp64", "amp_fp16_linear", "amp_fp64_delay", "amp_fp16_linear_lagged", "amp_fp64_ur32",
                             "amp_fp32_ur32"])
    ap.add_argument("--ref-iters", type=int, default=0, help="--impl reference: iterations per step (0 = sized to the workload)")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: ONE system row-sharded over the N ranks (amp_pcg_solve_sharded: halo of p and the three inner "
                         "products exchanged by the loop kernels over peer memory; strong scaling) instead of N replicas")
    ap.add_argument("--shard-local", type=int, default=0,
                    help="one GPU: emulate this many ranks of the row-sharded solve in one process (lock-step launches on one "
                         "stream; functional check and overhead of the sharded kernels, not a scaling number)")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture of THIS round
    (profiles/r03_ncu_traffic.csv names the capture each value comes from), else None."""
    path = os.path.join(ROOT, "profiles", "r03_ncu_traffic.csv")
    try:
        for line in open(path).read().splitlines()[1:]:
            f = line.split(",")
            if len(f) >= 3 and f[0] == workload and f[1] == kernel:
                return float(f[2])
    except (OSError, ValueError):
        pass
    return None


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
    return dict(POLICIES[name])


def config_dict(s, policy: str, world: int):
    """the `config` object: identical for our arm and the reference arm (same workload, tolerance, policy)"""
    return {"workload": s.name, "n": s.n, "nnz": s.nnz, "tol": s.tol, "maxit": s.maxit, "policy": policy_label(policy),
            "precond": "jacobi", "x0": "zero",
            "l2": "L2 flushed (256 MiB write) before every timed solve; per-iteration working set > 126 MB L2 "
                  "(c1 excepted: it lives in L2 by construction)",
            "replicas": world}


# --------------------------------------------------------------------------------------------
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def omp_set_threads(n: int):
    """thread count of the oracle's OpenMP loops (libgomp is already loaded by the oracle library)"""
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def oracle_sample_iters(s):
    """iterations of the bounded CPU sample: about 10-30 s of host work for all legs together"""
    per_it_all = s.nnz * 1.4e-10 + s.n * 1.2e-9  # rough seconds per oracle iteration on ~16 threads (round-1 runs)
    return int(max(5, min(150, 5.0 / per_it_all)))


def cpu_baseline_leg(s, kw):
    """SURVEY.md section 8(d) "CPU baseline": the oracle's FP64 PCG on all host cores and on one thread, the AMP-PCG
    emulation (software rounding: artificially slow) beside it; a bounded sample of the same solve."""
    import oracle as O

    ncores = os.cpu_count() or 1
    cap = min(oracle_sample_iters(s), s.maxit)
    out = {"unit": UNIT, "kind": "oracle", "cores": ncores, "cpu_model": cpu_model()}
    omp_set_threads(ncores)
    t0 = time.perf_counter()
    r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, cap, O.make_policy(amp=0))
    dt = time.perf_counter() - t0
    out["value"] = r.iters / dt
    out["sample"] = (f"oracle FP64 PCG (Alg 3.1), first {r.iters} iterations of the solve of {s.name} "
                     f"({dt:.1f} s, OpenMP, {ncores} threads)")
    t0 = time.perf_counter()
    r2 = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, cap, O.make_policy(**kw))
    dt2 = time.perf_counter() - t0
    out["amp_emulation"] = {"value": r2.iters / dt2, "kind": "oracle_amp_emulation", "cores": ncores,
                            "sample": f"first {r2.iters} iterations of AMP-PCG with software-rounded storage ({dt2:.1f} s)"}
    if omp_set_threads(1):
        cap1 = max(3, cap // 6)
        t0 = time.perf_counter()
        r1 = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, cap1, O.make_policy(amp=0))
        dt1 = time.perf_counter() - t0
        out["one_thread"] = {"value": r1.iters / dt1, "cores": 1,
                             "sample": f"oracle FP64 PCG, first {r1.iters} iterations, 1 thread ({dt1:.1f} s)"}
        omp_set_threads(ncores)
    return out


def run_reference(args, rank: int, world: int):
    """--impl reference: the CPU oracle as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle as O
    from workloads import make_config

    s = make_config(args.workload, args.size)
    kw = policy_kwargs(args.policy)
    pol = O.make_policy(**kw)
    cap = min(args.ref_iters or max(3, oracle_sample_iters(s) // 3), s.maxit)
    times, its = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, cap, pol)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt); its += r.iters
    total = sum(times)
    val = its / total
    sample = f"each step = the first {cap} iterations of the AMP-PCG solve of {s.name} (software-rounded storage)"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / max(len(times), 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
        "config": config_dict(s, args.policy, world),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def time_weighted(prof: dict, kernel: str) -> dict:
    """all launches of one kernel over the phases of a solve: total compulsory bytes / total time, and the worst phase"""
    tb = tt = 0.0
    nl = 0
    worst, worst_gbs = None, float("inf")
    for phase, ks in prof.items():
        r = ks.get(kernel)
        if not r:
            continue
        tb += r["algorithmic_bytes_per_launch"] * r["launches"]
        tt += r["us_per_launch"] * r["launches"]
        nl += r["launches"]
        if r["achieved_gbs"] < worst_gbs:
            worst, worst_gbs = phase, r["achieved_gbs"]
    if nl == 0:
        return {"achieved_gbs": 0.0, "us_per_launch": 0.0, "launches": 0, "bytes_per_launch": 0.0, "worst_phase": None, "worst_frac": 0.0}
    return {"achieved_gbs": tb / tt * 1e-3, "us_per_launch": tt / nl, "launches": nl, "bytes_per_launch": tb / nl,
            "worst_phase": worst, "worst_frac": worst_gbs}


# --------------------------------------------------------------------------------------------
class Runner:
    """one workload resident on one GPU: timed solves of a policy, each preceded by an L2 flush"""

    def __init__(self, A, torch, s, dev, loop, spmv_kernel, share=None, precond=None, **opts):
        self.A, self.torch, self.s, self.dev = A, torch, s, dev
        if share is not None:  # same matrix already on the device
            self.rp, self.ci, self.va, self.b = share.rp, share.ci, share.va, share.b
        else:
            self.rp, self.ci, self.va, self.b = (torch.from_numpy(a).to(dev) for a in (s.rowptr, s.colidx, s.vals, s.b))
        t0 = time.perf_counter()
        self.h = A.AmpPcg(self.rp, self.ci, self.va, A.PRECOND_JACOBI if precond is None else precond,
                          spmv_kernel=spmv_kernel, **opts)
        torch.cuda.synchronize()
        self.create_s = time.perf_counter() - t0
        self.loop = loop
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # 256 MiB > 126 MB L2
        self.x = torch.zeros(s.n, dtype=torch.float64, device=dev)
        self.stream = torch.cuda.current_stream(dev)

    def policy(self, name_or_kw, **extra):
        kw = policy_kwargs(name_or_kw) if isinstance(name_or_kw, str) else dict(name_or_kw)
        kw.update(extra)
        kw.setdefault("loop_mode", self.loop)
        return self.A.Policy.default(x0_zero=1, **kw)

    def timed(self, policy, count, host=False, bh=None, xh=None):
        """count solves, each bracketed by CUDA events on the solve stream, L2 flushed before each."""
        torch, s, h = self.torch, self.s, self.h
        ms, its, launches, last = [], 0, 0, None
        for _ in range(count):
            self.flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.stream)
            if host:
                st = h.solve_host(bh, xh, s.tol, s.maxit, policy)
            else:
                st = h.solve(self.b, self.x, s.tol, s.maxit, policy)
            e1.record(self.stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1)); its += st.iters; launches += h.last_launch_count(); last = st
        return ms, its, launches, last

    def summary(self, name_or_kw, reps, **extra):
        """median time-to-tolerance of a policy + its true residual (one extra, untimed solve with true_residual=1)"""
        pol = self.policy(name_or_kw, **extra)
        self.timed(pol, 1)
        ms, _, _, st = self.timed(pol, reps)
        t = statistics.median(ms) * 1e-3
        st_true = self.h.solve(self.b, self.x, self.s.tol, self.s.maxit, self.policy(name_or_kw, true_residual=1, **extra))
        return {"time_to_tol_s": t, "iters": st.iters, "iterations_per_s": st.iters / t,
                "switch_iters": {"ur32": st.it_ur32, "uz32": st.it_uz32, "uz16": st.it_uz16},
                "relres_updated": st.relres_updated, "relres_true": st_true.relres_true,
                "relres_true_le_tol": bool(st_true.relres_true <= self.s.tol)}, st

    def kernel_profile(self, name_or_kw, peak, **extra):
        """per-kernel device times inside the loop (stream loop, an event between every two kernels)"""
        A = self.A
        pol = self.policy(name_or_kw, loop_mode=A.LOOP_STREAM, profile_kernels=1, **extra)
        self.flush.fill_(1)
        self.h.solve(self.b, self.x, self.s.tol, self.s.maxit, pol)
        recs = self.h.kernel_times()
        names = {0: "fp64", 1: "fp32", 2: "fp16"}
        out = {}
        for r in recs:
            us = 1e3 * r["total_ms"] / r["launches"]
            gbs = r["bytes_per_launch"] / us * 1e-3
            out.setdefault(f"uz={names[r['uz']]},ur={names[r['ur']]}", {})[r["kernel"]] = {
                "launches": r["launches"], "us_per_launch": us, "algorithmic_bytes_per_launch": r["bytes_per_launch"],
                "achieved_gbs": gbs, "frac": gbs / peak}
        return out

    def close(self):
        self.h.close()


def run_ours(args, rank: int, local_rank: int, world: int):
    import numpy as np  # noqa: F401
    import torch

    t_start = time.perf_counter()

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

    loop = {"auto": A.LOOP_AUTO, "stream": A.LOOP_STREAM, "graph": A.LOOP_GRAPH, "persistent": A.LOOP_PERSISTENT}[args.loop]
    spmv_kernel = {"auto": A.SPMV_AUTO, "direct": A.SPMV_DIRECT, "pipelined": A.SPMV_PIPELINED}[args.spmv_kernel]
    s = make_config(args.workload, args.size)
    vec_kernel = {"auto": A.VEC_AUTO, "direct": A.VEC_DIRECT, "staged": A.VEC_STAGED}[args.vec_kernel]
    fuse = {"auto": A.FUSE_AUTO, "off": A.FUSE_OFF, "on": A.FUSE_ON}[args.fuse]
    R = Runner(A, torch, s, dev, loop, spmv_kernel, vec_kernel=vec_kernel, fuse_vec=fuse)
    h = R.h
    if args.profile_iters > 0:
        kwp = {"pcg_fp64": dict(amp=0), "amp_fp16_linear": dict(u0=A.FP16, eta_rule=A.ETA_LINEAR, eps32=1e-30),
               "amp_fp16_linear_lagged": dict(u0=A.FP16, eta_rule=A.ETA_LINEAR, eps32=1e-30, scale_mode=A.SCALE_LAGGED),
               # phases (FP64, FP32) and (FP32, FP32) from k = 5 on: u_z held by the thresholds, u_r forced down
               "amp_fp64_ur32": dict(u0=A.FP64, eta_rule=A.ETA_LINEAR, eps32=1e-30, tau_zs=0.0, tau_zh=0.0),
               "amp_fp32_ur32": dict(u0=A.FP32, eta_rule=A.ETA_LINEAR, eps32=1e-30, tau_zs=0.0, tau_zh=0.0),
               "amp_fp64_delay": dict()}[args.profile_policy]
        lp = A.LOOP_STREAM if args.loop == "auto" else loop
        stp = h.solve(R.b, R.x, s.tol, args.profile_iters, A.Policy.default(x0_zero=1, loop_mode=lp, **kwp))
        print("profile run:", stp.asdict(), file=sys.stderr)
        R.close()
        return
    kw = policy_kwargs(args.policy)
    pol = R.policy(args.policy)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up, then EXACTLY K timed steps between barriers ----
    R.timed(pol, args.warmup)
    barrier()
    with ClockSampler(local_rank) as clk:
        ms, its, launches, st = R.timed(pol, args.steps)
    barrier()
    total_ms = sum(ms)
    (total_ms_max,), (its_all, launches_all) = reduce_over_ranks(dist, [total_ms], [its, launches], dev)
    launches_all = int(launches_all)
    value = its_all / (total_ms_max * 1e-3)

    # ---- end-to-end through the host-buffer entry point (H2D of b, solve, D2H of x inside) ----
    bh = torch.from_numpy(s.b).pin_memory()
    xh = torch.zeros(s.n, dtype=torch.float64).pin_memory()
    R.timed(pol, 1, host=True, bh=bh, xh=xh)
    barrier()
    ms_e, its_e, _, _ = R.timed(pol, args.steps, host=True, bh=bh, xh=xh)
    barrier()
    (tot_e,), (its_e,) = reduce_over_ranks(dist, [sum(ms_e)], [its_e], dev)
    e2e_value = its_e / (tot_e * 1e-3)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    reps = max(2, min(args.steps, 3))
    peak, peak_src = peaks()
    # ---- the headline policy again with its true residual, this library's own FP64 PCG (north_star: AMP must beat
    #      it), the theta-split policy that guarantees true relres <= tol (reading R12), the lagged variant (R17) ----
    amp_sum, _ = R.summary(args.policy, reps)
    fp64_sum, st64 = R.summary(dict(amp=0), reps)
    paper_sum, _ = R.summary(PAPER_POLICY, reps)
    theta_sums = {nm: R.summary(nm, reps)[0] for nm in ("amp_fp64_delay_strict", "amp_fp64_delay_strict_t05") if nm != args.policy}
    # AMP-PCG(FP16) with the linear indicator (4.11): the variant the paper times in Example 7
    fp16_sums = {nm: R.summary(nm, reps)[0] for nm in ("amp_fp16_linear", "amp_fp16_linear_strict_t03")}
    lag_sum, _ = R.summary(args.policy, reps, scale_mode=A.SCALE_LAGGED)
    rms_sum, _ = R.summary(args.policy, reps, scale_mode=A.SCALE_RMS)
    t_amp = statistics.median(ms) * 1e-3
    t_fp64 = fp64_sum["time_to_tol_s"]
    for d in (paper_sum, lag_sum, rms_sum, *theta_sums.values(), *fp16_sums.values()):
        d["speedup_vs_own_fp64"] = t_fp64 / d["time_to_tol_s"]

    # ---- roofline: the kernels the loop runs, timed inside the loop ----
    prof = R.kernel_profile(args.policy, peak)
    prof_lag = R.kernel_profile(args.policy, peak, scale_mode=A.SCALE_LAGGED)
    prof64 = R.kernel_profile(dict(amp=0), peak)
    dom_phase = "uz=fp16,ur=fp32"
    if dom_phase not in prof or "k_spmv" not in prof[dom_phase]:
        dom_phase = max(prof, key=lambda ph: prof[ph].get("k_spmv", {}).get("launches", 0))
    dom = prof[dom_phase]["k_spmv"]
    wl = s.name.split("@")[0]
    tw = time_weighted(prof, "k_spmv")
    roofline = {
        # the dominant kernel is the mat-vec (a4); achieved / frac are TIME-WEIGHTED over all its launches of one solve (every
        # precision phase: bytes of each phase's format and precisions / time of that phase's launches), the per-phase table
        # is in kernels_by_phase and the worst phase is named
        "bound": "hbm", "achieved": tw["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": tw["achieved_gbs"] / peak,
        "traffic": ncu_traffic(wl, "k_spmv"), "traffic_is_for_phase": "uz=fp16,ur=fp32",
        "kernel": "k_spmv (in-loop, all phases of the solve, time-weighted)", "us_per_launch": tw["us_per_launch"],
        "launches_averaged": tw["launches"], "algorithmic_bytes_per_launch": tw["bytes_per_launch"],
        "worst_phase": tw["worst_phase"], "worst_phase_frac": tw["worst_frac"] / peak,
        "vec_fused_time_weighted": {k: v for k, v in time_weighted(prof, "k_vec_fused").items() if k != "worst_frac"}
        if any("k_vec_fused" in v for v in prof.values()) else None,
        "last_phase": {"phase": dom_phase, "k_spmv_frac": dom["frac"], "k_spmv_us": dom["us_per_launch"]},
        "peak_source": peak_src,
        "how": "stream-driven loop, CUDA event between every two kernels (policy.profile_kernels); average over all "
               "launches of the phase inside one solve; working set per iteration >> L2",
        "kernels": prof[dom_phase], "kernels_by_phase": prof,
        "kernels_lagged_variant": prof_lag.get(dom_phase), "kernels_fp64_pcg": prof64.get("uz=fp64,ur=fp64"),
    }
    loop_gbs = st.algorithmic_bytes / t_amp * 1e-9
    loop64_gbs = st64.algorithmic_bytes / t_fp64 * 1e-9
    roofline["whole_loop"] = {"amp_gbs": loop_gbs, "amp_frac": loop_gbs / peak, "amp_frac_of_8TBs": loop_gbs / 8000.0,
                              "fp64_gbs": loop64_gbs, "fp64_frac": loop64_gbs / peak}

    # ---- NEXT-4: the same solve with the Chebyshev-accelerated Jacobi preconditioner (the paper's smoother) ----
    cheb = {}
    for deg in [int(t) for t in args.cheb_degrees.split(",") if t]:
        Rc = Runner(A, torch, s, dev, loop, spmv_kernel, share=R, precond=A.PRECOND_CHEBJACOBI, cheb_degree=deg, vec_kernel=vec_kernel)
        a_, _ = Rc.summary(args.policy, 2)
        f_, _ = Rc.summary(dict(amp=0), 2)
        cheb[f"degree_{deg}"] = {"amp": a_, "fp64_pcg": f_, "amp_speedup_vs_fp64_same_precond": f_["time_to_tol_s"] / a_["time_to_tol_s"],
                                 "speedup_vs_jacobi_amp": t_amp / a_["time_to_tol_s"],
                                 "matvecs_per_solve": deg * a_["iters"]}
        Rc.close()
        del Rc

    # ---- the other BASELINE.json configs (parity-test cases; reported for context) ----
    others = {}
    for name in [t for t in args.others.split(",") if t and t != args.workload]:
        if time.perf_counter() - t_start > args.time_budget:
            others.setdefault("skipped_for_time", []).append(name)
            continue
        so = make_config(name)
        Ro = Runner(A, torch, so, dev, loop, spmv_kernel, vec_kernel=vec_kernel, fuse_vec=fuse)
        a_, sta = Ro.summary(args.policy, 2)
        f_, _ = Ro.summary(dict(amp=0), 2)
        l_, _ = Ro.summary(args.policy, 2, scale_mode=A.SCALE_LAGGED)
        r_, _ = Ro.summary(args.policy, 2, scale_mode=A.SCALE_RMS)
        pp_, _ = Ro.summary(PAPER_POLICY, 2)
        po = Ro.kernel_profile(args.policy, peak)
        last = max(po, key=lambda ph: (ph.count("fp16"), ph.count("fp32")))  # the final (lowest-precision) phase of the solve
        lg = sta.algorithmic_bytes / a_["time_to_tol_s"] * 1e-9
        others[so.name] = {"value": a_["iterations_per_s"], "time_to_tol_s": a_["time_to_tol_s"], "iters": a_["iters"],
                           "relres_true": a_["relres_true"], "relres_true_le_tol": a_["relres_true_le_tol"],
                           "switch_iters": a_["switch_iters"],
                           "algorithmic_bytes": sta.algorithmic_bytes, "whole_loop_gbs": lg, "whole_loop_frac": lg / peak,
                           "whole_loop_frac_of_8TBs": lg / 8000.0,
                           "k_spmv_time_weighted_frac": time_weighted(po, "k_spmv")["achieved_gbs"] / peak,
                           "k_vec_time_weighted_frac": time_weighted(po, "k_vec_fused")["achieved_gbs"] / peak,
                           "last_phase": last, "last_phase_kernels": {k: {"us_per_launch": v["us_per_launch"], "frac": v["frac"], "launches": v["launches"]}
                                                                      for k, v in po[last].items()},
                           "paper_policy_time_to_tol_s": pp_["time_to_tol_s"], "paper_policy_relres_true": pp_["relres_true"],
                           "paper_policy_speedup_vs_own_fp64": f_["time_to_tol_s"] / pp_["time_to_tol_s"],
                           "fp64_pcg_time_to_tol_s": f_["time_to_tol_s"],
                           "amp_speedup_vs_own_fp64": f_["time_to_tol_s"] / a_["time_to_tol_s"],
                           "lagged_time_to_tol_s": l_["time_to_tol_s"],
                           "lagged_speedup_vs_own_fp64": f_["time_to_tol_s"] / l_["time_to_tol_s"],
                           "fp64_pcg_iters": f_["iters"], "rms_scale_iters": r_["iters"],
                           "rms_scale_time_to_tol_s": r_["time_to_tol_s"],
                           "rms_scale_speedup_vs_own_fp64": f_["time_to_tol_s"] / r_["time_to_tol_s"]}
        Ro.close()
        del Ro

    # ---- CPU oracle on the host cores (reported baseline, not the target) ----
    cpu = None if args.no_cpu_baseline else cpu_baseline_leg(s, kw)

    loop_name = {0: "auto", 1: "stream", 2: "graph", 3: "persistent"}[st.loop_mode]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": DTYPE, "data": "synthetic",
        "config": config_dict(s, args.policy, world), "loop_driver": loop_name,
        "time_to_tol_s": t_amp, "iters": st.iters, "us_per_iteration": 1e6 * t_amp / max(st.iters, 1),
        "switch_iters": {"ur32": st.it_ur32, "uz32": st.it_uz32, "uz16": st.it_uz16},
        "relres_updated": st.relres_updated, "relres_true": amp_sum["relres_true"],
        "relres_true_le_tol": amp_sum["relres_true_le_tol"],
        "fp64_pcg": fp64_sum,
        "amp_speedup_vs_own_fp64": t_fp64 / t_amp,
        "amp_speedup_claim_rests_on": "the headline policy (config.policy), which stops at the same true accuracy as the FP64 arm "
                                      "(true relres <= tol); Algorithm 4.1 as printed and the lagged variant are reported beside it",
        "paper_policy_as_printed": paper_sum,
        "other_theta_splits": theta_sums,
        "amp_pcg_fp16_linear": fp16_sums,
        "lagged_scale_variant": lag_sum,
        "rms_scale_variant": rms_sum,
        "paper_speedup_context": "1.63x on A100 SXM 40GB, matrix-free FEM (PAPER.md:506) - other hardware and operator",
        "create_s": R.create_s,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * s.n, "d2h_bytes_per_step": 8 * s.n,
                "ms_per_step": tot_e / args.steps, "api": "amp_pcg_solve_host (pinned host b, x)"},
        "gpu_launches": launches_all,
        "clocks": clk.result,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    if cheb:
        line["chebyshev_jacobi_preconditioner"] = cheb
    if others:
        line["other_workloads"] = others
    print(json.dumps(line), flush=True)
    R.close()
    if dist is not None:
        dist.destroy_process_group()


def run_sharded(args, rank: int, local_rank: int, world: int):
    """One system row-sharded over the ranks: --shard under torchrun (one process per
    GPU, peers wired through CUDA IPC) or --shard-local W (W ranks emulated on one GPU by one process)."""
    import torch

    import paper_2505_04155_b200 as A
    from workloads import make_config

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    s = make_config(args.workload, args.size)
    local = args.shard_local > 0
    nranks = args.shard_local if local else world
    dist = None
    if not local:
        import torch.distributed as dist_

        dist = dist_
        dist.init_process_group("nccl", device_id=dev)
    plan = A.shard_plan(s.rowptr, s.colidx, nranks)
    mine = list(range(nranks)) if local else [rank]
    handles, bs, xs = [], [], []
    for r in mine:
        sh = plan[r]
        rp, ci, va = A.shard_extract(s.rowptr, s.colidx, s.vals, sh)
        handles.append(A.AmpPcg(torch.from_numpy(rp).to(dev), torch.from_numpy(ci).to(dev), torch.from_numpy(va).to(dev),
                                A.PRECOND_JACOBI, halo_lo=sh.halo_lo, halo_hi=sh.halo_hi))
        bs.append(torch.from_numpy(s.b[sh.row0:sh.row1].copy()).to(dev))
        xs.append(torch.zeros(sh.row1 - sh.row0, dtype=torch.float64, device=dev))
    if local:
        g = A.ShardGroup.attach_local(handles)
    else:
        blobs = [None] * world
        dist.all_gather_object(blobs, A.ShardGroup.export(handles[0]))   # plumbing: the IPC handles of every rank
        g = A.ShardGroup.attach_ipc(handles[0], rank, blobs)
    pol = A.Policy.default(x0_zero=1, **policy_kwargs(args.policy))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if dist is not None:
            dist.barrier()      # also required by the library: no rank starts a solve before all have finished the last
        torch.cuda.synchronize()

    def timed(count):
        ms, st = [], None
        for _ in range(count):
            flush.fill_(1)
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            st = g.solve(bs, xs, s.tol, s.maxit, pol)[0]
            e1.record(stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        return ms, st

    timed(args.warmup)
    barrier()
    with ClockSampler(local_rank) as clk:
        ms, st = timed(args.steps)
    barrier()
    (tot,), _ = reduce_over_ranks(dist, [sum(ms)], [0], dev)
    st_true = g.solve(bs, xs, s.tol, s.maxit, A.Policy.default(x0_zero=1, true_residual=1, **policy_kwargs(args.policy)))[0]
    launches = sum(h.last_launch_count() for h in handles)
    if rank == 0:
        halo = [int(p_.halo_lo + p_.halo_hi) for p_ in plan]
        line = {
            "metric": METRIC, "value": args.steps * st.iters / (tot * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
            "config": dict(config_dict(s, args.policy, 1), sharded_ranks=nranks,
                           mode="emulated on one GPU (lock-step launches)" if local else "one process per GPU, CUDA IPC peers"),
            "iters": st.iters, "switch_iters": {"ur32": st.it_ur32, "uz32": st.it_uz32, "uz16": st.it_uz16},
            "relres_updated": st.relres_updated, "relres_true": st_true.relres_true, "time_to_tol_s": statistics.median(ms) * 1e-3,
            "rows_per_rank": [int(p_.row1 - p_.row0) for p_ in plan], "halo_entries_per_rank": halo,
            "halo_bytes_per_iteration_fp16": 2 * sum(halo), "halo_bytes_per_iteration_fp64": 8 * sum(halo),
            "gpu_launches": launches, "clocks": clk.result,
        }
        print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.shard_local > 0 or (args.shard and world > 1):
        run_sharded(args, rank, local_rank, world)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
