"""Write tests/golden/oracle_full_size.json: the CPU oracle's results on the five BASELINE.json
configs at FULL size, for the policies the GPU parity tests and bench.py use.

This script calls only ``oracle/`` and ``workloads/`` (never the CUDA path).  The paper prints
no iteration counts for these synthetic systems, so these values are "parity unpinned" by the
paper: they pin GPU <-> oracle agreement only ("Oracle pins").

    python tests/golden/make_oracle_golden.py [--force] [c1 c2 ...]      # minutes of CPU time

Policies already present in the file for a config are kept (their inputs are seeded and the oracle is
deterministic); --force recomputes them.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle as O  # noqa: E402
from workloads import CONFIGS, make_config  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_full_size.json")

POLICIES = {
    "pcg_fp64": dict(amp=0),
    "amp_fp64_delay": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY),
    "amp_fp16_linear": dict(amp=1, u0=O.FP16, eta_rule=O.ETA_LINEAR),
    "amp_fp64_delay_strict": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY, eta_safety=0.1, stop_safety=0.9),
    # the (3.10) split "switch at eta <= theta tol ||b||, stop at ||r|| <= (1 - theta) tol ||b||" for
    # other theta: the sweep behind bench.py's choice of the headline policy (rule: true relres <= tol on c2-c4, then the
    # fewest iterations with the FP64 matrix + extra iterations at the end; reading R12)
    "amp_fp64_delay_strict_t02": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY, eta_safety=0.2, stop_safety=0.8),
    "amp_fp64_delay_strict_t03": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY, eta_safety=0.3, stop_safety=0.7),
    "amp_fp64_delay_strict_t05": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY, eta_safety=0.5, stop_safety=0.5),
    "amp_fp64_delay_lagged": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY, scale_mode=O.SCALE_LAGGED),
    # omega = sqrt(n)/||r_k|| ("other scaling factors can be used"): the evidence for the scaling
    # decision of DESIGN.md section 2 (reading R10) — FP16 subnormal exposure and iteration counts at full size
    "amp_fp64_delay_rms": dict(amp=1, u0=O.FP64, eta_rule=O.ETA_DELAY, scale_mode=O.SCALE_RMS),
    "amp_fp16_linear_rms": dict(amp=1, u0=O.FP16, eta_rule=O.ETA_LINEAR, scale_mode=O.SCALE_RMS),
}


def main(names):
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    data["_about"] = ("CPU-oracle results at full size (written by tests/golden/make_oracle_golden.py, which calls "
                      "only oracle/ and workloads/). Not printed by the paper: GPU<->oracle parity only.")
    for name in names:
        t0 = time.time()
        s = make_config(name)
        rng_p = 2.0 * np.modf(np.arange(s.n) * 0.6180339887498949)[0] - 1.0  # deterministic probe vector
        q = O.spmv_fp64(s.rowptr, s.colidx, s.vals, rng_p)
        sample = np.linspace(0, s.n - 1, 64).astype(np.int64)
        old = data.get(name, {}).get("policies", {}) if not FORCE else {}
        entry = {"n": s.n, "nnz": s.nnz, "tol": s.tol, "maxit": s.maxit, "gen_s": round(time.time() - t0, 1),
                 "spmv_probe": {"rows": sample.tolist(), "q": [float(v) for v in q[sample]],
                                "q_norm2": float(np.sqrt(O.dot(q, q)))},
                 "policies": {}}
        for pname, kw in POLICIES.items():
            if pname in old:
                entry["policies"][pname] = old[pname]
                continue
            t1 = time.time()
            r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(**kw))
            entry["policies"][pname] = {
                "status": r.status, "iters": r.iters, "it_ur32": r.it_ur32, "it_uz32": r.it_uz32, "it_uz16": r.it_uz16,
                "relres_updated": r.relres_updated, "relres_true": r.relres_true,
                "fp16_subnormal_frac": (r.fp16_subnormal / r.fp16_stored) if r.fp16_stored else 0.0,
                "fp16_flushed_frac": (r.fp16_flushed / r.fp16_stored) if r.fp16_stored else 0.0,
                "oracle_seconds": round(time.time() - t1, 2), "threads": os.cpu_count(),
            }
            print(name, pname, entry["policies"][pname], flush=True)
        data[name] = entry
        json.dump(data, open(OUT, "w"), indent=1)


FORCE = "--force" in sys.argv

if __name__ == "__main__":
    main([a for a in sys.argv[1:] if not a.startswith("--")] or list(CONFIGS))
