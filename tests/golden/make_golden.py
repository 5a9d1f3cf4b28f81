"""Writes tests/golden/cfgK.json: values of the CPU ORACLE (plain mode) on BASELINE.json config K.

Calls only oracle/ and the seeded input generator (paper_0809_3098_b200/workloads.py, which holds
no arithmetic of the method).  Nothing here ever comes from the CUDA path.  Full-length configs 3-5
take 35-60 min of one core each; their outputs are stored so the GPU parity tests
can check the full-length runs at sampled points and through the diagnostics.

Usage:  python tests/golden/make_golden.py K [K ...]        (K in 1..5)

Stored per checkpoint (after `step` time steps; config 5 also has a checkpoint "poisson" after its
10 000 Poisson-only sweeps, reading G14): the a4 diagnostics, max|psi|, max|omega| over all points
and over interior points (the denominators of the G18 error norm), min psi, and psi / omega at the
sample points  (j, i) in SAMPLE x SAMPLE  (ring rows/columns included, so wall vorticity is sampled).
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_0809_3098_b200 import workloads as W  # noqa: E402

CHECKPOINTS = {1: [1, 10, 100, 200], 2: [1, 10, 100, 1000, 2000], 3: [1, 10, 100, 1000, 5000],
               4: [1, 10, 100, 1000], 5: [1, 10, 100, 1000]}


def sample_index(N):
    fr = [0, 1, 2, 3, N // 8, N // 4 - 1, N // 4, 3 * N // 8, N // 2 - 1, N // 2, N // 2 + 1, 5 * N // 8,
          3 * N // 4, 7 * N // 8, N - 3, N - 2, N - 1, N]
    return sorted(set(int(v) for v in fr if 0 <= v <= N))


def snapshot(o, N, label):
    psi, w = o.get_fields()
    d = o.diag()
    s = sample_index(N)
    I = (slice(1, N), slice(1, N))
    return {
        "label": label, "step": int(d["step"]), "t": d["t"],
        "res_inf": d["res_inf"], "res_l2": d["res_l2"],
        "kinetic_energy": d["kinetic_energy"], "enstrophy": d["enstrophy"],
        "psi_absmax": float(np.max(np.abs(psi))), "omega_absmax": float(np.max(np.abs(w))),
        "omega_absmax_interior": float(np.max(np.abs(w[I]))), "psi_min": float(np.min(psi)),
        "sample_index": s,
        "psi": [[float(psi[j, i]) for i in s] for j in s],
        "omega": [[float(w[j, i]) for i in s] for j in s],
    }


def run(k):
    wl = W.config(k)
    t0 = time.time()
    o = oracle.OracleCavity(wl.N, wl.Re, wl.dt, wl.sor_omega, wl.sweeps_per_stage, oracle.MODE_PLAIN)
    o.set_fields(*W.initial_fields(wl))
    out = {"config": k, "name": wl.name, "N": wl.N, "Re": wl.Re, "dt": wl.dt, "sor_omega": wl.sor_omega,
           "sweeps_per_stage": wl.sweeps_per_stage, "seed": wl.seed, "noise": wl.noise,
           "smooth_amp": wl.smooth_amp, "poisson_sweeps": wl.poisson_sweeps,
           "written_by": "tests/golden/make_golden.py (oracle/cavity_oracle.cpp, ORC_MODE_PLAIN)",
           "checkpoints": []}
    if wl.poisson_sweeps:
        o.poisson(wl.poisson_sweeps)
        out["checkpoints"].append(snapshot(o, wl.N, "poisson"))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg%d.json" % k)

    def write():
        # rewritten after every checkpoint: an interrupted run leaves a valid file with the checkpoints reached so far
        out["oracle_wall_seconds"] = round(time.time() - t0, 1)
        with open(path + ".tmp.%d" % os.getpid(), "w") as f:
            json.dump(out, f, indent=1)
        os.replace(path + ".tmp.%d" % os.getpid(), path)

    done = 0
    for cp in CHECKPOINTS[k]:
        o.step(cp - done)
        done = cp
        out["checkpoints"].append(snapshot(o, wl.N, "step%d" % cp))
        print("cfg%d step %d  %.1f s" % (k, cp, time.time() - t0), flush=True)
        write()
    print("wrote", path)


if __name__ == "__main__":
    for a in sys.argv[1:]:
        run(int(a))
