"""Run-to-steady-state driver: the paper's production runs (Table 1: 1024 x 1024 points,
dt = 0.001, Re = 5 000 ... 30 000) stepped until RES_psi and RES_omega (eq 26-27) fall below the paper's tolerances
(1e-12 / 1e-10 for Re <= 20 000, 1e-10 / 1e-8 above), through the C ABI (cav_run_to_steady).

    python -m paper_0809_3098_b200.run_to_steady --Re 5000 [--points 1024] [--dt 0.001] [--sweeps 20] [--beta 1.97]
                                                 [--max-steps 3000000] [--check-every 1000] [--budget-s 1100] [--report-every 50]
                                                 [--sweep redblack|compact9]

The paper states neither its sweep count nor its stopping rule for the inner iteration (D3); S and beta here are this build's.
Prints one JSON line per report and a final summary line.  GPU only: there is no CPU fallback.
"""
import argparse
import json
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--Re", type=float, default=5000.0)
    ap.add_argument("--points", type=int, default=1024, help="grid points per side (the paper: 1024)")
    ap.add_argument("--dt", type=float, default=0.001)
    ap.add_argument("--sweeps", type=int, default=20)
    ap.add_argument("--beta", type=float, default=1.97)
    ap.add_argument("--max-steps", type=int, default=3000000)
    ap.add_argument("--check-every", type=int, default=1000)
    ap.add_argument("--budget-s", type=float, default=1100.0, help="stop after this much wall time even if not converged")
    ap.add_argument("--report-every", type=int, default=50, help="print every this many checks")
    ap.add_argument("--sweep", default="redblack", choices=["redblack", "compact9"],
                    help="Poisson operator / sweep: the 5-point red-black SOR of BASELINE.json, or the paper's own compact 9-point operator")
    args = ap.parse_args()
    from . import binding
    N = args.points - 1
    tol_psi, tol_w = (1e-12, 1e-10) if args.Re <= 20000 else (1e-10, 1e-8)
    cav = binding.Cavity(N, args.Re, args.dt, args.beta, args.sweeps)
    if args.sweep != "redblack":
        cav.set_sweep(args.sweep)
    cav.set_fields(None, np.zeros((N + 1, N + 1)))                               # fluid at rest, impulsive lid start (G11)
    print(json.dumps({"plan": cav.describe(), "Re": args.Re, "points": args.points, "dt": args.dt, "S": args.sweeps,
                      "beta": args.beta, "sweep": args.sweep, "tol": [tol_psi, tol_w]}), flush=True)
    t0 = time.perf_counter()
    steps, nchk, m = 0, 0, None
    chunk = args.check_every * args.report_every
    while steps < args.max_steps and time.perf_counter() - t0 < args.budget_s:
        m = cav.run_to_steady(min(chunk, args.max_steps - steps), args.check_every, tol_psi, tol_w)
        steps += m["steps"]
        nchk += 1
        d = cav.diag()
        psi, _ = cav.get_fields()
        print(json.dumps({"steps": steps, "t": steps * args.dt, "wall_s": round(time.perf_counter() - t0, 1),
                          "res_psi": m["res_psi"], "res_omega": m["res_omega"], "psi_min": float(psi.min()),
                          "kinetic_energy": d["kinetic_energy"], "res_inf": d["res_inf"], "converged": m["converged"]}), flush=True)
        if m["converged"] or not np.isfinite(m["res_psi"]):
            break
    wall = time.perf_counter() - t0
    print(json.dumps({"summary": True, "Re": args.Re, "steps": steps, "wall_s": round(wall, 1), "ms_per_step": 1e3 * wall / max(steps, 1),
                      "converged": bool(m and m["converged"]), "res_psi": m and m["res_psi"], "res_omega": m and m["res_omega"],
                      "tol_psi": tol_psi, "tol_omega": tol_w}), flush=True)
    cav.close()


if __name__ == "__main__":
    main()
