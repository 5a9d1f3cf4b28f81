#!/usr/bin/env python
"""bench.py — throughput of the fp64 SSPRK(5,4) cavity step (arXiv 0809.3098) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

A "step" is one pass of the whole hot path over the workload: one SSPRK(5,4) time step = 5 x [S red-black SOR
sweeps (a1), Thom wall vorticity (a2), transport RHS + stage combination (a3)] on the (N+1)^2 grid.
The workload is BASELINE.json configs[3] (1025 x 1025, Re 10 000, S = 200, beta = 1.995): the one the metric's
target is quoted on.  Metric: fp64 grid-point-stage updates per second, GPSU/s = 5 (N+1)^2 steps / time
(Poisson sweeps included).

One JSON line on stdout (rank 0).  Keys beyond the base contract:
  roofline      the dominant kernel (k_resident: one launch = one whole time step), bound "alu": the path is bound by the fp64
                pipe, not by HBM (with the sweeps fused the working set stays on chip).
                achieved = algorithmic fp64 instructions per launch (5 per point-sweep + 30 per point-stage)
                / the launch's CUDA-event duration; peak = the DFMA-chain rate MEASURED in the same run
                (cav_measure_fp64_peak), the nominal 148 SMs x 64 lanes x clock beside it; traffic = DRAM bytes per launch from
                the ncu capture in profiles/, with the DRAM GB/s that follows.  `sweeps_only` repeats it for a1 alone
                (cav_poisson launches), `hbm_streaming_equiv` keeps BASELINE's "% of HBM bandwidth" reading as a secondary,
                clearly labelled figure (bytes a one-pass-per-sweep kernel would move; this kernel does not move them).
  other_configs / poisson_only   configs 1, 2, 3, 5 with bounded step counts, and the 10 000-sweep Poisson-only run of config 5.
  cpu_baseline  the oracle (oracle/, single thread, as it stands) timed on this box on a bounded sample.
  e2e           the same metric through the C ABI with HOST buffers every step (cav_set_fields from pinned
                memory -> cav_step(1) -> cav_get_fields), copies inside the timed region.

--impl reference times the CPU oracle instead (there is no reference implementation of the paper).
N > 1: replicas only (one independent context per GPU, no data-path collective).  Launched by
torchrun (RANK / WORLD_SIZE in the environment) or bare: `python bench.py --gpus N` then spawns the N ranks itself.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 grid-point-stage updates/s (incl. Poisson sweeps)"
UNIT = "GPSU/s"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
SM_COUNT, FP64_LANES_PER_SM = 148, 64   # B200: 148 SMs x 64 fp64 lanes
FP64_INSTR_PER_POINT_SWEEP = 5     # 3 DADD + 2 DFMA
FP64_INSTR_PER_POINT_STAGE = 30    # a2 + a3 ("5 S + 30 fp64 instructions per grid-point-stage")
# dram__bytes_read.sum + dram__bytes_write.sum of ONE k_resident launch (one time step of config 4) from the ncu --set full
# capture summarised in profiles/ (cold L2 under ncu).  The figure belongs to ONE build: it is reported only while the kernel's
# sources still have the git blob ids the capture was taken on; after any change to them the line says traffic: null and why.
NCU_DRAM_BYTES_PER_STEP_LAUNCH = 46.44e6
NCU_DRAM_SOURCE = "profiles/r3_final.md (ncu --set full, one launch = one time step of config 4: 19.69 MB read + 26.75 MB written)"
# (cavity_resident.cu was captured as blob 483d2b76; the later blob 11118681 differs only in the compact-operator instances, KIND == 1:
#  the SASS of the timed instance k_resident<4,6,16,false,0> is instruction for instruction the same, profiles/r3_sass.md)
NCU_DRAM_BUILD = {"paper_0809_3098_b200/csrc/cavity_resident.cu": "11118681061ee6e44afb35f324e9f81df19fc72e",
                  "paper_0809_3098_b200/csrc/cavity_scheme.cuh": "2dc6c4f7694d00fc9620b710a2bde93d8820fc00"}


def ncu_capture_is_current():
    """True if the kernel sources are byte for byte those of the ncu capture (git blob id = sha1("blob <len>\\0" + content))."""
    import hashlib
    for rel, want in NCU_DRAM_BUILD.items():
        try:
            data = open(os.path.join(ROOT, rel), "rb").read()
        except OSError:
            return False
        if hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest() != want:
            return False
    return True


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config 1..5 (default 4, the metric's)")
    ap.add_argument("--engine", default="auto", choices=["auto", "stream", "resident"])
    ap.add_argument("--sweep", default="redblack", choices=["redblack", "jacobi", "compact9"],
                    help="a1 variant (default: the red-black sweeps the metric is quoted on; compact9 = the paper's own operator, NEXT-1)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the other configs and the Poisson-only run")
    return ap.parse_args()


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(p.get("sm_max_mhz", 1965.0))
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------------
# the CPU oracle, timed (cpu_baseline leg and --impl reference)
# ----------------------------------------------------------------------------------------------------------

def oracle_sample_rate(wl, seconds_budget, nsamples=None):
    """Times the oracle as it stands (single thread) on whole time steps of `wl`; returns (GPSU/s, description)."""
    import oracle
    from paper_0809_3098_b200 import workloads as W
    o = oracle.OracleCavity(wl.N, wl.Re, wl.dt, wl.sor_omega, wl.sweeps_per_stage, oracle.MODE_PLAIN)
    o.set_fields(*W.initial_fields(wl))
    G = (wl.N + 1) ** 2
    t0 = time.perf_counter()
    o.step(1)
    t1 = time.perf_counter() - t0
    n = nsamples if nsamples is not None else max(1, min(20, int(seconds_budget / max(t1, 1e-9)) - 1))
    t0 = time.perf_counter()
    o.step(n)
    dt = time.perf_counter() - t0
    o.close()
    return 5.0 * G * n / dt, "%d SSPRK(5,4) time steps of %s (after 1 untimed), %.1f s of one core" % (n, wl.name, dt)


def run_reference(args, wl):
    """--impl reference: the oracle on the host cores.  Each 'step' is a bounded sample of the workload: one whole
    time step when K + W of them fit in ~170 s, else one RK-stage-equivalent (S sweeps + Thom via orc_poisson, then
    the transport operator via orc_rhs) = (N+1)^2 grid-point-stage updates."""
    import numpy as np
    import oracle
    from paper_0809_3098_b200 import workloads as W
    K = args.steps if args.steps is not None else 20
    Wm = args.warmup if args.warmup is not None else 3
    G = (wl.N + 1) ** 2
    o = oracle.OracleCavity(wl.N, wl.Re, wl.dt, wl.sor_omega, wl.sweeps_per_stage, oracle.MODE_PLAIN)
    o.set_fields(*W.initial_fields(wl))
    t0 = time.perf_counter()
    o.poisson(wl.sweeps_per_stage)
    psi, w = o.get_fields()
    oracle.rhs(wl.N, wl.Re, psi, w)
    t_stage = time.perf_counter() - t0
    full = (K + Wm) * 5.0 * t_stage <= 170.0
    units = 5.0 * G if full else 1.0 * G

    def one():
        if full:
            o.step(1)
        else:
            o.poisson(wl.sweeps_per_stage)
            p, ww = o.get_fields()
            oracle.rhs(wl.N, wl.Re, p, ww)

    for _ in range(Wm):
        one()
    t0 = time.perf_counter()
    for _ in range(K):
        one()
    dt = time.perf_counter() - t0
    o.close()
    value = units * K / dt
    sample = ("one whole SSPRK(5,4) time step of %s per step" % wl.name) if full else \
             ("one RK-stage-equivalent of %s per step (S=%d sweeps + Thom + transport operator = (N+1)^2 GPSU)"
              % (wl.name, wl.sweeps_per_stage))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": Wm, "ms_per_step": 1e3 * dt / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "grid": "%dx%d" % (wl.N + 1, wl.N + 1), "Re": wl.Re,
                       "sweeps_per_stage": wl.sweeps_per_stage, "sor_omega": wl.sor_omega, "dt": wl.dt,
                       "note": "no reference implementation of the paper exists; this arm is the CPU oracle"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------------

def run_ours(args, wl, rank, world, local_rank):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_0809_3098_b200 import binding, replicas
    from paper_0809_3098_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    use_dist = world > 1
    if use_dist:
        dist.init_process_group("nccl", device_id=dev)
    K = args.steps if args.steps is not None else 200
    Wm = args.warmup if args.warmup is not None else 5
    Wm = max(Wm, 3)

    wl = replicas.replica_workload(wl, rank, world)
    G = (wl.N + 1) ** 2
    P = (wl.N - 1) ** 2
    S = wl.sweeps_per_stage
    beta = wl.sor_omega if args.sweep == "redblack" else min(wl.sor_omega, 0.8)
    cav = binding.Cavity(wl.N, wl.Re, wl.dt, beta, S, engine=args.engine)
    if args.sweep != "redblack":
        cav.set_sweep(args.sweep)          # beta <= 1: the paper's under-relaxed range for its operator; the work per sweep does not depend on it
    psi0, w0 = W.initial_fields(wl)
    cav.set_fields(psi0, w0)
    if wl.poisson_sweeps:
        cav.poisson(wl.poisson_sweeps, want_residual=False)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)       # > 126 MB of L2

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps, L2 flushed (untimed) before each, CUDA events on the launch stream ----
    for _ in range(Wm):
        cav.step_async(1)
    barrier()
    sampler = ClockSampler(local_rank)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    l0 = cav.launch_count()
    barrier()
    for k in range(K):
        flush.fill_(k & 0xFF)
        ev[k][0].record()
        cav.step_async(1)
        ev[k][1].record()
    barrier()
    launches = cav.launch_count() - l0
    clocks = sampler.stop()
    per_step_ms = [a.elapsed_time(b) for a, b in ev]
    t_local = sum(per_step_ms) * 1e-3
    units_total, t_max = replicas.combine(5.0 * G * K, t_local, world, dist if use_dist else None, dev)
    value = units_total / t_max

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        hp = torch.empty((wl.N + 1, wl.N + 1), dtype=torch.float64).pin_memory()
        hw = torch.empty((wl.N + 1, wl.N + 1), dtype=torch.float64).pin_memory()
        hp_n, hw_n = hp.numpy(), hw.numpy()
        cav.get_fields(hp_n, hw_n)
        Ke = K
        for _ in range(3):
            cav.set_fields(hp_n, hw_n); cav.step(1); cav.get_fields(hp_n, hw_n)
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            cav.set_fields(hp_n, hw_n)          # H2D: psi and omega
            cav.step(1)
            cav.get_fields(hp_n, hw_n)          # D2H: psi and omega (the step's result)
        torch.cuda.synchronize()
        te = time.perf_counter() - t0
        ue, tmax_e = replicas.combine(5.0 * G * Ke, te, world, dist if use_dist else None, dev)
        e2e = {"value": ue / tmax_e, "unit": UNIT, "h2d_bytes_per_step": 2 * G * 8, "d2h_bytes_per_step": 2 * G * 8,
               "ms_per_step": 1e3 * tmax_e / Ke, "api": "cav_set_fields(host) -> cav_step(1) -> cav_get_fields(host)"}

    # ---- roofline of the dominant kernel, measured live.  k_resident runs a whole time step per launch: the per-step CUDA
    # events above ARE its launch durations.  Bound: the fp64 pipe; peak: a DFMA-chain kernel timed now.
    hbm_gbs, peak_src, sm_max_mhz = measured_peaks()
    desc = cav.describe()
    resident = "engine resident" in desc
    dfma_peak, nominal_mhz = cav.measure_fp64_peak()
    fp64_nominal = SM_COUNT * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    launches_per_step = launches / float(K)
    ips = 9 if args.sweep == "compact9" else FP64_INSTR_PER_POINT_SWEEP      # compact operator: 6 DADD + 3 DFMA per point-sweep
    instr_per_step = 5.0 * P * (ips * S + FP64_INSTR_PER_POINT_STAGE)
    step_s = statistics.mean(per_step_ms) * 1e-3
    achieved = instr_per_step / step_s
    # a1 alone: sweep-only launches of the step's own shape (S sweeps), timed by the library's events around the a1 launch
    extra = 2 if not resident else 1                # cav_poisson also launches Thom (and, streaming engine, the q scaling)
    for _ in range(3):
        cav.poisson(S, want_residual=False)
    reps, tsw, lsw = 25, 0.0, 0
    for k in range(reps):
        if k % 5 == 0:
            flush.fill_(1)
        l1 = cav.launch_count()
        cav.poisson(S, want_residual=False)
        tsw += cav.last_elapsed_ms() * 1e-3
        lsw += cav.launch_count() - l1 - extra
    sweep_rate = ips * P * S * reps / tsw
    current = ncu_capture_is_current()
    traffic = NCU_DRAM_BYTES_PER_STEP_LAUNCH if (wl.N == 1024 and S == 200 and resident and current) else None
    roofline = {"bound": "alu", "achieved": achieved / 1e12, "peak": dfma_peak / 1e12, "unit": "T fp64 instr/s",
                "frac": achieved / dfma_peak, "traffic": traffic,
                "traffic_source": NCU_DRAM_SOURCE if traffic else (None if current else "null: the kernel sources changed since the ncu capture of "
                                                                   + NCU_DRAM_SOURCE.split(" ")[0] + "; re-capture and update NCU_DRAM_* in bench.py"),
                "dram_GBps": (traffic / step_s / 1e9) if traffic else None,
                "peak_source": "measured in this run: DFMA-chain kernel, 16 warps per SM, 8 chains per thread (cav_measure_fp64_peak)",
                "peak_nominal": fp64_nominal / 1e12, "peak_nominal_model": "148 SMs x 64 fp64 lanes x sm_max_mhz",
                "frac_of_nominal": achieved / fp64_nominal,
                "kernel": ("k_resident, one launch per time step; " if resident else "") + desc,
                "instr_model": "5 fp64 instr per point-sweep (3 DADD + 2 DFMA) + 30 per grid-point-stage (a2 + a3), interior points, "
                               "useful work only (the redundant halo work of temporal blocking is not counted)",
                "algorithmic_instr_per_launch": instr_per_step / launches_per_step, "avg_launch_us": 1e6 * step_s / launches_per_step,
                "launches_per_step": launches_per_step,
                "sweeps_only": {"achieved": sweep_rate / 1e12, "frac": sweep_rate / dfma_peak, "avg_call_us": 1e6 * tsw / reps,
                                "launches_per_call": lsw / reps, "us_per_sweep": 1e6 * tsw / reps / S,
                                "share_of_step": 5.0 * (tsw / reps) / step_s,
                                "note": "S sweeps of a1 alone per cav_poisson call, timed by the library's CUDA events"}}
    b0 = 24.0 * S + 33.6
    hbm_equiv = value / max(world, 1) * b0 / 1e9

    # ---- the other configs (bounded step counts) and the Poisson-only run of config 5 (BASELINE.json configs[4]) ----
    others, poisson_only = None, None
    if rank == 0 and world == 1 and not args.no_others and args.sweep == "redblack":
        cav.close()
        others = {}
        for kcfg in (1, 2, 3, 5):
            if kcfg == args.config:
                continue
            w2 = W.config(kcfg)
            c2 = binding.Cavity(w2.N, w2.Re, w2.dt, w2.sor_omega, w2.sweeps_per_stage, engine=args.engine)
            c2.set_fields(*W.initial_fields(w2))
            if w2.poisson_sweeps:
                # the Poisson-only sweep-throughput run: 10 000 sweeps on the restart field, timed by the library's events
                c2.poisson(200, want_residual=False)
                c2.set_fields(*W.initial_fields(w2))
                c2.poisson(w2.poisson_sweeps, want_residual=False)
                tp = c2.last_elapsed_ms() * 1e-3
                poisson_only = {"workload": w2.name, "sweeps": w2.poisson_sweeps, "seconds": tp,
                                "point_sweeps_per_s": (w2.N - 1) ** 2 * w2.poisson_sweeps / tp,
                                "us_per_sweep": 1e6 * tp / w2.poisson_sweeps,
                                "residual_inf_after": c2.diag()["res_inf"]}
            nst = {1: 400, 2: 200, 3: 100, 5: 50}[kcfg]
            c2.step(5)
            ts = []
            for _ in range(3):
                c2.step(nst)
                ts.append(c2.last_elapsed_ms() * 1e-3 / nst)
            t1 = min(ts)
            others["cfg%d" % kcfg] = {"workload": w2.name, "ms_per_step": 1e3 * t1, "GPSU_per_s": 5.0 * (w2.N + 1) ** 2 / t1,
                                      "steps_timed": nst, "timing": "best of 3 cav_step(%d) calls, CUDA events of the library, "
                                      "device-resident, L2 not flushed (the working set is on chip)" % nst,
                                      "plan": c2.describe()}
            c2.close()
        # NEXT-1: the paper's own operator (4th-order compact 9-point, four-colour SOR) on the metric's config, resident engine
        w4 = W.config(args.config)
        c9 = binding.Cavity(w4.N, w4.Re, w4.dt, 0.8, w4.sweeps_per_stage, engine=args.engine)
        c9.set_sweep("compact9")
        c9.set_fields(*W.initial_fields(w4))
        c9.step(2)
        ts = []
        for _ in range(3):
            c9.step(10)
            ts.append(c9.last_elapsed_ms() * 1e-3 / 10)
        others["compact9_" + "cfg%d" % args.config] = {"workload": w4.name + ", compact 9-point operator (eq 14-21), beta 0.8", "ms_per_step": 1e3 * min(ts),
                                                       "GPSU_per_s": 5.0 * (w4.N + 1) ** 2 / min(ts), "ratio_to_5_point_path": min(ts) / step_s,
                                                       "steps_timed": 10, "plan": c9.describe()}
        c9.close()
        # NEXT-3: damped Jacobi (beta 0.9) on the metric's config: one kernel per sweep over global memory inside a CUDA graph of the
        # time step (every engine; the sweeps are not in the resident kernel), so that the line carries every sweep kind
        cj = binding.Cavity(w4.N, w4.Re, w4.dt, 0.9, w4.sweeps_per_stage, engine=args.engine)
        cj.set_sweep("jacobi")
        cj.set_fields(*W.initial_fields(w4))
        cj.step(2)
        ts = []
        for _ in range(3):
            cj.step(5)
            ts.append(cj.last_elapsed_ms() * 1e-3 / 5)
        others["jacobi_" + "cfg%d" % args.config] = {"workload": w4.name + ", damped Jacobi sweeps (G21), beta 0.9", "ms_per_step": 1e3 * min(ts),
                                                     "GPSU_per_s": 5.0 * (w4.N + 1) ** 2 / min(ts), "ratio_to_red_black_path": min(ts) / step_s,
                                                     "steps_timed": 5, "plan": "one k_jacobi_sweep launch per sweep over global memory (ping-pong fields), CUDA graph of one time step"}
        cj.close()
        # cav_diag_noalloc (the a4 reductions on caller-owned device buffers, no allocation): an HBM-bound kernel, timed alone on the
        # largest grid it takes (N = 8192: 2 fields x 537 MB, larger than L2), CUDA events on the launching stream
        nmax = binding.noalloc_max_n()
        gen = torch.Generator(device=dev).manual_seed(8192)
        pd = torch.randn((nmax + 1, nmax + 1), dtype=torch.float64, device=dev, generator=gen) * 0.05
        wd = torch.randn((nmax + 1, nmax + 1), dtype=torch.float64, device=dev, generator=gen) * 3.0
        o4 = torch.zeros(4, dtype=torch.float64, device=dev)
        st_ = torch.cuda.current_stream(dev)
        for _ in range(3):
            binding.diag_noalloc(nmax, pd, wd, o4, stream=st_.cuda_stream)
        ts = []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st_)
            binding.diag_noalloc(nmax, pd, wd, o4, stream=st_.cuda_stream)
            e1.record(st_)
            e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        nbytes = 2.0 * 8.0 * (nmax + 1) ** 2           # algorithmic bytes: psi and omega read once (16 B per grid point), 32 B written
        others["diag_noalloc_%d" % (nmax + 1)] = {"workload": "a4 diagnostics of a %d x %d state in caller-owned device buffers (cav_diag_noalloc)" % (nmax + 1, nmax + 1),
                                                  "ms_per_call": 1e3 * min(ts), "launches_per_call": 1, "bound": "hbm", "algorithmic_bytes": nbytes,
                                                  "achieved_GBps": nbytes / min(ts) / 1e9, "peak_GBps": hbm_gbs, "frac": nbytes / min(ts) / 1e9 / hbm_gbs,
                                                  "timing": "best of 5 calls, inputs larger than L2, includes the 256-byte counter clear"}
        del pd, wd, o4
    else:
        cav.close()

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": 1e3 * t_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"sweep": args.sweep, "workload": wl.name if world == 1 else W.config(args.config).name + " (rank 0) + Table-1 Re replicas",
                       "grid": "%dx%d" % (wl.N + 1, wl.N + 1), "Re": wl.Re, "sweeps_per_stage": S,
                       "sor_omega": beta, "dt": wl.dt, "parallelism": "replicas x%d" % world,
                       "l2": "flushed before every timed step (256 MiB write, outside the per-step CUDA events)",
                       "timing": "sum of per-step CUDA-event times on the launch stream, max over ranks"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "hbm_streaming_equiv": {"bytes_per_gpsu": b0, "GBps_per_gpu": hbm_equiv, "frac_of_measured_peak": hbm_equiv / hbm_gbs,
                                    "frac_of_8TBps_nominal": hbm_equiv / 8000.0,
                                    "note": "SECONDARY figure: bytes a one-pass-per-sweep streaming kernel would move (24 S + 33.6 per "
                                            "grid-point-stage, SURVEY S8(d) item 2) x the measured rate.  The resident kernel does "
                                            "NOT move them (see roofline.traffic): BASELINE's >= 0.70 HBM target does not apply to a "
                                            "temporally blocked kernel; the binding roofline is roofline (alu)"},
            "ms_per_step_min": min(per_step_ms), "ms_per_step_median": statistics.median(per_step_ms),
            "other_configs": others, "poisson_only": poisson_only}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, sample = oracle_sample_rate(W.config(args.config), 15.0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                                "host_cores": os.cpu_count()}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.destroy_process_group()


def run_stub(args, wl, rank, world):
    """CAV_BENCH_STUB=1 (tests only, CPU): the launch / rendezvous / combine logic of the N-rank path over gloo with a stubbed
    step (a sleep of 10 ms x (rank + 1)); prints a line of the same shape whose metric and unit say STUB and with `"stub": true`.
    No kernel runs: never a bench value.  Refused (exit 2) outside a pytest run, so a leaked environment variable cannot
    turn a driver run into a fake number."""
    if "PYTEST_CURRENT_TEST" not in os.environ:
        sys.stderr.write("bench.py: CAV_BENCH_STUB=1 is honoured only inside a pytest run; unset it\n")
        raise SystemExit(2)
    import torch
    import torch.distributed as dist
    from paper_0809_3098_b200 import replicas
    if world > 1:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = replicas.replica_workload(wl, rank, world)
    K = args.steps if args.steps is not None else 3
    t0 = time.perf_counter()
    for _ in range(K):
        time.sleep(0.01 * (rank + 1))
    t_local = time.perf_counter() - t0
    units, t_max = replicas.combine(5.0 * (wl.N + 1) ** 2 * K, t_local, world, dist if world > 1 else None, torch.device("cpu"))
    if rank == 0:
        print(json.dumps({"metric": "STUB: no kernel ran, not a measurement", "value": units / t_max, "unit": "stub units/s", "n_gpus": world, "steps": K, "stub": True,
                          "ms_per_step": 1e3 * t_max / K, "config": {"workload": wl.name}}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(n, argv):
    """`python bench.py --gpus N` without a launcher: re-executes this file as N ranks (RANK / LOCAL_RANK / WORLD_SIZE /
    MASTER_* in their environment), one per GPU; rank 0's JSON line is this process's output.  Returns the exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for r in range(n):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(n), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), BENCH_SPAWNED="1")
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + argv, env=env))
    rc = 0
    for pr in procs:
        rc = pr.wait() or rc
    return rc


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        raise SystemExit(spawn_ranks(args.gpus, sys.argv[1:]))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_0809_3098_b200 import workloads as W
    wl = W.config(args.config)
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, wl)
        return
    if os.environ.get("CAV_BENCH_STUB") == "1":
        run_stub(args, wl, rank, world)
        return
    run_ours(args, wl, rank, world, local_rank)


if __name__ == "__main__":
    main()
