#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path over one synthetic geometry:
node preparation + the operator's stored part (whole matrix of Eq. (3.16), leading block, or nothing) + restarted
GMRES with that operator, every stage of the config (config 4: 4 stages, the later ones through bie_build_update).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference] [--operator ...]

Prints ONE JSON line (rank 0).  Default workload: BASELINE.json configs[4] (n = 16384, restart 100, tol 1e-13), the
largest single-GPU configuration.

  value         whole-step throughput: n^2 matrix entries applied per second of a step, inputs resident in HBM
  build/gmres   the two halves of BASELINE.json's metric on their own: Gentries/s of bie_build (stand-alone calls,
                median and best of 20), ms of the solve inside the step
  per_config    configs 1-4 with SURVEY 8(d)'s protocol: 3 warm-ups, median and best of 20 builds / 100 matvecs /
                10 solves per operator; config 4 as its 4-stage sequence
  e2e           the same step through bie_solve_host with pinned HOST buffers (H2D of nodes+rhs, D2H of the density)
  roofline      dominant kernel = the persistent GMRES kernel of the operator the step uses
  roofline_build  the entry builder against its two bounds (HBM write, FP64 pipe)
  cpu_baseline  the oracle (oracle/, as it stands) REALLY run on this box's host cores: oracle.build_matrix +
                oracle.gmres on the same inputs, all cores (and one thread where that takes seconds)

--impl reference times the oracle alone (this tier has no reference implementation).
N > 1: replicas only: every rank runs the same step on its own GPU, no data-path collective.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "matrix build Gentries/s and GMRES solve ms (FP64); % of FP64 / HBM roofline"
UNIT = "Gentries/s"
# FP64-pipe instructions per matrix entry (DFMA + DMUL + DADD), SASS counts from the ncu captures under profiles/
# (profiles/r02b_build.md, profiles/r02_free.md); the hand counts of DESIGN.md section 5 are 10 / 10 / 6.5 + reduction
FP64_PER_ENTRY_BUILD = 10.1     # bie_build_kernel, difference form
FP64_PER_ENTRY_SYM = 6.92       # symmetric pair loops: 13 per pair of entries + lane reduction of the reverse sums
FP64_PER_ENTRY_VORTEX_BUILD = 11.0   # vortex-sheet / normal-velocity builds: row-side difference form (bie_build.cu)
FP64_PER_PAIR_VORTEX = 13.0     # vortex-sheet matrix in the matrix-free operator, (X, Y) form
NOMINAL_FP64_INSTR_S = 148 * 64 * 1.965e9   # B200: 148 SMs x 64 FP64 lanes x 1.965 GHz = 18.6 T instr/s
HBM_FALLBACK_GBS = 6650.0      # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")   # dram bytes per launch from `ncu --set full`


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--operator", default="auto", choices=["auto", "dense", "free", "hybrid"],
                    help="dense: bie_build + GMRES on the stored matrix; free: matrix-free GMRES (entries recomputed on the "
                         "fly, no matrix); hybrid: the leading block of bie_hybrid_cols(n) rows and columns stored and streamed "
                         "while everything else is recomputed; auto (default): all are timed during warm-up and the fastest is the timed step")
    ap.add_argument("--matrix-free", action="store_true", help="same as --operator free")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (configs 1-4)")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the stand-alone timings of the SURVEY 8(f) rows")
    ap.add_argument("--cpu-seconds", type=float, default=150.0, help="wall budget of the whole --impl reference run")
    a = ap.parse_args()
    if a.matrix_free:
        a.operator = "free"
    return a


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, a read+write copy)"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def n_gemv(iters: int, restart: int) -> int:
    """operator applications of one bie_gmres launch: one per Arnoldi step, one residual per restart, one final true residual"""
    cycles = max(1, -(-iters // restart))
    return iters + (cycles - 1) + 1


def traffic_bytes(config: int, op: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of the GMRES kernel of (config, operator), one launch, from the committed
    `ncu --set full` capture of THIS code state (profiles/r02_dram_traffic.csv names the commit); None when not captured"""
    try:
        for row in csv.DictReader(open(TRAFFIC_CSV)):
            if int(row["config"]) == config and row["operator"] == op:
                return {"bytes": float(row["dram_bytes"]), "capture": row.get("capture", ""), "code_state": row.get("code_state", "")}
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------------------
# clocks during the timed region
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
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
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [t.strip() for t in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        hi = [s for s, p in zip(sm, pw) if p >= 0.5 * max(pw)] or sm  # samples under load
        return {"sm_mhz": float(np.median(hi)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------
# oracle legs (the only places bench.py executes oracle/)
# ---------------------------------------------------------------------------------------------------
def oracle_step(P, threads=None):
    """ONE real pass of the oracle over the workload, as it stands: oracle.build_matrix + oracle.gmres for every stage.
    -> dict with the measured seconds.  threads: None = all cores."""
    import oracle
    allc = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    try:
        tb = tg = 0.0
        its = []
        A = None
        rr = 0.0
        for g, b in zip(P.stages, P.rhs):
            t0 = time.perf_counter()
            A = oracle.build_matrix(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, out=A)
            t1 = time.perf_counter()
            x, it, rr, hist, st = oracle.gmres(A, b, P.tol, P.restart, P.max_iters)
            t2 = time.perf_counter()
            tb += t1 - t0; tg += t2 - t1; its.append(int(it))
        return {"build_s": tb, "gmres_s": tg, "step_s": tb + tg, "iters": its, "relres_true": float(rr),
                "threads": int(threads or allc)}
    finally:
        if threads:
            oracle.set_num_threads(allc)


def oracle_bounded_step(P, budget_s, build_s_per_entry, iters):
    """A bounded sample of one step for machines where the full oracle step does not fit the budget: the build on R of the n
    rows and the GEMV on that block, scaled to the whole step.  -> (estimated step seconds, description)"""
    import oracle
    g = P.geometry
    n = g.n
    rng = np.random.default_rng(0)
    R = int(min(n, max(64, n * min(1.0, 0.25 * budget_s / max(build_s_per_entry * n * n, 1e-9)))))
    rows = np.sort(rng.choice(n, size=R, replace=False))
    t0 = time.perf_counter()
    blk = oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, rows)
    t_build = (time.perf_counter() - t0) * n / R
    x = rng.standard_normal(n)
    reps, t0 = 0, time.perf_counter()
    while True:
        oracle.matvec(blk, x); reps += 1
        if time.perf_counter() - t0 > 0.5 * budget_s or reps >= 100:
            break
    t_gemv = (time.perf_counter() - t0) / reps * n / R
    ng = n_gemv(iters, P.restart)
    t_gs = ng * 0.5 * min(iters, P.restart) * 4 * 8 * n / 2.0e10      # modified Gram-Schmidt: 4 n j flops per step, memory-bound, ~20 GB/s
    est = len(P.stages) * (t_build + ng * t_gemv + t_gs)
    return est, (f"ESTIMATED (the full oracle step does not fit {budget_s:.1f} s here): oracle.build_rows on {R} of {n} rows, {reps} "
                 f"oracle GEMVs on that block; step = stages * (n/R build + {ng} GEMVs * n/R block GEMV + Gram-Schmidt 2 n j^2 flops)")


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, same config/metric/unit (rank 0 only).  Every step is ONE real
    oracle pass (build_matrix + gmres, all stages) when that fits the run's wall budget, else a bounded sample marked estimated."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_2108_01786_b200 import inputs
    P = inputs.make_config(args.config)
    n = P.n
    args.op, args.nd = "dense", 0     # the oracle stores the matrix
    nsteps = max(1, args.steps + args.warmup)
    per = args.cpu_seconds / nsteps
    first = oracle_step(P)                      # one real pass tells whether the rest fit
    full = first["step_s"] <= per
    times, parts, desc = [], first, None
    for k in range(1, nsteps):
        if full:
            r = oracle_step(P)
            if k >= args.warmup:
                times.append(r["step_s"]); parts = r
        else:
            est, desc = oracle_bounded_step(P, per, first["build_s"] / len(P.stages) / (n * n), first["iters"][-1])
            if k >= args.warmup:
                times.append(est)
    if not times:
        times = [first["step_s"]]
    step_s = float(np.mean(times))
    val = len(P.stages) * n * n / step_s / 1e9
    cores = oracle.num_threads()
    sample = (f"every step = one REAL oracle pass (oracle.build_matrix + oracle.gmres on all {len(P.stages)} stage(s)), "
              f"{cores} threads" if full else desc)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_s * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "estimated": (not full),
            "config": workload_config(P, args, first["iters"][-1]),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "estimated": (not full)},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "build": {"gentries_per_s": len(P.stages) * n * n / parts["build_s"] / 1e9, "ms": parts["build_s"] * 1e3},
            "gmres": {"ms": parts["gmres_s"] * 1e3, "iters": parts["iters"][-1], "relres_true": parts["relres_true"]}}
    print(json.dumps(line), flush=True)


def l2_policy(n, stored):
    """what the timed iterations stream: the stored part of the matrix (entries) against the 126 MB L2"""
    nbytes = 8.0 * stored
    if stored == 0:
        return ("no matrix stored (matrix-free operator): the O(n) node tables are L2-resident by design, the kernel is "
                "FP64-bound; nothing to flush")
    if nbytes > 2.5e8:
        return "stored part of the matrix (%.0f MB) is %.1fx the 126 MB L2: every operator application streams it from HBM; no flush needed" % (nbytes / 1e6, nbytes / 126e6)
    return "stored part of the matrix (%.0f MB) fits the 126 MB L2: L2-resident, reported as such (not as HBM bandwidth)" % (nbytes / 1e6)


def stored_entries(n, op, nd):
    return {"dense": n * n, "free": 0, "hybrid": nd * nd}[op]


def workload_config(P, args, iters):
    g = P.geometry
    se = stored_entries(g.n, args.op, getattr(args, "nd", 0))
    return {"workload": f"BASELINE.json configs[{P.config - 1}]: {P.name}", "n": int(g.n),
            "counts": [int(c) for c in g.counts], "restart": int(P.restart), "tol": P.tol,
            "operator": {"dense": "dense (whole matrix stored)", "free": "matrix-free (symmetric pair loops)",
                         "hybrid": "hybrid (stored leading block + recomputed rest)"}[args.op]
                        + (" (chosen by measurement)" if args.operator == "auto" else ""),
            "matrix_bytes": int(8 * se), "stored_entries": int(se),
            "l2_policy": l2_policy(g.n, se),
            "stages_per_step": len(P.stages), "replicas": int(args.gpus)}


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
class Timer:
    """SURVEY 8(d) protocol: warm-ups, then every repetition timed on the device with its own pair of CUDA events (on the
    current stream, which is the stream the binding launches on); optional L2 flush between repetitions."""

    def __init__(self, torch):
        self.torch = torch
        self.flush_buf = None

    def flush(self):
        if self.flush_buf is None:
            self.flush_buf = self.torch.empty(256 << 20, dtype=self.torch.uint8, device="cuda")   # 2x the 126 MB L2
        self.flush_buf.zero_()

    def __call__(self, fn, reps, warm=3, flush=False):
        t = self.torch
        for _ in range(warm):
            fn()
        t.cuda.synchronize()
        ms = []
        for _ in range(reps):
            if flush:
                self.flush()
            a, c = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
            a.record(); fn(); c.record()
            t.cuda.synchronize()
            ms.append(a.elapsed_time(c))
        return {"median_ms": float(np.median(ms)), "best_ms": float(np.min(ms)), "reps": reps}


class Workload:
    """one config on the device: buffers, the three operators' steps"""

    def __init__(self, torch, bie, ctx, P):
        self.torch, self.bie, self.ctx, self.P = torch, bie, ctx, P
        g, n = P.geometry, P.n
        self.g, self.n = g, n
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        self.stages = [(gs, tuple(dev(a) for a in (gs.zeta, gs.dzeta, gs.d2zeta)), dev(bs)) for gs, bs in zip(P.stages, P.rhs)]
        self.z, self.dz, self.d2z = self.stages[0][1]
        self.A = torch.empty((n, n + (n & 1)), dtype=torch.float64, device="cuda")
        self.x = torch.empty(n + (n & 1), dtype=torch.float64, device="cuda")[:n]
        self.ws = torch.empty(ctx.bie_gmres_workspace_bytes(n, P.restart), dtype=torch.uint8, device="cuda")
        self.oi = torch.zeros(2, dtype=torch.int32, device="cuda")
        self.of = torch.zeros(1, dtype=torch.float64, device="cuda")
        ctx.bie_set_geometry(g.counts, g.kinds, self.z, self.dz, self.d2z)
        self.nd = ctx.bie_hybrid_cols(n)
        self.blk = (torch.empty(max(ctx.bie_hybrid_block_bytes(self.nd) // 8, 2), dtype=torch.float64, device="cuda")
                    if self.nd else None)

    def step(self, op, ev=None):
        ctx, P = self.ctx, self.P
        for si, (gs, (zs, dzs, d2zs), bs) in enumerate(self.stages):
            if ev and si == 0: ev[0].record()
            if op == "dense":
                if si == 0:
                    ctx.bie_build(gs.counts, gs.kinds, zs, dzs, d2zs, self.A)      # 2 launches: node prep + tile kernel
                else:
                    ctx.bie_build_update(gs.counts, gs.kinds, zs, dzs, d2zs, self.A)   # only the blocks touching Gamma_0
            elif op == "free":
                ctx.bie_set_geometry(gs.counts, gs.kinds, zs, dzs, d2zs)      # 1 launch: node prep
            else:
                ctx.bie_build_block(gs.counts, gs.kinds, zs, dzs, d2zs, self.nd, self.blk)   # 2 launches: node prep + block tiles
            if ev and si == 0: ev[1].record()
            if op == "hybrid":       # near matrix (3 launches, once per geometry) + 1 cooperative launch
                ctx.bie_gmres_hybrid(self.blk, self.nd, bs, self.x, P.tol, P.restart, P.max_iters, self.ws, self.oi, self.of)
            else:                    # dense: 1 cooperative launch; matrix-free: near matrix (3) + (symmetric work list 1) + 1
                ctx.bie_gmres(self.A if op == "dense" else None, bs, self.x, P.tol, P.restart, P.max_iters, self.ws, self.oi, self.of)
        if ev: ev[2].record()

    def ops(self):
        return ["dense", "free"] + (["hybrid"] if self.nd else [])

    def result(self):
        return int(self.oi[0]), int(self.oi[1]), float(self.of[0])


def gmres_roofline(n, op, nd, ng, gmres_ms, dfma_per_s, clocks_mhz, config):
    """roofline of the persistent GMRES kernel for one launch of ng operator applications taking gmres_ms"""
    peak, peak_src = hbm_peak()
    t = gmres_ms * 1e-3
    tr = traffic_bytes(config, op)
    if op == "dense":
        ach = ng * 8.0 * n * n / t / 1e9
        return {"bound": "hbm", "kernel": "bie_gmres_kernel<dense> (persistent; GEMV phases dominate)", "achieved": ach, "peak": peak,
                "unit": "GB/s", "frac": ach / peak, "traffic": tr and tr["bytes"], "traffic_capture": tr, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ng * 8 * n * n, "operator_applications_per_launch": ng}
    entries = ng * (n * n - (nd * nd if op == "hybrid" else 0))
    instr = entries * FP64_PER_ENTRY_SYM + (ng * nd * nd if op == "hybrid" else 0)     # + one DFMA per streamed block entry
    ach = instr / t
    alu = {"achieved": ach / 1e12, "unit": "T FP64 instr/s", "fp64_instr_per_entry": FP64_PER_ENTRY_SYM,
           "recomputed_entries_per_launch": entries, "peak_probe": dfma_per_s / 1e12, "frac_of_probe": ach / dfma_per_s,
           "peak_nominal": NOMINAL_FP64_INSTR_S / 1e12, "frac_of_nominal": ach / NOMINAL_FP64_INSTR_S,
           "sm_mhz_during_step": clocks_mhz,
           "peak_source": "bie_probe_dfma in this run; nominal = 148 SMs x 64 FP64 lanes x 1.965 GHz (DESIGN.md section 7)"}
    if op == "free":
        return {"bound": "alu", "kernel": "bie_gmres_kernel<matrix-free> (persistent; symmetric pair loops dominate)",
                "achieved": alu["achieved"], "peak": alu["peak_probe"], "unit": alu["unit"], "frac": alu["frac_of_probe"],
                "traffic": tr and tr["bytes"], "traffic_capture": tr, "operator_applications_per_launch": ng, "alu": alu}
    gbs = ng * 8.0 * nd * nd / t / 1e9
    hbm = {"achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "algorithmic_bytes_per_launch": ng * 8 * nd * nd,
           "peak_source": peak_src}
    binding = "hbm" if hbm["frac"] >= alu["frac_of_probe"] else "alu"
    return {"bound": "hbm+alu", "binding_leg": binding, "kernel": "bie_gmres_kernel<hybrid> (persistent; block stream and pair loops at once)",
            "achieved": hbm["achieved"] if binding == "hbm" else alu["achieved"],
            "peak": hbm["peak"] if binding == "hbm" else alu["peak_probe"],
            "unit": hbm["unit"] if binding == "hbm" else alu["unit"],
            "frac": max(hbm["frac"], alu["frac_of_probe"]), "traffic": tr and tr["bytes"], "traffic_capture": tr,
            "operator_applications_per_launch": ng, "hbm": hbm, "alu": alu}


def measure_config(torch, bie, ctx, c, timer, dfma_per_s):
    """per_config entry: build, matvec (dense, with L2 flush where the matrix is near the L2 size; matrix-free),
    and the step with every operator -- median and best of 20 / 100 / 10"""
    from paper_2108_01786_b200 import inputs
    P = inputs.make_config(c)
    W = Workload(torch, bie, ctx, P)
    g, n = W.g, W.n
    peak, _ = hbm_peak()
    out = {"n": n, "counts": [int(v) for v in g.counts], "restart": int(P.restart), "stages": len(P.stages)}
    b = timer(lambda: ctx.bie_build(g.counts, g.kinds, W.z, W.dz, W.d2z, W.A), 20)
    b.update({"gentries_per_s_median": n * n / (b["median_ms"] * 1e-3) / 1e9, "gentries_per_s_best": n * n / (b["best_ms"] * 1e-3) / 1e9,
              "hbm_write_frac": 8.0 * n * n / (b["median_ms"] * 1e-3) / 1e9 / peak,
              "fp64_frac_of_probe": n * n * FP64_PER_ENTRY_BUILD / (b["median_ms"] * 1e-3) / dfma_per_s,
              "fp64_frac_of_nominal": n * n * FP64_PER_ENTRY_BUILD / (b["median_ms"] * 1e-3) / NOMINAL_FP64_INSTR_S})
    out["build"] = b
    if len(P.stages) > 1:
        M0 = int(g.counts[0])
        u = timer(lambda: ctx.bie_build_update(g.counts, g.kinds, W.z, W.dz, W.d2z, W.A), 20)
        ue = n * n - (n - M0) * (n - M0)
        u.update({"entries": ue, "share_of_matrix": ue / float(n * n), "gentries_per_s_median": ue / (u["median_ms"] * 1e-3) / 1e9})
        out["build_update"] = u
    xv = torch.from_numpy(np.random.default_rng(1).standard_normal(n)).cuda()
    yv = torch.empty(n + (n & 1), dtype=torch.float64, device="cuda")[:n]
    nbytes = 8.0 * n * n
    flush = 0.4 * 126e6 < nbytes < 4 * 126e6       # near the L2 size: flush between repetitions, else the number is an L2 number
    mv = timer(lambda: ctx.bie_matvec(W.A, xv, yv), 100, flush=flush)
    mv.update({"gbs_median": nbytes / (mv["median_ms"] * 1e-3) / 1e9, "l2_flushed_between_reps": bool(flush),
               "regime": ("HBM (matrix %.0f MB, L2 flushed between repetitions)" % (nbytes / 1e6)) if flush else
                         ("L2-resident (matrix %.1f MB): an L2 / latency number, not HBM bandwidth" % (nbytes / 1e6) if nbytes < 126e6
                          else "HBM (matrix %.0f MB streams)" % (nbytes / 1e6)),
               "hbm_frac": (nbytes / (mv["median_ms"] * 1e-3) / 1e9 / peak) if nbytes >= 0.4 * 126e6 else None})
    out["matvec_dense"] = mv
    ctx.bie_set_geometry(g.counts, g.kinds, W.z, W.dz, W.d2z)
    mf = timer(lambda: ctx.bie_matvec_free(xv, yv), 100)
    mf.update({"gentries_per_s_median": n * n / (mf["median_ms"] * 1e-3) / 1e9,
               "fp64_frac_of_probe": n * n * FP64_PER_ENTRY_SYM / (mf["median_ms"] * 1e-3) / dfma_per_s})
    out["matvec_free"] = mf
    steps = {}
    for op in W.ops():
        r = timer(lambda: W.step(op), 10)
        it, st, rr = W.result()
        r.update({"iters_last_stage": it, "status": st, "relres_true": rr,
                  "us_per_iter_median": r["median_ms"] * 1e3 / max(1, it * len(P.stages))})
        steps[op] = r
    if n <= 1024 and "dense" in steps:
        # small stored-matrix solves run on one thread-block cluster when the rows of A fit its shared memory (bie_gmres_cluster.cu);
        # the grid-wide kernel on the same system, for comparison
        ctx.bie_set_small_gmres(0)
        r = timer(lambda: W.step("dense"), 10)
        ctx.bie_set_small_gmres(1)
        it, st, rr = W.result()
        r.update({"iters_last_stage": it, "status": st, "relres_true": rr,
                  "us_per_iter_median": r["median_ms"] * 1e3 / max(1, it * len(P.stages))})
        out["dense_grid_wide_kernel"] = r
        out["dense_solver_note"] = ("`dense` ran on one thread-block cluster when all but four rows of A per CTA fit the cluster's shared "
                                    "memory (n <= 640), else on the grid-wide kernel; `dense_grid_wide_kernel` is the latter, forced")
    best = min(steps, key=lambda k: steps[k]["median_ms"])
    out["step"] = steps
    out["operator_chosen"] = best
    it = steps[best]["iters_last_stage"]
    ng = n_gemv(it, P.restart) * len(P.stages)
    se = stored_entries(n, best, W.nd)
    out["l2_policy"] = l2_policy(n, se)
    rf = gmres_roofline(n, best, W.nd, ng, steps[best]["median_ms"], dfma_per_s, None, c)
    out["roofline"] = {k: rf[k] for k in ("bound", "achieved", "peak", "unit", "frac") if k in rf}
    if best == "dense" and 8.0 * n * n < 126e6:
        out["roofline"]["bound"] = "l2/latency"
        out["roofline"]["note"] = ("the matrix is L2-resident and the step is dominated by grid barriers: `achieved` is algorithmic bytes "
                                   "over the whole step, not an HBM statement")
    del W
    torch.cuda.empty_cache()
    return out


def cpu_baseline(cfgs):
    """the oracle really run (build_matrix + gmres, every stage) on all host cores for every config asked for, and on ONE thread
    where that takes seconds (configs 1-3)"""
    from paper_2108_01786_b200 import inputs
    out = {}
    for c in cfgs:
        P = inputs.make_config(c)
        n = P.n
        r = oracle_step(P)
        e = {"n": n, "cores": r["threads"], "build_s": r["build_s"], "gmres_s": r["gmres_s"], "step_s": r["step_s"], "iters": r["iters"],
             "gentries_per_s": len(P.stages) * n * n / r["step_s"] / 1e9, "build_gentries_per_s": len(P.stages) * n * n / r["build_s"] / 1e9,
             "estimated": False}
        if c <= 3:
            s1 = oracle_step(P, threads=1)
            e["single_thread"] = {"build_s": s1["build_s"], "gmres_s": s1["gmres_s"], "step_s": s1["step_s"]}
        else:
            e["single_thread"] = None    # minutes of CPU time: not run
        out[str(c)] = e
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    from paper_2108_01786_b200 import bie, inputs, ranks, build as _build

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: the CUDA path has no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    R = ranks.from_env("nccl")      # replicas only: NCCL serves the timing barrier and the max, nothing else
    rank, local, world = R.rank, R.local_rank, R.world
    if rank == 0:
        _build.build_library()
    ranks.barrier(R)

    def barrier():
        ranks.barrier(R, torch.cuda.synchronize)

    def max_over_ranks(v: float) -> float:
        return ranks.max_over_ranks(R, v)

    P = inputs.make_config(args.config)
    g, n = P.geometry, P.n
    ctx = bie.Context(local)
    timer = Timer(torch)
    W = Workload(torch, bie, ctx, P)
    nstage = len(P.stages)

    def time_steps(op, k):
        torch.cuda.synchronize()
        a_, c_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a_.record()
        for _ in range(k):
            W.step(op)
        c_.record(); torch.cuda.synchronize()
        return a_.elapsed_time(c_) / k

    # operator choice by measurement (north_star: "matrix-free fused rebuild+matvec variant chosen by measurement")
    choice_ms = {}
    op = args.operator
    if op == "hybrid" and W.nd == 0:
        raise SystemExit("bench: n is too small for the hybrid operator")
    if op == "auto":
        for name in W.ops():
            W.step(name)
            # best of three single steps: the two fastest operators are 2-3 % apart and a two-step mean picked the slower one in
            # one run of six
            choice_ms[name] = max_over_ranks(min(time_steps(name, 1) for _ in range(3)))
        op = min(choice_ms, key=choice_ms.get)
    args.op, args.nd = op, W.nd
    solve_mode = {"dense": 0, "free": 1, "hybrid": 2}[op]

    for _ in range(max(args.warmup, 3)):
        W.step(op)
    barrier()
    iters, status, relres = W.result()
    if status != 0 or not (relres <= 1e-12):
        raise SystemExit(f"bench: GMRES did not converge (status {status}, relres {relres})")

    # FP64 pipe rate of this GPU, now (roofline denominator of the FP64-bound kernels)
    probe_out = torch.zeros(1, dtype=torch.float64, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx.bie_probe_dfma(1 << 15, probe_out)
    torch.cuda.synchronize()
    e0.record(); total_fma = ctx.bie_probe_dfma(1 << 17, probe_out); e1.record()
    torch.cuda.synchronize()
    dfma_per_s = total_fma / (e0.elapsed_time(e1) * 1e-3)

    # ---- timed region: K steps, device time, max over ranks ------------------------------------------
    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    for k in range(K):
        W.step(op, evs[k])
    t_end.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(t_start.elapsed_time(t_end))
    prep_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    gmres_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    ms_per_step = total_ms / K
    value = world * nstage * n * n / (ms_per_step * 1e-3) / 1e9

    # ---- stand-alone calls (outside the timed region; median and best of 20 / 100) -----------------
    peak, peak_src = hbm_peak()
    xv = torch.from_numpy(np.random.default_rng(1).standard_normal(n)).cuda()
    yv = torch.empty(n + (n & 1), dtype=torch.float64, device="cuda")[:n]
    A, z, dz, d2z = W.A, W.z, W.dz, W.d2z
    bt = timer(lambda: ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A), 20)
    build_ms = bt["median_ms"]
    upd = timer(lambda: ctx.bie_build_update(g.counts, g.kinds, z, dz, d2z, A), 20)
    M0_ = int(g.counts[0])
    upd_entries = n * n - (n - M0_) * (n - M0_)
    mv = timer(lambda: ctx.bie_matvec(A, xv, yv), 100)
    rd = timer(lambda: ctx.bie_probe_read(A, probe_out), 20)          # read-only stream of the same buffer, same run
    read_gbs = A.numel() * 8.0 / (rd["median_ms"] * 1e-3) / 1e9
    matvec = {"dense": dict(mv, gbs=8.0 * n * n / (mv["median_ms"] * 1e-3) / 1e9,
                            hbm_frac=8.0 * n * n / (mv["median_ms"] * 1e-3) / 1e9 / peak,
                            read_peak_gbs=read_gbs, frac_of_read_peak=8.0 * n * n / (mv["median_ms"] * 1e-3) / 1e9 / read_gbs,
                            read_peak_source="bie_probe_read on the matrix buffer in this run (128-bit evict-first loads from every SM)",
                            note="read-only stream against the read+write copy peak; about 75 MB of the matrix stay L2-resident by design "
                                 "(DESIGN.md section 6), so a fraction above 1 exceeds the copy peak, not the hardware")}
    ctx.bie_set_geometry(g.counts, g.kinds, z, dz, d2z)
    mf = timer(lambda: ctx.bie_matvec_free(xv, yv), 100)
    matvec["matrix_free"] = dict(mf, gentries_per_s=n * n / (mf["median_ms"] * 1e-3) / 1e9, fp64_instr_per_entry=FP64_PER_ENTRY_SYM,
                                 fp64_frac_of_probe=n * n * FP64_PER_ENTRY_SYM / (mf["median_ms"] * 1e-3) / dfma_per_s,
                                 fp64_frac_of_nominal=n * n * FP64_PER_ENTRY_SYM / (mf["median_ms"] * 1e-3) / NOMINAL_FP64_INSTR_S)

    # ---- SURVEY 8(f) NEXT rows, stand-alone calls outside the timed region ----------------------------
    next_rows = {}
    if not args.no_next_rows:
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        vx = timer(lambda: ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A, variant=2), 10)
        next_rows["vortex_sheet_matrix"] = {"call": "bie_build(variant=BIE_VARIANT_VORTEX)", "ms": vx["median_ms"], "best_ms": vx["best_ms"],
                                            "gentries_per_s": n * n / (vx["median_ms"] * 1e-3) / 1e9,
                                            "fp64_instr_per_entry": FP64_PER_ENTRY_VORTEX_BUILD,
                                            "fp64_frac_of_probe": n * n * FP64_PER_ENTRY_VORTEX_BUILD / (vx["median_ms"] * 1e-3) / dfma_per_s,
                                            "hbm_write_frac": 8.0 * n * n / (vx["median_ms"] * 1e-3) / 1e9 / peak}
        ctx.bie_set_geometry(g.counts, g.kinds, z, dz, d2z, variant=2)
        vmf = timer(lambda: ctx.bie_matvec_free(xv, yv), 20)
        next_rows["vortex_sheet_matrix"]["matrix_free_matvec_ms"] = vmf["median_ms"]
        next_rows["vortex_sheet_matrix"]["matrix_free_fp64_frac_of_probe"] = n * n * FP64_PER_PAIR_VORTEX / (vmf["median_ms"] * 1e-3) / dfma_per_s
        if P.centers:
            ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A, variant=1)
            cy = timer(lambda: ctx.bie_add_cyl_columns(g.counts, g.kinds, z, P.centers, A), 10)
            nobs_cols = int(sum(int(cn) for cn, kd in zip(g.counts, g.kinds) if kd == 2))
            next_rows["appendix_b_columns"] = {"call": "bie_add_cyl_columns (in place on the variant-B matrix)", "ms": cy["median_ms"],
                                               "entries": n * nobs_cols, "gbs": 16.0 * n * nobs_cols / (cy["median_ms"] * 1e-3) / 1e9,
                                               "hbm_frac": 16.0 * n * nobs_cols / (cy["median_ms"] * 1e-3) / 1e9 / peak}
        # NEXT-3: 2 functions (Phi', Phi_t of Eq. 5.3) at 65 536 points below the free surface
        npts_e = 65536
        rng_e = np.random.default_rng(3)
        ie = rng_e.integers(0, int(g.counts[0]), size=npts_e)
        zp_e = dev(g.zeta[ie] - 1j * rng_e.uniform(0.01, 0.3, size=npts_e))
        f_e = dev(np.vstack([np.exp(1j * g.zeta), np.exp(2j * g.zeta)]))
        out_e = torch.empty((2, npts_e), dtype=torch.complex128, device="cuda")
        ev = timer(lambda: ctx.bie_cauchy_eval(g.counts, g.kinds, z, dz, f_e, zp_e, out=out_e), 5)
        ev_instr = 9 + 4 * 3      # FP64-pipe instructions per pair: differences, denominator, reciprocal (9) + four per numerator (Cauchy sum and nf = 2 functions)
        next_rows["cauchy_eval_near_boundary"] = {"call": "bie_cauchy_eval (nf = 2)", "points": npts_e, "sources": n, "ms": ev["median_ms"],
                                                  "gpairs_per_s": npts_e * n / (ev["median_ms"] * 1e-3) / 1e9,
                                                  "fp64_instr_per_pair": ev_instr,
                                                  "fp64_frac_of_probe": npts_e * n * ev_instr / (ev["median_ms"] * 1e-3) / dfma_per_s}
        del zp_e, f_e, out_e
        M0 = int(g.counts[0])
        Nm = A.view(-1)[: M0 * A.stride(0)].view(M0, A.stride(0))       # the first M_0 rows of the same allocation
        wv = torch.from_numpy(np.random.default_rng(2).standard_normal(n)).cuda()
        uv = torch.empty(M0 + (M0 & 1), dtype=torch.float64, device="cuda")[:M0]
        nb = timer(lambda: ctx.bie_build_normal_velocity(g.counts, g.kinds, z, dz, d2z, Nm), 10)
        na = timer(lambda: ctx.bie_matvec_rect(Nm, wv, uv), 20)
        next_rows["normal_velocity"] = {"call": "bie_build_normal_velocity + bie_matvec_rect", "rows": M0, "cols": n,
                                        "build_ms": nb["median_ms"], "build_gentries_per_s": M0 * n / (nb["median_ms"] * 1e-3) / 1e9,
                                        "build_hbm_write_frac": 8.0 * M0 * n / (nb["median_ms"] * 1e-3) / 1e9 / peak,
                                        "apply_ms": na["median_ms"], "apply_gbs": 8.0 * M0 * n / (na["median_ms"] * 1e-3) / 1e9,
                                        "apply_hbm_frac": 8.0 * M0 * n / (na["median_ms"] * 1e-3) / 1e9 / peak}
        del Nm

    # ---- end to end through bie_solve_host, pinned host buffers ---------------------------------------------
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hz, hdz, hd2z, hb = pin(g.zeta.view(np.float64)), pin(g.dzeta.view(np.float64)), pin(g.d2zeta.view(np.float64)), pin(P.rhs[0])
    hx = torch.empty(n, dtype=torch.float64).pin_memory()
    del W, A
    torch.cuda.empty_cache()
    sws = torch.empty(ctx.bie_solve_workspace_bytes(n, P.restart, solve_mode), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        ctx.bie_solve_host(g.counts, g.kinds, hz, hdz, hd2z, hb, hx, P.tol, P.restart, P.max_iters, sws, solve_mode)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        e_it, e_rr, e_st = ctx.bie_solve_host(g.counts, g.kinds, hz, hdz, hd2z, hb, hx, P.tol, P.restart, P.max_iters,
                                              sws, solve_mode)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks((time.perf_counter() - t0) / K)
    h2d = 3 * 16 * n + 8 * n
    d2h = 8 * n + 8 + 8
    del sws
    torch.cuda.empty_cache()

    # ---- per_config (configs 1-4) ------------------------------------------------------------------------------
    per_config = {}
    if not args.no_per_config and args.config == 5 and world == 1:
        for c in (1, 2, 3, 4):
            per_config[str(c)] = measure_config(torch, bie, ctx, c, timer, dfma_per_s)

    if rank != 0:
        ranks.finish(R)
        return

    # ---- rooflines -------------------------------------------------------------------------------------------
    ng = n_gemv(iters, P.restart) * nstage       # operator applications in the GMRES bracket of one step
    nd = args.nd
    roof = gmres_roofline(n, op, nd, ng, gmres_ms, dfma_per_s, clocks and clocks.get("sm_mhz"), args.config)
    ach = n * n * FP64_PER_ENTRY_BUILD / (build_ms * 1e-3)
    roof_build = {"bound": "hbm", "kernel": "bie_build_kernel (+ node prep), stand-alone calls",
                  "achieved": 8.0 * n * n / (build_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s (write)",
                  "frac": 8.0 * n * n / (build_ms * 1e-3) / 1e9 / peak, "peak_source": peak_src,
                  "fp64": {"achieved": ach / 1e12, "unit": "T FP64 instr/s", "fp64_instr_per_entry": FP64_PER_ENTRY_BUILD,
                           "frac_of_probe": ach / dfma_per_s, "frac_of_nominal": ach / NOMINAL_FP64_INSTR_S,
                           "peak_probe": dfma_per_s / 1e12, "peak_nominal": NOMINAL_FP64_INSTR_S / 1e12},
                  "note": "with 10 FP64 instructions per entry the HBM write of 8 B per entry is the binding bound; the FP64 fractions "
                          "are the non-binding leg"}
    # kernels launched per step: node prep (1) [+ tile kernel (1)] + GMRES (1) per stage; the near matrix (count, scan, fill) and the
    # symmetric work list (1) once per stage geometry for the matrix-free and hybrid operators
    launches = {"dense": 3, "free": 2 + 4, "hybrid": 3 + 4}[op] * nstage

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(P, args, iters),
            "build": {"gentries_per_s": n * n / (build_ms * 1e-3) / 1e9, "ms": build_ms, "best_ms": bt["best_ms"], "reps": bt["reps"],
                      "in_step": op == "dense",
                      "note": "full bie_build, stand-alone calls outside the timed region (median of 20); inside the step the %s operator "
                              "spent %.4f ms on its own preparation per first stage (node tables%s)"
                              % (op, prep_ms, {"dense": " + whole matrix", "free": "", "hybrid": " + leading block of %d rows" % nd}[op])},
            "build_update": {"ms": upd["median_ms"], "best_ms": upd["best_ms"], "entries": upd_entries,
                             "gentries_per_s": upd_entries / (upd["median_ms"] * 1e-3) / 1e9, "share_of_matrix": upd_entries / float(n * n)},
            "gmres": {"ms": gmres_ms, "iters": iters, "relres_true": relres, "us_per_iter": gmres_ms * 1e3 / max(iters * nstage, 1),
                      "stages": nstage, "note": "ms covers all stages of the step (incl. their rebuilds after the first); iters is the last stage's"},
            "e2e": {"value": world * n * n / e2e_s / 1e9, "unit": UNIT, "ms_per_step": e2e_s * 1e3,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "api": "bie_solve_host (first stage of the config)", "iters": e_it},
            "gpu_launches": launches * K,
            "roofline": roof, "roofline_build": roof_build, "matvec": matvec, "clocks": clocks,
            "fp64_probe_tflops": 2 * dfma_per_s / 1e12,
            "operator_choice_ms_per_step": choice_ms or None, "per_config": per_config or None, "next_rows": next_rows or None}
    if not args.no_cpu_baseline:
        cfgs = sorted(set([args.config] + ([1, 2, 3, 4] if per_config else [])))
        cb = cpu_baseline(cfgs)
        h = cb[str(args.config)]
        line["cpu_baseline"] = {"value": h["gentries_per_s"], "unit": UNIT, "cores": h["cores"], "kind": "oracle", "estimated": False,
                                "sample": "ONE real pass of the oracle over the whole workload (oracle.build_matrix + oracle.gmres, every "
                                          "stage) on all host cores; per_config holds the same for configs 1-4 and one-thread runs for 1-3",
                                "ms_per_step": h["step_s"] * 1e3, "build_gentries_per_s": h["build_gentries_per_s"],
                                "gmres_ms": h["gmres_s"] * 1e3, "iters": h["iters"], "per_config": cb}
    print(json.dumps(line), flush=True)
    ranks.finish(R)


if __name__ == "__main__":
    main()
