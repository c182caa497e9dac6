#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path over one synthetic geometry:
node preparation + dense build of the matrix of Eq. (3.16) (bie_build) + restarted GMRES on it (bie_gmres).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference] [--matrix-free]

Prints ONE JSON line (rank 0).  Default workload: BASELINE.json configs[4] (n = 16384, 2.1 GB matrix, restart 100,
tol 1e-13), the largest single-GPU configuration; its matrix is 17x the L2, so every GEMV streams from HBM.

  value         whole-step throughput: n^2 matrix entries built AND solved per second, inputs resident in HBM
  build/gmres   the two halves of BASELINE.json's metric on their own: Gentries/s of the build, ms of the solve
  e2e           the same step through bie_solve_host with pinned HOST buffers (H2D of nodes+rhs, D2H of the density)
  roofline      dominant kernel = the persistent GMRES kernel (HBM-bound GEMVs): algorithmic bytes / event time
  roofline_build  the entry builder against the FP64 pipe (DFMA rate measured by bie_probe_dfma in this run)
  cpu_baseline  the oracle (oracle/, as it stands) on this box's host cores, on a bounded sample of the same workload

--impl reference times the oracle alone (this tier has no reference implementation).
N > 1: replicas only: every rank runs the same step on its own GPU, no data-path collective.
"""
from __future__ import annotations

import argparse
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
FP64_INSTR_PER_ENTRY = 13      # FP64-pipe instructions per stored matrix entry (SASS count)
FP64_INSTR_PER_PAIR_FREE = 11  # one-directional pair loops (hybrid operator): FP64-pipe instructions per entry (bie_free.cuh)
FP64_INSTR_PER_ENTRY_SYM = 7.7  # symmetric pair loops (whole-matrix matrix-free operator, bie_free_sym.cuh): 15 per pair of
                                # entries + 9 DADD of the lane reduction per 32 pairs, i.e. 7.64 per entry; own blocks 11
HBM_FALLBACK_GBS = 6650.0      # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# dram__bytes_read.sum + dram__bytes_write.sum of the GMRES kernel, one launch, from the committed ncu capture
# (profiles/r01_ncu_full_gmres_cfg5.md); None for workloads that were not captured
TRAFFIC_BYTES = {(5, "dense"): 341.50e9, (5, "hybrid"): 142.37e9}   # profiles/r01b_ncu_full_cfg5.md, r01e_launches_cfg5.md


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--operator", default="auto", choices=["auto", "dense", "free", "hybrid"],
                    help="dense: bie_build + GMRES on the stored matrix; free: matrix-free GMRES (entries recomputed on the "
                         "fly, no matrix); hybrid: a slab of bie_hybrid_cols(n) columns stored and streamed while the other "
                         "sources are recomputed; auto (default): all are timed during warm-up and the fastest is the timed step")
    ap.add_argument("--matrix-free", action="store_true", help="same as --operator free")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="budget of the oracle sample")
    a = ap.parse_args()
    if a.matrix_free:
        a.operator = "free"
    return a


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def n_gemv(iters: int, restart: int) -> int:
    """GEMVs of one bie_gmres launch: one per Arnoldi step, one residual per restart, one final true residual"""
    cycles = max(1, -(-iters // restart))
    return iters + (cycles - 1) + 1


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
def oracle_sample(P, iters: int, seconds: float):
    """Times the oracle, as it stands, on a bounded sample of the workload: a block of R rows of the matrix
    (oracle_build_rows), the GEMV on that block (oracle_matvec_rect) and, when the whole problem fits the budget,
    nothing is extrapolated.  Returns (step_seconds_estimate, description, cores)."""
    import oracle
    g = P.geometry
    n = g.n
    cores = oracle.num_threads()
    rng = np.random.default_rng(0)
    # rate of the build on 64 rows, then as many rows as fit ~40 % of the budget
    rows = np.sort(rng.choice(n, size=min(n, 64), replace=False))
    t = time.perf_counter()
    oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, rows)
    dt = max(time.perf_counter() - t, 1e-6)
    R = int(min(n, max(64, 0.4 * seconds / dt * rows.size)))
    rows = np.sort(rng.choice(n, size=R, replace=False))
    t = time.perf_counter()
    blk = oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, rows)
    t_build_rows = time.perf_counter() - t
    x = rng.standard_normal(n)
    oracle.matvec(blk, x)
    reps, t_mv = 0, 0.0
    t0 = time.perf_counter()
    while True:
        oracle.matvec(blk, x)
        reps += 1
        t_mv = time.perf_counter() - t0
        if t_mv > 0.4 * seconds or reps >= 200:
            break
    t_build = t_build_rows * n / R
    t_gemv = t_mv / reps * n / R
    ng = n_gemv(iters, P.restart)
    est = t_build + ng * t_gemv
    desc = (f"oracle_build_rows on {R} of {n} rows ({t_build_rows:.2f} s) and {reps} oracle GEMVs on that {R}x{n} block "
            f"({t_mv:.2f} s); step = n/R * build + {ng} GEMVs (the GPU run's count) * n/R * block GEMV; "
            f"Gram-Schmidt O(n*iters) not included")
    return est, desc, cores, {"build_s": t_build, "gemv_s": t_gemv, "gemvs": ng}


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, same config/metric/unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2108_01786_b200 import inputs
    P = inputs.make_config(args.config)
    n = P.n
    args.op, args.stored_cols = "dense", n     # the oracle stores the matrix
    iters_nominal = {1: 18, 2: 33, 3: 74, 4: 127, 5: 158}[args.config]  # the oracle's own counts (tests)
    per = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(P, iters_nominal, per)
    ests = []
    for _ in range(args.steps):
        est, desc, cores, parts = oracle_sample(P, iters_nominal, per)
        ests.append(est)
    est = float(np.mean(ests))
    val = n * n / est / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": est * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(P, args, iters_nominal),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "build": {"gentries_per_s": n * n / parts["build_s"] / 1e9, "ms": parts["build_s"] * 1e3},
            "gmres": {"ms": parts["gemv_s"] * parts["gemvs"] * 1e3, "iters": iters_nominal}}
    print(json.dumps(line), flush=True)


def l2_policy(n, stored_cols):
    """what the timed iterations stream: the stored part of the matrix against the 126 MB L2"""
    stored = 8.0 * n * stored_cols
    if stored_cols == 0:
        return ("no matrix stored (matrix-free operator): the O(n) node tables are L2-resident by design, the kernel is "
                "FP64-bound; nothing to flush")
    if stored > 2.5e8:
        return "stored part of the matrix (%.0f MB) is %.1fx the 126 MB L2: every operator application streams it from HBM; no flush needed" % (stored / 1e6, stored / 126e6)
    return "stored matrix (%.0f MB) fits the 126 MB L2: L2-resident GEMV, reported as such" % (stored / 1e6)


def workload_config(P, args, iters):
    g = P.geometry
    return {"workload": f"BASELINE.json configs[{P.config - 1}]: {P.name}", "n": int(g.n),
            "counts": [int(c) for c in g.counts], "restart": int(P.restart), "tol": P.tol,
            "operator": {"dense": "dense", "free": "matrix-free", "hybrid": "hybrid (stored slab + recomputed sources)"}[args.op]
                        + (" (chosen by measurement)" if args.operator == "auto" else ""),
            "matrix_bytes": int(8 * g.n * args.stored_cols), "stored_columns": int(args.stored_cols),
            "l2_policy": l2_policy(g.n, args.stored_cols),
            "stages_per_step": len(P.stages), "replicas": int(args.gpus)}


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
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
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    z, dz, d2z, b = dev(g.zeta), dev(g.dzeta), dev(g.d2zeta), dev(P.rhs[0])
    # the stored matrix is also needed for the stand-alone dense GEMV timing, whichever operator the step uses
    A = torch.empty((n, n + (n & 1)), dtype=torch.float64, device="cuda")
    x = torch.empty(n + (n & 1), dtype=torch.float64, device="cuda")[:n]
    ws = torch.empty(ctx.bie_gmres_workspace_bytes(n, P.restart), dtype=torch.uint8, device="cuda")
    oi = torch.zeros(2, dtype=torch.int32, device="cuda")
    of = torch.zeros(1, dtype=torch.float64, device="cuda")

    # BASELINE.json configs[3] is a SEQUENCE of stages (Gamma_0 moves, the solids stay): one step = all its stages, the
    # first with a full build, the others with bie_build_update (a4); every other config has one stage
    stages = [(gs, tuple(dev(a) for a in (gs.zeta, gs.dzeta, gs.d2zeta)), dev(bs)) for gs, bs in zip(P.stages, P.rhs)]
    nstage = len(stages)

    def step_dense(ev=None):
        for si, (gs, (zs, dzs, d2zs), bs) in enumerate(stages):
            if ev and si == 0: ev[0].record()
            if si == 0:
                ctx.bie_build(gs.counts, gs.kinds, zs, dzs, d2zs, A)      # 2 launches: node prep + tile kernel
            else:
                ctx.bie_build_update(gs.counts, gs.kinds, zs, dzs, d2zs, A)   # only the blocks touching Gamma_0
            if ev and si == 0: ev[1].record()
            ctx.bie_gmres(A, bs, x, P.tol, P.restart, P.max_iters, ws, oi, of)  # 1 cooperative launch
        if ev: ev[2].record()

    def step_free(ev=None):
        for si, (gs, (zs, dzs, d2zs), bs) in enumerate(stages):
            if ev and si == 0: ev[0].record()
            ctx.bie_set_geometry(gs.counts, gs.kinds, zs, dzs, d2zs)      # 1 launch: node prep
            if ev and si == 0: ev[1].record()
            ctx.bie_gmres(None, bs, x, P.tol, P.restart, P.max_iters, ws, oi, of)  # near matrix (3) + 1 cooperative launch
        if ev: ev[2].record()

    nd = ctx.bie_hybrid_cols(n)

    def step_hybrid(ev=None):
        for si, (gs, (zs, dzs, d2zs), bs) in enumerate(stages):
            if ev and si == 0: ev[0].record()
            ctx.bie_build_block(gs.counts, gs.kinds, zs, dzs, d2zs, nd, A)  # 2 launches: node prep + block tiles
            if ev and si == 0: ev[1].record()
            ctx.bie_gmres_hybrid(A, nd, bs, x, P.tol, P.restart, P.max_iters, ws, oi, of)  # near matrix (3) + 1 launch
        if ev: ev[2].record()

    def time_steps(fn, k):
        torch.cuda.synchronize()
        a_, c_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a_.record()
        for _ in range(k):
            fn()
        c_.record(); torch.cuda.synchronize()
        return a_.elapsed_time(c_) / k

    # operator choice by measurement (north_star: "matrix-free fused rebuild+matvec variant chosen by measurement")
    steps = {"dense": step_dense, "free": step_free}
    if nd > 0:
        steps["hybrid"] = step_hybrid
    choice_ms = {}
    op = args.operator
    if op == "hybrid" and nd == 0:
        raise SystemExit("bench: n is too small for the hybrid operator")
    if op == "auto":
        for name, fn in steps.items():
            fn()
            choice_ms[name] = max_over_ranks(time_steps(fn, 2))
        op = min(choice_ms, key=choice_ms.get)
    step = steps[op]
    args.op = op
    args.stored_cols = {"dense": n, "free": 0, "hybrid": nd}[op]
    args.matrix_free = (op == "free")
    launches_per_step = {"dense": 3, "free": 5, "hybrid": 6}[op] * nstage
    solve_mode = {"dense": 0, "free": 1, "hybrid": 2}[op]

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    iters, status, relres = int(oi[0]), int(oi[1]), float(of[0])
    if status != 0 or not (relres <= 1e-12):
        raise SystemExit(f"bench: GMRES did not converge (status {status}, relres {relres})")

    # FP64 pipe rate of this GPU, now (roofline denominator of the build)
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
        step(evs[k])
    t_end.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(t_start.elapsed_time(t_end))
    build_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    gmres_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    ms_per_step = total_ms / K
    value = world * nstage * n * n / (ms_per_step * 1e-3) / 1e9

    # ---- the stand-alone operator calls (outside the timed region; matvec against HBM) ---------
    def time_call(fn, reps):
        fn(); torch.cuda.synchronize()
        a, c = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        c.record(); torch.cuda.synchronize()
        return a.elapsed_time(c) / reps

    xv = torch.from_numpy(np.random.default_rng(1).standard_normal(n)).cuda()
    yv = torch.empty(n + (n & 1), dtype=torch.float64, device="cuda")[:n]
    matvec = {}
    prep_ms = build_ms
    if args.op != "dense":   # the full dense build is not part of this step: time it on its own (stand-alone calls, warm)
        build_ms = time_call(lambda: ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A), 20)
    # a4: partial rebuild (only the blocks touching Gamma_0), stand-alone, on the matrix just built
    ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A)
    upd_ms = time_call(lambda: ctx.bie_build_update(g.counts, g.kinds, z, dz, d2z, A), 20)
    M0_ = int(g.counts[0])
    upd_entries = n * n - (n - M0_) * (n - M0_)
    mv_ms = time_call(lambda: ctx.bie_matvec(A, xv, yv), 50)
    matvec["dense"] = {"ms": mv_ms, "gbs": 8.0 * n * n / (mv_ms * 1e-3) / 1e9, "hbm_frac": 8.0 * n * n / (mv_ms * 1e-3) / 1e9 / hbm_peak()[0]}
    mf_ms = time_call(lambda: ctx.bie_matvec_free(xv, yv), 20)
    matvec["matrix_free"] = {"ms": mf_ms, "gentries_per_s": n * n / (mf_ms * 1e-3) / 1e9,
                             "fp64_instr_per_entry": FP64_INSTR_PER_ENTRY_SYM,
                             "fp64_frac": n * n * FP64_INSTR_PER_ENTRY_SYM / (mf_ms * 1e-3) / dfma_per_s}

    # ---- SURVEY 8(f) NEXT rows built so far, stand-alone calls outside the timed region ----------------------------
    next_rows = {}
    vx_ms = time_call(lambda: ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A, variant=2), 10)
    next_rows["vortex_sheet_matrix"] = {"call": "bie_build(variant=BIE_VARIANT_VORTEX)", "ms": vx_ms,
                                        "gentries_per_s": n * n / (vx_ms * 1e-3) / 1e9,
                                        "fp64_frac": n * n * FP64_INSTR_PER_ENTRY / (vx_ms * 1e-3) / dfma_per_s,
                                        "hbm_write_frac": 8.0 * n * n / (vx_ms * 1e-3) / 1e9 / hbm_peak()[0]}
    ctx.bie_set_geometry(g.counts, g.kinds, z, dz, d2z, variant=2)
    vmf_ms = time_call(lambda: ctx.bie_matvec_free(xv, yv), 20)
    next_rows["vortex_sheet_matrix"]["matrix_free_matvec_ms"] = vmf_ms
    next_rows["vortex_sheet_matrix"]["matrix_free_fp64_frac"] = n * n * 13 / (vmf_ms * 1e-3) / dfma_per_s
    if P.centers:
        ctx.bie_build(g.counts, g.kinds, z, dz, d2z, A, variant=1)
        cyl_ms = time_call(lambda: ctx.bie_add_cyl_columns(g.counts, g.kinds, z, P.centers, A), 10)
        nobs_cols = int(sum(int(cn) for cn, kd in zip(g.counts, g.kinds) if kd == 2))
        next_rows["appendix_b_columns"] = {"call": "bie_add_cyl_columns (in place on the variant-B matrix)", "ms": cyl_ms,
                                           "entries": n * nobs_cols, "gbs": 16.0 * n * nobs_cols / (cyl_ms * 1e-3) / 1e9,
                                           "hbm_frac": 16.0 * n * nobs_cols / (cyl_ms * 1e-3) / 1e9 / hbm_peak()[0]}
    # NEXT-3: 2 functions (Phi', Phi_t of Eq. 5.3) at 65 536 points below the free surface
    npts_e = 65536
    rng_e = np.random.default_rng(3)
    ie = rng_e.integers(0, int(g.counts[0]), size=npts_e)
    zp_e = dev(g.zeta[ie] - 1j * rng_e.uniform(0.01, 0.3, size=npts_e))
    f_e = dev(np.vstack([np.exp(1j * g.zeta), np.exp(2j * g.zeta)]))
    zc_e, dzc_e = dev(g.zeta), dev(g.dzeta)
    out_e = torch.empty((2, npts_e), dtype=torch.complex128, device="cuda")
    ev_ms = time_call(lambda: ctx.bie_cauchy_eval(g.counts, g.kinds, zc_e, dzc_e, f_e, zp_e, out=out_e), 5)
    ev_instr = 12 + 4 * 3     # FP64-pipe instructions per pair: cot (12) + denominator and two numerators (4 each)
    next_rows["cauchy_eval_near_boundary"] = {"call": "bie_cauchy_eval (nf = 2)", "points": npts_e, "sources": n, "ms": ev_ms,
                                              "gpairs_per_s": npts_e * n / (ev_ms * 1e-3) / 1e9,
                                              "fp64_instr_per_pair": ev_instr,
                                              "fp64_frac": npts_e * n * ev_instr / (ev_ms * 1e-3) / dfma_per_s}
    del zp_e, f_e, out_e
    M0 = int(g.counts[0])
    Nm = A.view(-1)[: M0 * A.stride(0)].view(M0, A.stride(0))       # the first M_0 rows of the same allocation
    wv = torch.from_numpy(np.random.default_rng(2).standard_normal(n)).cuda()
    uv = torch.empty(M0 + (M0 & 1), dtype=torch.float64, device="cuda")[:M0]
    nb_ms = time_call(lambda: ctx.bie_build_normal_velocity(g.counts, g.kinds, z, dz, d2z, Nm), 10)
    na_ms = time_call(lambda: ctx.bie_matvec_rect(Nm, wv, uv), 20)
    next_rows["normal_velocity"] = {"call": "bie_build_normal_velocity + bie_matvec_rect", "rows": M0, "cols": n,
                                    "build_ms": nb_ms, "build_gentries_per_s": M0 * n / (nb_ms * 1e-3) / 1e9,
                                    "build_hbm_write_frac": 8.0 * M0 * n / (nb_ms * 1e-3) / 1e9 / hbm_peak()[0],
                                    "apply_ms": na_ms, "apply_gbs": 8.0 * M0 * n / (na_ms * 1e-3) / 1e9,
                                    "apply_hbm_frac": 8.0 * M0 * n / (na_ms * 1e-3) / 1e9 / hbm_peak()[0]}
    del Nm

    # ---- end to end through bie_solve_host, pinned host buffers ---------------------------------------------
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hz, hdz, hd2z, hb = pin(g.zeta.view(np.float64)), pin(g.dzeta.view(np.float64)), pin(g.d2zeta.view(np.float64)), pin(P.rhs[0])
    hx = torch.empty(n, dtype=torch.float64).pin_memory()
    del A
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

    if rank != 0:
        ranks.finish(R)
        return

    # ---- rooflines -------------------------------------------------------------------------------------------
    peak, peak_src = hbm_peak()
    # operator applications in the GMRES bracket of one step (all stages; the last stage's count stands for each)
    ng = n_gemv(iters, P.restart) * nstage
    if args.op != "dense":
        sc = args.stored_cols          # 0 (matrix-free) or the slab width (hybrid)
        pairs = ng * n * (n - sc)
        per_entry = FP64_INSTR_PER_PAIR_FREE if sc else FP64_INSTR_PER_ENTRY_SYM   # hybrid: one-directional loops
        instr = pairs * per_entry + ng * n * sc          # + one DFMA per streamed slab entry
        roof = {"bound": "alu", "kernel": "bie_gmres_kernel<%s> (persistent; pair loops dominate)" % args.op,
                "achieved": instr / (gmres_ms * 1e-3) / 1e12, "peak": dfma_per_s / 1e12,
                "unit": "T FP64 instr/s", "traffic": TRAFFIC_BYTES.get((args.config, args.op)),
                "fp64_instr_per_entry": per_entry,
                "pairs_per_launch": pairs, "operator_applications_per_launch": ng,
                "peak_source": "bie_probe_dfma in this run (nominal 148 SM x 64 lanes x 1.965 GHz = 18.6)"}
        if sc:   # the slab is streamed from HBM by the other warps at the same time
            gbs = ng * 8.0 * n * sc / (gmres_ms * 1e-3) / 1e9
            roof["hbm_concurrent"] = {"achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                                      "algorithmic_bytes_per_launch": ng * 8 * n * sc, "peak_source": peak_src}
    else:
        roof = {"bound": "hbm", "kernel": "bie_gmres_kernel (persistent; GEMV phases dominate)",
                "achieved": ng * 8.0 * n * n / (gmres_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                "traffic": TRAFFIC_BYTES.get((args.config, args.op)), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ng * 8 * n * n, "gemvs_per_launch": ng}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof_build = None
    if True:
        ach = n * n * FP64_INSTR_PER_ENTRY / (build_ms * 1e-3)
        roof_build = {"bound": "alu", "kernel": "bie_build_kernel (+ node prep)", "achieved": ach / 1e12,
                      "peak": dfma_per_s / 1e12, "unit": "T FP64 instr/s", "frac": ach / dfma_per_s,
                      "peak_source": "bie_probe_dfma in this run (nominal 148 SM x 64 lanes x 1.965 GHz = 18.6)",
                      "fp64_instr_per_entry": FP64_INSTR_PER_ENTRY,
                      "hbm_write_gbs": 8.0 * n * n / (build_ms * 1e-3) / 1e9, "hbm_write_frac": 8.0 * n * n / (build_ms * 1e-3) / 1e9 / peak}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(P, args, iters),
            "build": {"gentries_per_s": n * n / (build_ms * 1e-3) / 1e9, "ms": build_ms,
                      "in_step": args.op == "dense",
                      "note": "inside the timed step" if args.op == "dense" else
                              "full bie_build, stand-alone calls outside the timed region; inside the step the %s operator "
                              "spent %.4f ms on its own preparation (node tables%s)"
                              % (args.op, prep_ms, " + slab of %d columns" % args.stored_cols if args.stored_cols else "")},
            "build_update": {"ms": upd_ms, "entries": upd_entries, "gentries_per_s": upd_entries / (upd_ms * 1e-3) / 1e9,
                             "share_of_matrix": upd_entries / float(n * n)},
            "gmres": {"ms": gmres_ms, "iters": iters, "relres_true": relres, "us_per_iter": gmres_ms * 1e3 / max(iters * nstage, 1),
                      "stages": nstage, "note": "ms covers all stages of the step (incl. their rebuilds after the first); iters is the last stage's"},
            "e2e": {"value": world * n * n / e2e_s / 1e9, "unit": UNIT, "ms_per_step": e2e_s * 1e3,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "api": "bie_solve_host", "iters": e_it},
            "gpu_launches": launches_per_step * K,
            "roofline": roof, "roofline_build": roof_build, "matvec": matvec, "clocks": clocks,
            "fp64_probe_tflops": 2 * dfma_per_s / 1e12,
            "operator_choice_ms_per_step": choice_ms or None, "next_rows": next_rows}
    if not args.no_cpu_baseline:
        est, desc, cores, parts = oracle_sample(P, iters, args.cpu_seconds)
        line["cpu_baseline"] = {"value": n * n / est / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                "ms_per_step": est * 1e3, "build_gentries_per_s": n * n / parts["build_s"] / 1e9,
                                "gmres_ms": parts["gemv_s"] * parts["gemvs"] * 1e3}
    print(json.dumps(line), flush=True)
    ranks.finish(R)


if __name__ == "__main__":
    main()
