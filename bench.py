#!/usr/bin/env python3
"""bench.py - one JSON line per run (driver contract).

A "step" is one pass of the WHOLE hot path over one batch of synthetic input:
  a1 incident expansion -> a2 RHS -> a3-a6 forward GMRES (on-the-fly translation + all-pairs matvec +
  T application + Arnoldi/Givens) -> a7 adjoint GMRES with a seeded random weight vector -> a8 scattered
  E field on a detector plane.
Metric (BASELINE.json): pair-block complex MAC/s = (all-pairs matvecs in the step) x (ordered pairs) x L^2 / time.
Default workload: BASELINE.json configs[4] = cfg5, the 200x200 lattice the north-star target (>= 50 % of FP64 peak for the
all-pairs kernel) is stated on and the largest single-GPU config.  Its full solve takes ~1500 GMRES iterations (minutes),
so the default step (--mode hotpath) runs every row of the path with the two GMRES solves BOUNDED to --cycle-iters Arnoldi
iterations each (labelled in config.step; 12 all-pairs launches of 1.6e9 ordered pairs per step, from which `roofline` is
computed).  The full solves to convergence stay visible in the `solve` sub-record (config 2, the paper's window size, full
forward + adjoint solves to 1e-10 per step) and in profiles/ (config 5 to 1e-8).  `--workload cfgN --mode full` runs full
solves of any config as the step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg5] [--mode hotpath|full|matvec]

N > 1 (torchrun): replicas only - every rank runs the same independent problem (the paper's windows are
independent units); no data-path collective; value = sum over ranks / max time.
"""
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

from paper_2107_09879_b200 import workloads as W  # noqa: E402

METRIC = "pair_block_complex_MAC_per_s"
UNIT = "cMAC/s"


def n_pairs(w):
    wp = np.asarray(w["win_ptr"], dtype=np.int64)
    c = np.diff(wp)
    return int(np.sum(c * (c - 1)))


def detector_points(w, n_side=64, height=5.0):
    pos = w["pos"]
    lo, hi = pos.min(axis=0), pos.max(axis=0)
    gx = np.linspace(lo[0], hi[0], n_side)
    gy = np.linspace(lo[1], hi[1], n_side)
    X, Y = np.meshgrid(gx, gy, indexing="xy")
    return np.ascontiguousarray(np.stack([X.ravel(), Y.ravel(), np.full(X.size, pos[0, 2] + height)], axis=1))


def adjoint_weight(w):
    if "w_adj" in w:
        return np.ascontiguousarray(w["w_adj"])
    rng = np.random.default_rng(1234)
    return W.complex_normal((w["pos"].shape[0], W.n_modes(w["lmax"])), rng)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index, interval_ms=250):
        self.rows, self.proc, self.index, self.interval_ms = [], None, index, interval_ms

    def start(self):
        if self.interval_ms <= 0:
            return
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-lms", str(self.interval_ms)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            # nvidia-smi's start-up (NVML initialisation) briefly stalls kernel launches: let it finish before the warm-up,
            # so that the hiccup cannot land in the timed region (seen as a 2-3x outlier in the first timed step)
            t0 = time.perf_counter()
            while not self.rows and time.perf_counter() - t0 < 10.0:
                time.sleep(0.05)
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) >= 7 and r[3 + k].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


# --------------------------------------------------------------------------------------------- reference arm
def run_reference(args, w, rank, world):
    """The oracle (CPU, as it stands) on a bounded sample of the same workload: its matrix-free all-pairs
    matvec (oracle/matvec_c.c, OpenMP) on a row sample per step."""
    if rank != 0:
        return
    from oracle import matvec as omv
    omv.build()
    N, L = w["pos"].shape[0], W.n_modes(w["lmax"])
    x = adjoint_weight(w)
    rng = np.random.default_rng(7)
    omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=np.arange(2, dtype=np.int32), win_ptr=w["win_ptr"])   # tables, load
    t0 = time.perf_counter()
    omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=np.arange(min(64, N), dtype=np.int32), win_ptr=w["win_ptr"])
    per_row = (time.perf_counter() - t0) / min(64, N)
    rows_per_step = int(max(4, min(N, 4.0 / per_row)))          # ~4 s of CPU work per step
    wp = np.asarray(w["win_ptr"])
    win_of = np.searchsorted(wp, np.arange(N), side="right") - 1
    times, pairs = [], []
    for it in range(args.warmup + args.steps):
        rows = np.sort(rng.choice(N, rows_per_step, replace=False)).astype(np.int32)
        t0 = time.perf_counter()
        omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=rows, win_ptr=w["win_ptr"])
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt)
            pairs.append(int(np.sum(wp[win_of[rows] + 1] - wp[win_of[rows]] - 1)))
    val = sum(pairs) * L * L / sum(times)
    sample = f"{rows_per_step} random target rows of one all-pairs matvec per step (oracle/matvec_c.c, OpenMP)"
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": config_record(w, args, "matvec" if args.mode not in ("hotpath", "full", "matvec") else args.mode),
           "reference_step": sample,
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": omv.num_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# --------------------------------------------------------------------------------------------- our arm
def max_over_ranks(values, dist, device):
    """Replicas only: the ranks share nothing but the clock - per-step times are reduced with
    MAX over ranks (one tiny all_reduce after the timed region; no data-path collective)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return list(values)
    import torch
    tt = torch.tensor(list(values), device=device, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt]


def aggregate_value(world, units_per_rank_step, t_step_ms):
    """Whole-job throughput: every rank processes the same units per step (weak scaling), time = max over ranks."""
    return world * units_per_rank_step / (t_step_ms * 1e-3)


def cpu_baseline(w):
    from oracle import matvec as omv
    omv.build()
    N, L = w["pos"].shape[0], W.n_modes(w["lmax"])
    x = adjoint_weight(w)
    omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=np.arange(2, dtype=np.int32), win_ptr=w["win_ptr"])   # tables, load
    t0 = time.perf_counter()
    omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=np.arange(min(64, N), dtype=np.int32), win_ptr=w["win_ptr"])
    per_row = (time.perf_counter() - t0) / min(64, N)
    n_rows = int(max(4, min(N, 12.0 / per_row)))
    rows = np.sort(np.random.default_rng(7).choice(N, n_rows, replace=False)).astype(np.int32)
    wp = np.asarray(w["win_ptr"])
    win_of = np.searchsorted(wp, np.arange(N), side="right") - 1
    t0 = time.perf_counter()
    omv.matvec_rows(w["lmax"], w["k"], w["pos"], x, rows=rows, win_ptr=w["win_ptr"])
    dt = time.perf_counter() - t0
    prs = int(np.sum(wp[win_of[rows] + 1] - wp[win_of[rows]] - 1))
    return {"value": prs * L * L / dt, "unit": UNIT, "cores": omv.num_threads(), "kind": "oracle",
            "sample": f"{n_rows} of {N} target rows of one all-pairs matvec ({prs} ordered pairs, {dt:.1f} s, oracle/matvec_c.c)"}


NOMINAL_LANES = {"fp64": 64, "fp32": 128}      # FMA lanes per SM (B200: 148 SMs x 64 FP64 / 128 FP32 lanes x 2 flop x SM clock)


def config_record(w, args, mode):
    """The `config` object of the JSON line: a function of the workload and the command line only, so that the reference
    arm (`--impl reference`) prints the identical object for the same command."""
    tol = args.tol or w["tol"]
    step = {"matvec": "one operator application y = (I - T A) x",
            "hotpath": f"incident expansion + RHS + forward GMRES bounded to {args.cycle_iters} Arnoldi iterations + adjoint GMRES bounded to "
                       f"{args.cycle_iters} iterations (+ the true-residual operator application of each) + E field on 64x64 detector points",
            "full": ("incident + forward GMRES solve to tol + E field (adjoint skipped: --forward-only)" if args.forward_only else
                     "incident + forward GMRES solve to tol + adjoint GMRES solve to tol + E field on 64x64 detector points")}[mode]
    return {"workload": w["name"], "n_scat": int(w["pos"].shape[0]), "lmax": int(w["lmax"]), "L": W.n_modes(w["lmax"]),
            "n_windows": len(w["win_ptr"]) - 1, "ordered_pairs": n_pairs(w), "tol": tol, "restart": int(w["restart"]),
            "mode": mode, "step": step, "precision": args.precision, "l2": "flushed between steps (256 MB write)"}


def measure(args, w, mode, steps, warmup, rank, world, local_rank, dist, st, peaks, legs=("e2e", "mixed", "cpu")):
    """Times `steps` steps of `mode` on workload `w` (after `warmup`) and returns the record (all ranks compute it; rank 0
    prints).  legs: which extra legs to run - "e2e" (host buffers through the C ABI), "mixed" (TM_MIXED, labelled),
    "cpu" (oracle on the host cores)."""
    import torch
    from paper_2107_09879_b200 import libtm
    prec = {"fp32": libtm.TM_FP32, "mixed": libtm.TM_MIXED}.get(args.precision, libtm.TM_FP64)
    N, L = w["pos"].shape[0], W.n_modes(w["lmax"])
    pairs = n_pairs(w)
    pts = detector_points(w)
    wadj = adjoint_weight(w)
    tol = args.tol or w["tol"]
    max_iter = args.cycle_iters if mode == "hotpath" else (args.max_iter or w["max_iter"])
    restart = min(w["restart"], max_iter) if mode == "hotpath" else w["restart"]

    with torch.cuda.stream(st):
        # TM_MIXED: all but one all-pairs launch per restart cycle run on the FP32 pipe, so that pipe's peak is the denominator
        peak_prec = libtm.TM_FP64 if prec == libtm.TM_FP64 else libtm.TM_FP32
        pipe = "fp64" if peak_prec == libtm.TM_FP64 else "fp32"
        if pipe not in peaks:
            peaks[pipe] = libtm.measure_fma_peak(peak_prec, st.cuda_stream)
        peak = peaks[pipe]
        kern_req = {"auto": libtm.TM_KERNEL_AUTO, "general": libtm.TM_KERNEL_GENERAL, "coplanar": libtm.TM_KERNEL_COPLANAR,
                    "sym3d": libtm.TM_KERNEL_SYM3D, "rot3d": libtm.TM_KERNEL_ROT3D}[args.kernel]
        s = libtm.solver_for_workload(w, precision=prec, stream=st.cuda_stream, kernel=kern_req)
        ws = torch.empty(s.workspace_bytes(restart), dtype=torch.uint8, device="cuda")
        s.set_workspace(ws)
        d_w = torch.from_numpy(wadj).cuda()
        d_pts = torch.from_numpy(pts).cuda()
        d_s = torch.empty((N, L), dtype=torch.complex128, device="cuda")
        d_lam = torch.empty_like(d_s)
        d_E = torch.empty((pts.shape[0], 3), dtype=torch.complex128, device="cuda")
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2

        def set_inc(sol):
            if w["inc_kind"] == "plane":
                sol.set_incident_plane(w["beta"], w["alpha"], w["A_beta"], w["A_alpha"])
            else:
                sol.set_incident_gauss(w["focus"], w["w0"], w["Ax"], w["Ay"])

        d_x = torch.from_numpy(wadj).cuda()
        d_y = torch.empty_like(d_x)

        def step_matvec():
            s.matvec(d_x, 0, out=d_y)
            one = libtm.SolveInfo(0, 0, 1, 1, 0.0, 0.0)
            zero = libtm.SolveInfo(0, 0, 1, 0, 0.0, 0.0)
            return [one], [zero], 0, 0

        solve_log = []

        def step_resident():
            set_inc(s)
            _, info, rc = s.solve(tol, restart, max_iter, out=d_s)
            solve_log.append(round(1e3 * info[0].seconds, 2))
            if args.forward_only:
                info2, rc2 = [libtm.SolveInfo(0, 0, 1, 0, 0.0, 0.0)], 0
            else:
                _, info2, rc2 = s.solve_adjoint(d_w, tol, restart, max_iter, out=d_lam)
            if not args.forward_only:
                solve_log.append(round(1e3 * info2[0].seconds, 2))
            s.fields(d_pts, d_s, libtm.TM_FIELD_E_SCA, out=d_E)
            return info, info2, rc, rc2

        def timed(fn, n_warm, n_steps, sol=None, timing_mode=-1):
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
            res = None
            import gc
            gc.collect()
            gc.disable()                                    # no collector pauses between the ~2000 launches of a step
            for it in range(n_warm + n_steps):
                flush.fill_(it & 0xff)                      # L2 flush between iterations (outside the timed bracket)
                if it == n_warm:
                    if sol is not None:
                        sol.kernel_time(reset=timing_mode)
                    if dist is not None:
                        dist.barrier()
                    torch.cuda.synchronize()
                if it >= n_warm:
                    ev[it - n_warm][0].record(st)
                res = fn()
                if it >= n_warm:
                    ev[it - n_warm][1].record(st)
            torch.cuda.synchronize()
            gc.enable()
            if dist is not None:
                dist.barrier()
            return [a.elapsed_time(b) for a, b in ev], res

        clocks = ClockSampler(local_rank, args.clock_interval_ms)
        clocks.start()
        # (1) the timed region proper: production mode (restart cycles of window-sized problems replayed as CUDA graphs)
        step_fn = step_matvec if mode == "matvec" else step_resident
        if args.profile:       # under ncu: timing mode only (launch by launch, no CUDA graph replay), one pass
            ms_list, (info, info2, rc, rc2) = timed(step_fn, warmup, steps, s, timing_mode=1)
            ap_ms, ap_launches, tot_launches = s.kernel_time(reset=False)
            ap_per_run, prof_steps, prof_ms = ap_launches, steps, ms_list
        else:
            ms_list, (info, info2, rc, rc2) = timed(step_fn, warmup, steps, s)
            _, ap_per_run, tot_launches = s.kernel_time(reset=False)
            # (2) the same steps in the library's timing mode (an event pair around every all-pairs launch, cycles issued launch
            #     by launch): average all-pairs launch duration for the roofline.  Its step time is reported beside (1).
            prof_steps = max(1, min(steps, 3))
            prof_ms, _ = timed(step_fn, 1, prof_steps, s, timing_mode=1)
            ap_ms, ap_launches, _ = s.kernel_time(reset=False)
            s.kernel_time(reset=-1)
        clk = clocks.stop()
        matvecs = info[0].matvecs + info2[0].matvecs
        total_ms = float(sum(ms_list))
        # physics self-check of the timed solution (outside the timed region, one extra all-pairs product): lossless scatterers
        # scatter what they extinguish,  -Re p^H s = |s|^2 + Re s^H A s  (SURVEY.md 8(c) O9 / identity S4b); holds at any size
        energy = None
        if mode == "full":
            s.matvec(d_s, 2, out=d_y)                                       # u = A s
            d_p = torch.empty_like(d_s)
            s.get_incident(out=d_p)
            ext = -float(torch.vdot(d_p.reshape(-1), d_s.reshape(-1)).real)
            sca = float(torch.vdot(d_s.reshape(-1), d_s.reshape(-1)).real + torch.vdot(d_s.reshape(-1), d_y.reshape(-1)).real)
            energy = {"extinction": ext, "scattering": sca, "rel_defect": abs(ext - sca) / abs(ext),
                      "note": "coefficient units (x pi/k^2 = cross-section for a unit plane wave); lossless T: defect ~ solver residual"}

        # end to end through the C ABI with HOST buffers: context creation (uploads positions, T, types), incident,
        # both solves and the field evaluation, every result copied back to host memory
        if w["t_kind"] in ("mie_types", "mie_sites"):
            T_host = np.stack([libtm.mie_tmatrix(w["lmax"], w["k"], r, w["eps_r"]) for r in w["radii"]])
        else:
            T_host = np.ascontiguousarray(w["t_full"])
        h_s = np.empty((N, L), dtype=np.complex128)
        h_lam = np.empty_like(h_s)
        h_E = np.empty((pts.shape[0], 3), dtype=np.complex128)
        h_y = np.empty_like(wadj)

        def step_e2e_matvec():
            s.matvec(wadj, 0, out=h_y)
            return [libtm.SolveInfo(0, 0, 1, 1, 0.0, 0.0)], [libtm.SolveInfo(0, 0, 1, 0, 0.0, 0.0)], 0, 0

        def step_e2e():
            s2 = libtm.Solver(w["pos"], w["lmax"], w["k"], win_ptr=w["win_ptr"], precision=prec, stream=st.cuda_stream)
            s2.set_workspace(ws)
            s2.set_tmatrices(T_host, w["type_of"], w["t_kind"] != "full_types")
            set_inc(s2)
            _, i1, _ = s2.solve(tol, restart, max_iter, out=h_s)
            _, i2, _ = s2.solve_adjoint(wadj, tol, restart, max_iter, out=h_lam)
            s2.fields(pts, h_s, libtm.TM_FIELD_E_SCA, out=h_E)
            s2.close()
            return i1, i2, 0, 0

        e2e_steps = max(1, min(steps, 5))
        e2e = None
        if "e2e" in legs and not args.profile:
            e2e_ms, (i1, i2, _, _) = timed(step_e2e_matvec if mode == "matvec" else step_e2e, 1, e2e_steps)
            e2e_matvecs = i1[0].matvecs + i2[0].matvecs
            if mode == "matvec":
                h2d, d2h = wadj.nbytes, h_y.nbytes
            else:
                h2d = w["pos"].nbytes + T_host.nbytes + np.asarray(w["type_of"]).nbytes + wadj.nbytes + pts.nbytes + h_s.nbytes
                d2h = h_s.nbytes + h_lam.nbytes + h_E.nbytes
            e2e = (e2e_ms, e2e_matvecs, h2d, d2h)
        fpinst, flop = s.pair_cost()
        # extra, clearly labelled leg: the same step in TM_MIXED (GMRES with iterative refinement: fp32 Krylov cycles, fp64
        # iterate and true residual - same tolerance, same true-residual test).  Not the contract value (that is fp64).
        mixed = None
        if "mixed" in legs and prec == libtm.TM_FP64 and mode == "full" and not args.profile and not args.forward_only:
            sm = libtm.solver_for_workload(w, precision=libtm.TM_MIXED, stream=st.cuda_stream, kernel=kern_req)
            wsm = torch.empty(sm.workspace_bytes(restart), dtype=torch.uint8, device="cuda")
            sm.set_workspace(wsm)

            def step_mixed():
                set_inc(sm)
                _, j1, r1 = sm.solve(tol, restart, max_iter, out=d_s)
                _, j2, r2 = sm.solve_adjoint(d_w, tol, restart, max_iter, out=d_lam)
                sm.fields(d_pts, d_s, libtm.TM_FIELD_E_SCA, out=d_E)
                return j1, j2, r1, r2
            mx_ms, (j1, j2, r1, r2) = timed(step_mixed, 2, 3)
            mt = float(sum(mx_ms)) / len(mx_ms)
            mixed = {"precision": "fp32 Krylov cycles + fp64 iterate / true residual (TM_MIXED)", "ms_per_step": mt, "steps": 3,
                     "value": (j1[0].matvecs + j2[0].matvecs) * pairs * L * L / (mt * 1e-3), "unit": UNIT,
                     "forward_iterations": max(i.iterations for i in j1), "adjoint_iterations": max(i.iterations for i in j2),
                     "forward_rel_residual": max(i.rel_residual for i in j1), "adjoint_rel_residual": max(i.rel_residual for i in j2),
                     "converged": bool(r1 == 0 and r2 == 0)}
            sm.close()
        kern = s.get_kernel()
        s.close()

    # max over ranks
    t_step = total_ms / len(ms_list)
    t_e2e = float(sum(e2e[0])) / len(e2e[0]) if e2e else 0.0
    t_step, t_e2e = max_over_ranks([t_step, t_e2e], dist, "cuda")
    cmac_step = matvecs * pairs * L * L
    value = aggregate_value(world, cmac_step, t_step)

    ap_avg_ms = ap_ms / max(1, ap_launches)
    achieved = pairs * flop / (ap_avg_ms * 1e-3) * 1e-12 if ap_launches else None
    traffic = None          # DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture
    tpath = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if os.path.exists(tpath):
        for ln in open(tpath).read().splitlines()[1:]:
            f = ln.split(",")
            if len(f) >= 3 and f[0] == w["name"]:
                traffic = float(f[2])
    sm_max = (clk.get("sm_max_mhz") or 1965.0) * 1e6
    nominal = 148 * NOMINAL_LANES[pipe] * 2 * sm_max * 1e-12
    cfg = config_record(w, args, mode)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": t_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {libtm.TM_FP64: "f64", libtm.TM_FP32: "f32"}.get(prec, "f32 cycles + f64 residual/iterate"), "data": "synthetic",
        "config": cfg,
        "launch": {"kernel": {libtm.TM_KERNEL_COPLANAR: "coplanar", libtm.TM_KERNEL_SYM3D: "sym3d", libtm.TM_KERNEL_ROT3D: "rot3d"}.get(kern, "general"),
                   "parallelism": "replicas" if world > 1 else "single"},
        "solve": {"forward_iterations": max(i.iterations for i in info), "adjoint_iterations": max(i.iterations for i in info2),
                  "forward_rel_residual": max(i.rel_residual for i in info), "adjoint_rel_residual": max(i.rel_residual for i in info2),
                  "forward_seconds": info[0].seconds, "adjoint_seconds": info2[0].seconds, "converged": bool(rc == 0 and rc2 == 0),
                  "bounded": mode == "hotpath", "matvecs_per_step": matvecs, "matvecs_per_s": matvecs / (t_step * 1e-3)},
        "gpu_launches": int(tot_launches),
        "roofline": {"bound": "alu", "kernel": {libtm.TM_KERNEL_COPLANAR: "k_allpairs_coplanar", libtm.TM_KERNEL_SYM3D: "k_allpairs_sym3d",
                                                 libtm.TM_KERNEL_ROT3D: "k_allpairs_rot3d"}.get(kern, "k_allpairs_general"),
                     "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": (achieved / peak) if achieved else None,
                     "peak_source": "builder microbenchmark: tm_measure_fma_peak (register-resident FMA chains) on this GPU in this run; "
                                    "MEASURED_PEAKS.json has no FP64/FP32 FMA figure",
                     "peak_pipe": pipe, "peak_nominal": nominal, "frac_of_nominal": (achieved / nominal) if achieved else None,
                     "peak_nominal_source": f"148 SMs x {NOMINAL_LANES[pipe]} {pipe} lanes x 2 flop x {sm_max * 1e-6:.0f} MHz (max SM clock)",
                     "flop_per_pair": flop, "fp_instr_per_pair": fpinst, "pairs_per_launch": pairs,
                     "avg_launch_ms": ap_avg_ms, "launches": int(ap_launches), "launches_per_step": ap_per_run / max(1, steps),
                     "share_of_step": (ap_avg_ms * ap_per_run / steps) / t_step if t_step else None,
                     "timing_pass": {"steps": prof_steps, "ms_per_step": float(sum(prof_ms)) / len(prof_ms),
                                     "note": "event pair around every all-pairs launch; restart cycles issued launch by launch (no CUDA graph)"},
                     "pipe_frac": (pairs * fpinst / (ap_avg_ms * 1e-3)) / (peak * 1e12 / 2) if ap_launches else None,
                     "pairs_per_s": pairs / (ap_avg_ms * 1e-3) if ap_launches else None, "traffic": traffic},
        "energy_balance": energy, "clocks": clk, "ms_steps": [round(v, 3) for v in ms_list],
        "solve_ms_log": solve_log[-2 * steps:] if mode != "matvec" else [],
    }
    if e2e:
        out["e2e"] = {"value": aggregate_value(world, e2e[1] * pairs * L * L, t_e2e), "unit": UNIT, "h2d_bytes_per_step": int(e2e[2]),
                      "d2h_bytes_per_step": int(e2e[3]), "ms_per_step": t_e2e, "steps": e2e_steps,
                      "ms_steps": [round(float(v), 3) for v in e2e[0]]}
    if mixed is not None:
        out["mixed_precision"] = mixed
    if "cpu" in legs and not args.no_cpu_baseline and world == 1 and rank == 0:
        out["cpu_baseline"] = cpu_baseline(w)
    return out


def run_ours(args, w, rank, world, local_rank):
    import torch
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if args.restart:
        w["restart"] = args.restart
    st = torch.cuda.Stream()
    peaks = {}
    out = measure(args, w, args.mode, args.steps, args.warmup, rank, world, local_rank, dist, st, peaks)
    # Labelled sub-record: full forward + adjoint solves TO CONVERGENCE on config 2 (the paper's window size), so
    # that solve seconds / iterations stay visible beside the bounded config-5 step of the contract line.
    if args.mode == "hotpath" and not args.no_solve_record and not args.profile:
        w2 = W.config(2)
        sub = measure(args, w2, "full", 5, 3, rank, world, local_rank, dist, st, peaks, legs=("mixed",))
        out["solve_record"] = {k: sub[k] for k in ("value", "unit", "ms_per_step", "steps", "warmup", "config", "solve", "gpu_launches",
                                                   "roofline", "energy_balance", "ms_steps") if k in sub}
        if "mixed_precision" in sub:
            out["solve_record"]["mixed_precision"] = sub["mixed_precision"]
    if rank == 0:
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_nyquist(args, w, rank=0, world=1, local_rank=0):
    """Recorded run of the paper's distribution strategy (NEXT-1; not the contract line): a Gaussian beam sampled on the
    lambda/2 grid -> jinc sources -> groups + padded windows batched on one GPU -> summed fields, against the undistributed
    solve of the same sources.  Under torchrun (--gpus N) the windows are DEALT to the ranks (nyquist.simulate(rank, world,
    dist): rank r solves windows r, r + N, ...) and the detector fields are summed by ONE all_reduce - the only exchange step of
    the paper's strategy; strong scaling of one fixed problem, time = max over ranks."""
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(local_rank)
    from paper_2107_09879_b200 import nyquist
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    half = float(np.abs(w["pos"][:, 0]).max()) + 0.25
    w0 = half / 2.0
    field = lambda x, y: (np.exp(-(x * x + y * y) / w0 ** 2), np.zeros_like(x))
    src, amp, gi = nyquist.jinc_sources(w["k"], (-half, half), (-half, half), 0.0, field, drop_below=1e-6)
    g = np.linspace(-half, half, 33)
    pts = np.array([[a, b, 5.0] for a in g for b in g])
    out = {"mode": "nyquist", "workload": w["name"], "n_scat": int(w["pos"].shape[0]), "n_sources": int(src.shape[0]),
           "group_samples": args.group, "padding": args.padding, "tol": args.tol or 1e-8, "n_gpus": world,
           "scaling": "strong (windows dealt to the ranks, one all_reduce of the detector field)"}
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    E, inf = nyquist.simulate(w, src, amp, gi, args.group, args.padding, pts, tol=args.tol or 1e-8, rank=rank, world=world, dist=dist)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    stats = max_over_ranks([wall, inf["seconds"]], dist, "cuda")
    out.update(distributed={"n_windows_this_rank": inf["n_windows"], "batched_scatterers_this_rank": inf["n_batched_scatterers"],
                            "iterations": inf["iterations"], "solve_seconds_max_over_ranks": stats[1], "wall_seconds_max_over_ranks": stats[0],
                            "max_rel_residual": inf["max_rel_residual"], "converged": inf["rc"] == 0})
    if rank == 0 and not args.no_undistributed:
        t0 = time.perf_counter()
        E0, inf0 = nyquist.simulate(w, src, amp, gi, None, 0.0, pts, tol=args.tol or 1e-8)
        torch.cuda.synchronize()
        out.update(undistributed={"iterations": inf0["iterations"], "solve_seconds": inf0["seconds"], "wall_seconds": time.perf_counter() - t0,
                                  "converged": inf0["rc"] == 0},
                   field_rel_l2_error=float(np.linalg.norm(E - E0) / np.linalg.norm(E0)))
    if rank == 0:
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_gradient(args, w):
    """Recorded run of the adjoint sensitivities (NEXT-2; not the contract line): forward solve, adjoint solve, then ALL radius
    and position derivatives of J = w^T s from tm_grad_tmatrix / tm_grad_positions."""
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    assert w["t_kind"] in ("mie_types", "mie_sites") and w["inc_kind"] == "plane"
    s = libtm.solver_for_workload(w)
    N, L = s.n_scat, s.L
    tol = args.tol or w["tol"]
    wv = adjoint_weight(w)
    t0 = time.perf_counter()
    sol, i1, rc1 = s.solve(tol, w["restart"], args.max_iter or w["max_iter"])
    lam, i2, rc2 = s.solve_adjoint(wv, tol, w["restart"], args.max_iter or w["max_iter"])
    t1 = time.perf_counter()
    dT = np.stack([libtm.mie_tmatrix_dR(w["lmax"], w["k"], r, w["eps_r"]) for r in w["radii"]])
    t2 = time.perf_counter()
    gR = s.grad_tmatrix(dT, lam, sol)
    t3 = time.perf_counter()
    p = s.get_incident()
    kv = w["k"] * np.array([np.sin(w["beta"]) * np.cos(w["alpha"]), np.sin(w["beta"]) * np.sin(w["alpha"]), np.cos(w["beta"])])
    dp = 1j * kv[None, :, None] * p[:, None, :]
    t4 = time.perf_counter()
    gX = s.grad_positions(lam, sol, dp=dp)
    t5 = time.perf_counter()
    print(json.dumps({"mode": "gradient", "workload": w["name"], "n_scat": N, "L": L, "design_variables": int(N + 3 * N),
                      "solves_seconds": t1 - t0, "forward_iterations": i1[0].iterations, "adjoint_iterations": i2[0].iterations,
                      "converged": rc1 == 0 and rc2 == 0, "grad_tmatrix_seconds": t3 - t2, "grad_positions_seconds": t5 - t4,
                      "grad_positions_allpairs_launches": 2, "grad_positions_lmax_of_products": w["lmax"] + 1, "norm_grad_R": float(np.linalg.norm(gR)),
                      "norm_grad_x": float(np.linalg.norm(gX))}), flush=True)
    s.close()


def run_multirhs(args, w):
    """Recorded run (NEXT-3, multi-RHS; not the contract line): n_rhs plane waves (both polarisations, then two oblique ones) on ONE
    geometry, (a) solved one after the other on a single-window context and (b) batched - the geometry replicated as n_rhs windows
    of one auxiliary context inside the library (tm_solve_multi), every window with its own right-hand side, Krylov scalars and convergence mask.  Also prints the measured
    FP64 tensor-core (DMMA) and FP64 FMA peaks: the bound of a dense-block multi-RHS route against that of the factorised apply."""
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    assert w["inc_kind"] == "plane" and w["t_kind"] in ("mie_types", "mie_sites")
    n_rhs = args.n_rhs
    waves = [(0.0, 0.0, 1.0, 0.0), (0.0, 0.0, 0.0, 1.0), (0.3, 0.4, 1.0, 0.0), (0.3, 0.4, 0.0, 1.0)][:n_rhs]
    tol, restart, max_iter = args.tol or w["tol"], args.restart or w["restart"], args.max_iter or w["max_iter"]
    N = w["pos"].shape[0]
    s1 = libtm.solver_for_workload(w)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    sols, ps, its = [], [], []
    for rep in range(2):                                    # first pass warms up (graphs, pools)
        sols, its = [], []
        e0, e1 = ev(), ev()
        e0.record()
        for (b, a, Ab, Aa) in waves:
            s1.set_incident_plane(b, a, Ab, Aa)
            sol, info, rc = s1.solve(tol, restart, max_iter)
            sols.append(sol); its.append(info[0].iterations)
        e1.record(); torch.cuda.synchronize()
        t_seq = e0.elapsed_time(e1)
    for (b, a, Ab, Aa) in waves:
        s1.set_incident_plane(b, a, Ab, Aa)
        ps.append(s1.get_incident())
    P = np.stack(ps)
    for rep in range(2):                                    # tm_solve_multi: the geometry replicated as windows inside the library
        e0, e1 = ev(), ev()
        e0.record()
        solb, infob, rcb = s1.solve_multi(P, tol, restart, max_iter)
        e1.record(); torch.cuda.synchronize()
        t_bat = e0.elapsed_time(e1)
    err = max(float(np.linalg.norm(solb[i] - sols[i]) / np.linalg.norm(sols[i])) for i in range(n_rhs))
    st = torch.cuda.current_stream().cuda_stream
    print(json.dumps({"mode": "multirhs", "workload": w["name"], "n_scat": N, "lmax": w["lmax"], "n_rhs": n_rhs, "tol": tol,
                      "sequential_ms": t_seq, "sequential_iterations": its, "batched_ms": t_bat,
                      "batched_iterations": [i[0].iterations for i in infob], "gain": t_seq / t_bat,
                      "max_rel_diff_batched_vs_sequential": err, "converged": bool(rcb == 0),
                      "fp64_fma_peak_tflops": libtm.measure_fma_peak(libtm.TM_FP64, st),
                      "fp64_tensor_dmma_peak_tflops": libtm.measure_fma_peak(libtm.TM_PEAK_FP64_TENSOR, st)}), flush=True)
    s1.close()


def run_nullfield(args):
    """Recorded run of NEXT-4 (not the contract line): null-field T-matrices of a library of cylinders (the paper's meta-atom
    library) at the paper's truncation lmax 6 in ONE tm_nullfield_tmatrix call; the oracle's literal
    surface quadrature timed on one shape beside it."""
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    lmax = args.lmax or 6
    n_shapes, n_panel = 256, 64
    radii = np.linspace(0.10, 0.24, n_shapes)
    gens = [W.generatrix_cylinder(r, 0.3, n_panel) for r in radii]
    libtm.nullfield_tmatrix(lmax, W.K_B, 4.0, gens[:2])                     # warm-up (module load, pool)
    ts = []
    for _ in range(5):
        t0 = time.perf_counter()
        T = libtm.nullfield_tmatrix(lmax, W.K_B, 4.0, gens, lmax_internal=args.lmax_internal)
        ts.append(time.perf_counter() - t0)
    n = T.shape[1]
    S = np.eye(n)[None] + 2.0 * T
    unit = float(np.abs(S @ np.conj(np.swapaxes(S, 1, 2)) - np.eye(n)[None]).max())
    out = {"mode": "nullfield", "lmax": lmax, "lmax_internal": args.lmax_internal or lmax, "L": n, "n_shapes": n_shapes, "nodes_per_shape": 3 * n_panel,
           "call_ms_median_incl_copies": 1e3 * float(np.median(ts)), "shapes_per_s": n_shapes / float(np.median(ts)),
           "max_unitarity_defect": unit}
    if not args.no_cpu_baseline:
        from oracle import nullfield as onf
        t0 = time.perf_counter()
        ref = onf.nullfield_tmatrix(lmax, W.K_B, 4.0, gens[100], lmax_internal=args.lmax_internal or None)
        out.update(oracle_seconds_per_shape=time.perf_counter() - t0,
                   max_rel_error_vs_oracle=float(np.abs(T[100] - ref).max() / np.abs(ref).max()))
    print(json.dumps(out), flush=True)


def run_ttable(args):
    """Recorded run (NEXT-4, not the contract line): T-matrices AND dT/dR of every scatterer of the paper's 120 um lens (112 x 112
    cylinders) from a 64-node radius table at the paper's truncation (lmax 6, full 96 x 96 T), one tm_ttable_interp
    call on device arrays.  Algorithmic bytes = the outputs written once (2 x n_out x L^2 x 16 B) + the table read once; the
    peak is MEASURED_PEAKS.json's HBM copy bandwidth."""
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    lmax = args.lmax or 6
    L = W.n_modes(lmax)
    n_tab, n_out = 64, (args.scale or 112) ** 2
    rng = np.random.default_rng(0)
    nodes = torch.linspace(0.05, 0.25, n_tab, dtype=torch.float64, device="cuda")
    tab = torch.randn((n_tab, L, L), dtype=torch.complex128, device="cuda")
    radii = torch.from_numpy(rng.uniform(0.05, 0.25, n_out)).cuda()
    T = torch.empty((n_out, L, L), dtype=torch.complex128, device="cuda")
    dT = torch.empty_like(T)
    st = torch.cuda.current_stream().cuda_stream
    for _ in range(3):
        libtm.ttable_interp(nodes, tab, radii, out=T, dout=dT, stream=st)
    ts = []
    for _ in range(args.steps or 20):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        libtm.ttable_interp(nodes, tab, radii, out=T, dout=dT, stream=st)
        e1.record(); torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    ms = float(np.median(ts))
    alg = 2 * n_out * L * L * 16 + n_tab * L * L * 16 + n_out * 8
    peak, src = 6540.5, "fallback"
    try:
        peak, src = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        pass
    out = {"mode": "ttable", "lmax": lmax, "L": L, "n_tab": n_tab, "n_out": n_out, "call_ms_median": ms, "tmatrices_per_s": n_out / ms * 1e3,
           "roofline": {"bound": "hbm", "achieved": alg / ms * 1e-6, "peak": peak, "unit": "GB/s", "frac": alg / ms * 1e-6 / peak,
                        "peak_source": src, "algorithmic_bytes": alg,
                        "note": "whole call incl. the per-site weight kernel, scratch allocation and the flag read-back"}}
    if not args.no_cpu_baseline:
        from oracle import ttable as ott
        pick = rng.choice(n_out, 8, replace=False)
        t0 = time.perf_counter()
        T_ref, dT_ref = ott.interp_table(nodes.cpu().numpy(), tab.cpu().numpy(), radii.cpu().numpy()[pick])
        out.update(oracle_seconds_per_site=(time.perf_counter() - t0) / len(pick),
                   max_rel_error_vs_oracle=float(np.abs(T[torch.from_numpy(pick).cuda()].cpu().numpy() - T_ref).max() / np.abs(T_ref).max()),
                   max_rel_error_derivative=float(np.abs(dT[torch.from_numpy(pick).cuda()].cpu().numpy() - dT_ref).max() / np.abs(dT_ref).max()))
    print(json.dumps(out), flush=True)


def run_fields(args, w):
    """Recorded run of row a8 (not the contract line): scattered E field of ALL scatterers of the workload on a --pts x --pts
    detector grid (default 256 x 256 = the static entry point's maximum), device arrays, CUDA events around tm_fields (k_fields_sym +
    k_fields_reduce) and, beside it, around tm_fields_static (same kernels, its own chunk count and scratch)."""
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    n_side = args.pts
    pts = torch.from_numpy(detector_points(w, n_side)).cuda()
    N, L = w["pos"].shape[0], W.n_modes(w["lmax"])
    rng = np.random.default_rng(0)
    sol = torch.from_numpy(W.complex_normal((N, L), rng)).cuda()
    pos = torch.from_numpy(w["pos"]).cuda()
    ctx = libtm.Solver(w["pos"], w["lmax"], w["k"])
    out = torch.empty((pts.shape[0], 3), dtype=torch.complex128, device="cuda")
    out_s = torch.empty_like(out)
    st = torch.cuda.current_stream().cuda_stream

    def timed(fn):
        for _ in range(2):
            fn()
        ts = []
        for _ in range(args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))
    ms = timed(lambda: ctx.fields(pts, sol, libtm.TM_FIELD_E_SCA, out=out))
    rec = {"mode": "fields", "workload": w["name"], "n_scat": N, "lmax": w["lmax"], "n_pts": int(pts.shape[0]), "tm_fields_ms": ms,
           "point_source_pairs_per_s": N * pts.shape[0] / ms * 1e3, "mode_evaluations_per_s": N * pts.shape[0] * L / ms * 1e3}
    if pts.shape[0] <= 65536 and not args.profile:
        ms_s = timed(lambda: libtm.fields_static(w["lmax"], w["k"], pos, sol, pts, libtm.TM_FIELD_E_SCA, out=out_s, stream=st))
        rec.update(tm_fields_static_ms=ms_s, max_rel_diff=float((out - out_s).abs().max() / out_s.abs().max()))
    print(json.dumps(rec), flush=True)
    ctx.close()


def run_paper_case(args):
    """Recorded run (not the contract line): the paper's own largest single-GPU case end to end on its own kind of meta-atom
    (workloads.paper_lens: 56 x 56 silicon cylinders, lmax 6; 1-1.5 h on a V100): null-field T-matrices of the
    radius library -> coupled solve to the paper's residual 1e-6 -> E field on the focal plane."""
    import torch
    assert torch.cuda.is_available()
    from paper_2107_09879_b200 import libtm
    lmax = args.lmax or 6
    w = W.paper_lens(args.scale or 56)
    N = w["pos"].shape[0]
    prec = {"fp64": libtm.TM_FP64, "fp32": libtm.TM_FP32, "mixed": libtm.TM_MIXED}[args.precision]
    libtm.nullfield_tmatrix(lmax, w["k"], w["eps_r"], W.generatrix_cylinder(w["radii"][0], w["height"], 8))      # module load
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    gens = [W.generatrix_cylinder(r, w["height"], 64) for r in w["radii"]]
    T = libtm.nullfield_tmatrix(lmax, w["k"], w["eps_r"], gens, lmax_internal=args.lmax_internal)
    t1 = time.perf_counter()
    s = libtm.Solver(w["pos"], lmax, w["k"], precision=prec)
    r_enc = np.sqrt(w["radii"] ** 2 + (0.5 * w["height"]) ** 2)
    s.set_tmatrices(T, w["type_of"], False, r_enclosing=r_enc)
    s.set_incident_plane(0.0, 0.0, 1.0, 0.0)
    s.kernel_time(reset=True)
    t2 = time.perf_counter()
    sol, info, rc = s.solve(args.tol or 1e-6, args.restart or 50, args.max_iter or 5000)
    t3 = time.perf_counter()
    g = (np.arange(64) - 31.5) * (10.0 / 64)
    X, Y = np.meshgrid(g, g)
    pts = np.stack([X.ravel(), Y.ravel(), np.full(X.size, w["focal"])], axis=1)
    E = s.fields(pts, sol) + s.fields(pts, sol, libtm.TM_FIELD_E_INC)
    t4 = time.perf_counter()
    ap_ms, ap_launches, _ = s.kernel_time(reset=False)
    u = s.matvec(sol, transpose=2)
    p = s.get_incident()
    ext = -float(np.real(np.vdot(p, sol)))
    sca = float(np.real(np.vdot(sol, sol)) + np.real(np.vdot(sol, u)))
    n = T.shape[1]
    S = np.eye(n)[None] + 2.0 * T
    I2 = np.sum(np.abs(E) ** 2, axis=1).reshape(64, 64)
    print(json.dumps({"mode": "paper_case", "workload": w["name"], "n_scat": N, "lmax": lmax, "L": n, "n_types": len(gens),
                      "lmax_internal": args.lmax_internal or lmax, "precision": args.precision, "tmatrix_seconds": t1 - t0, "setup_seconds": t2 - t1, "solve_seconds": t3 - t2,
                      "fields_seconds": t4 - t3, "total_seconds": t4 - t0, "iterations": info[0].iterations,
                      "matvecs": info[0].matvecs, "rel_residual": info[0].rel_residual, "converged": rc == 0,
                      "allpairs_ms_per_launch": ap_ms / max(1, ap_launches), "kernel": s.get_kernel(),
                      "library_unitarity_defect": float(np.abs(S @ np.conj(np.swapaxes(S, 1, 2)) - np.eye(n)[None]).max()),
                      "energy_balance": {"extinction": ext, "scattering": sca, "rel_defect": abs(ext - sca) / abs(ext)},
                      "focal_plane": {"peak_intensity_over_incident": float(I2.max()),
                                      "peak_offset_wavelengths": [float(X.ravel()[I2.argmax()]), float(Y.ravel()[I2.argmax()])]}}),
          flush=True)
    s.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--mode", default=None, choices=["hotpath", "full", "matvec", "nyquist", "gradient", "nullfield", "paper_case", "multirhs", "ttable", "fields"],
                    help="hotpath (default for cfg5): every row of the path with both GMRES solves bounded to --cycle-iters iterations; "
                         "full (default otherwise): solves to tolerance; matvec: operator applications only; others: recorded runs")
    ap.add_argument("--cycle-iters", type=int, default=5, help="hotpath mode: Arnoldi iterations per (forward / adjoint) solve")
    ap.add_argument("--no-solve-record", action="store_true", help="hotpath mode: skip the config-2 full-solve sub-record")
    ap.add_argument("--n-rhs", type=int, default=2, choices=[1, 2, 3, 4], help="multirhs mode: right-hand sides on one geometry")
    ap.add_argument("--group", type=int, default=16, help="nyquist mode: samples per group side")
    ap.add_argument("--padding", type=float, default=4.0, help="nyquist mode: padding in wavelengths")
    ap.add_argument("--no-undistributed", action="store_true", help="nyquist mode: skip the undistributed reference solve")
    ap.add_argument("--kernel", default="auto", choices=["auto", "general", "coplanar", "sym3d", "rot3d"], help="force the all-pairs kernel variant")
    ap.add_argument("--lmax", type=int, default=None, help="override the VSWF truncation of a Mie config (lmax 6 = the paper's, PAPER.md:271)")
    ap.add_argument("--lmax-internal", type=int, default=0,
                    help="paper_case / nullfield modes: internal truncation of the null-field method (0 = lmax, the paper's setting)")
    ap.add_argument("--pts", type=int, default=256, help="--mode fields: detector grid side")
    ap.add_argument("--scale", type=int, default=None, help="lattice side override (parity-size runs)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"],
                    help="mixed: GMRES with iterative refinement (fp32 Krylov cycles, fp64 iterate and true residual)")
    ap.add_argument("--max-iter", type=int, default=None)
    ap.add_argument("--restart", type=int, default=None, help="override the GMRES restart length of the workload (<= 300)")
    ap.add_argument("--tol", type=float, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--clock-interval-ms", type=int, default=250, help="nvidia-smi sampling period during the timed region")
    ap.add_argument("--forward-only", action="store_true", help="recorded big-config runs: skip the adjoint solve (not the contract step)")
    ap.add_argument("--profile", action="store_true", help="for ncu: 1 warm-up, no e2e leg, no CPU baseline (not a bench value)")
    args = ap.parse_args()
    if args.mode is None:
        args.mode = "hotpath" if args.workload == "cfg5" and args.scale is None else "full"
    if args.profile:
        args.no_cpu_baseline = True
        args.warmup = min(args.warmup, 1)
    elif args.impl == "ours":
        args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.workload == "paper_lens":        # the paper's own kind of layout (silicon cylinders, null-field T-matrices): nyquist mode
        assert args.mode == "nyquist", "--workload paper_lens is for --mode nyquist (or use --mode paper_case)"
        import torch
        torch.cuda.set_device(local_rank)
        from paper_2107_09879_b200 import libtm
        w = W.paper_lens(args.scale or 56)
        lmax = args.lmax or 6
        gens = [W.generatrix_cylinder(r, w["height"], 64) for r in w["radii"]]
        w.update(lmax=lmax, t_kind="full_types", win_ptr=np.array([0, w["pos"].shape[0]], dtype=np.int32),
                 t_full=libtm.nullfield_tmatrix(lmax, w["k"], w["eps_r"], gens, lmax_internal=args.lmax_internal or 10))
        run_nyquist(args, w, rank, world, local_rank)
        return
    name = args.workload[3:] if args.workload.startswith("cfg") else args.workload
    w = W.config(name if name == "3b" else int(name), scale=args.scale)
    if args.lmax is not None:
        assert w["t_kind"] != "full_types", "--lmax needs a Mie config"
        w["lmax"] = args.lmax
        w["name"] += f"_lmax{args.lmax}"
        if "w_adj" in w:
            del w["w_adj"]
    if args.mode == "nullfield":
        if rank == 0:
            run_nullfield(args)
    elif args.mode == "ttable":
        if rank == 0:
            run_ttable(args)
    elif args.mode == "paper_case":
        if rank == 0:
            run_paper_case(args)
    elif args.mode == "nyquist":
        run_nyquist(args, w, rank, world, local_rank)
    elif args.mode == "gradient":
        if rank == 0:
            run_gradient(args, w)
    elif args.mode == "multirhs":
        if rank == 0:
            run_multirhs(args, w)
    elif args.mode == "fields":
        if rank == 0:
            run_fields(args, w)
    elif args.impl == "reference":
        run_reference(args, w, rank, world)
    else:
        run_ours(args, w, rank, world, local_rank)


if __name__ == "__main__":
    main()
