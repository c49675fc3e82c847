#!/usr/bin/env python
"""bench.py -- FP64 MG-FGMRES solve time to rtol 1e-8 on one B200 (BASELINE.json metric), with the HBM
roofline of the dominant kernel and the CPU oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C1] [--impl reference]

A STEP is one complete ``mg_solve`` (FGMRES preconditioned by the toroidal semi-coarsening V-cycle, to
rtol 1e-8) of one seeded synthetic right-hand side on the workload BASELINE.json's metric is quoted on
(configs[1] "Medium": 2,000 poloidal nodes x 16 planes, b = 36, 4 levels).  The hierarchy (mg_setup) is built
once, outside the timed region (it is the paper's lagged "refresh"), and reported in ``config``.

* ``value``  = seconds per solve, device time between CUDA events inside the library with the right-hand
  side already resident in HBM (``mg_solve_info.solve_ms``), MAX over ranks.
* ``e2e``    = the same K solves timed around the public host-buffer call ``mg_solve_host`` (pinned host
  rhs -> device, solve, x -> pinned host), CUDA events on the library's stream, MAX over ranks.
* ``roofline`` = the kernel class with the largest share of the step: algorithmic bytes per launch
  (paper_2506_16676_b200/traffic.py) / its mean CUDA-event duration, measured
  in a short event-bracketed pass right after the timed steps, against MEASURED_PEAKS.json's HBM copy rate.
* ``cpu_baseline`` = the oracle (oracle/, as it stands) TIMED on the host cores on bounded units of the same
  workload (fine-level SpMV, one Chebyshev-PBJ sweep, one V-cycle, coarsest-level PBJ-GMRES iterations); the solve
  figure is built from those unit times and iteration counts the ORACLE produced (tests/golden/solve_*.json) and is
  labelled an estimate.  A reported baseline, not the target.
* N > 1: REPLICAS ONLY -- the path does not shard (north_star: one GPU); N independent solves.

``--impl reference`` times the oracle alone (no GPU work) and prints the same line with "impl": "reference".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "mg_fgmres_solve_time_to_rtol_1e-8"
UNIT = "s"
RTOL = 1e-8
# Why the N = 1 line is on configs[1] (C1) and not on the largest single-GPU config (C3, 74 GB hierarchy): the driver times
# 20 complete solves; C3 takes ~150 s per solve in the configs' mode (profiles/r02_configs.md), 20 x 150 s does not fit
# its window.  `bench.py --workload C3` produces the C3 line.
WHY_NOT_LARGEST = ("C3 (largest single-GPU config): ~150 s per default-mode solve (profiles/r02_configs.md), x 20 timed steps "
                   "exceeds the driver's window; bench.py --workload C3 times it")


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------------- helpers
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=open(self.path, "w"),
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        try:
            for line in open(self.path):
                f = [t.strip() for t in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), power_w_max=max(pw), reasons=sorted(reasons),
                       samples=len(sm))
        return out


def measured_traffic(workload: str, level: int, kind: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures
    (profiles/r02_dram_traffic.csv, else round 1's; the commands are in the .md beside each), or None."""
    import csv
    for name in ("r02_dram_traffic.csv", "r01_dram_traffic.csv"):
        path = os.path.join(ROOT, "profiles", name)
        if not os.path.exists(path):
            continue
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and int(row["level"]) == level and row["kind"] == kind:
                    return int(row["dram_bytes_per_launch"])
    return None


def level_sizes(solver):
    from paper_2506_16676_b200.traffic import LevelSize
    out = []
    for l in range(solver.levels):
        g = solver.get_level(l)
        out.append(LevelSize(n_brows=g["n_brows"], nnzb=g["nnzb"], b=solver.b))
    return out


def class_bytes(sizes, level, kind, restart_by_level, direct_bytes: int = 0):
    """Algorithmic bytes of ONE launch of a (level, kind) class (traffic.py)."""
    L = sizes[level]
    if kind == "direct":    # one direct coarsest-level solve: 2 sum n_k^2 doubles + the off-diagonal blocks (mg_direct_info)
        return direct_bytes
    if kind in ("spmv", "resid", "sweep", "sweep_nod", "pbj", "restrict", "prolong"):
        return L.by_kind(kind)
    if kind == "cycle":     # one whole restart cycle of the coarsest-level GMRES: m iterations, j = 0..m-1
        m = restart_by_level.get(level, 1)
        return sum(L.gmres_iteration(j) for j in range(m))
    return 0                # orth / other: sized from the iteration counts (orth_bytes)


# ------------------------------------------------------------------------------------------------- oracle arm
def golden_counts(workload: str):
    """Iteration counts the ORACLE produced for this workload (tests/golden/solve_*.json, written by
    tests/golden/make_solve_goldens.py from oracle/ alone): outer FGMRES iterations of a complete solve with the direct
    coarsest-level solve, and coarsest-level PBJ-GMRES iterations per V-cycle of the configs' own mode.  None if absent."""
    gdir = os.path.join(ROOT, "tests", "golden")
    out = {}
    for key, fname in (("outer", f"solve_{workload}_direct.json"), ("coarse", f"solve_{workload}_default_2its.json"),
                       ("full", f"solve_{workload}_default.json")):
        path = os.path.join(gdir, fname)
        if os.path.exists(path):
            with open(path) as f:
                out[key] = json.load(f)
    if "full" in out:
        g = out["full"]
        return dict(outer_iters=g["iters"], coarse_per_cycle=g["coarse_iters_total"] / max(1, g["iters"]),
                    source=f"tests/golden/solve_{workload}_default.json (complete oracle solve)")
    if "outer" in out and "coarse" in out:
        pc = out["coarse"]["coarse_iters_per_cycle"]
        return dict(outer_iters=out["outer"]["iters"], coarse_per_cycle=sum(pc) / max(1, len(pc)),
                    source=f"outer count: tests/golden/solve_{workload}_direct.json (complete oracle solve, direct coarse solve); "
                           f"coarsest-level iterations per V-cycle: tests/golden/solve_{workload}_default_2its.json (oracle, first "
                           f"{len(pc)} cycles)")
    return None


class OracleUnits:
    """The oracle's hierarchy of one workload and timers for bounded units of its solve."""

    def __init__(self, w):
        from oracle import mg as oracle_mg
        import numpy as np
        self.mg, self.np, self.w = oracle_mg, np, w
        t0 = time.perf_counter()
        # coarse_fixed_sweeps = 0: the V-cycle without its coarsest-level solve (timed separately, per iteration)
        self.H = oracle_mg.setup(w.row_ptr, w.col_idx, w.vals, w.b, w.n_pol, w.n_phi, w.levels,
                                 oracle_mg.Options(coarse_mode=1, coarse_fixed_sweeps=0))
        self.setup_s = time.perf_counter() - t0
        self.threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
        self.rc = np.random.default_rng(7).uniform(-1.0, 1.0, self.H.levels[-1].n)

    def sample(self, coarse_its: int = 40, full: bool = False) -> dict:
        """One timed sample: seconds of each unit (the oracle exactly as the parity tests call it)."""
        mg, H, w = self.mg, self.H, self.w
        L0, Lc = H.levels[0], H.levels[-1]
        out = {}
        t0 = time.perf_counter()
        mg.spmv(L0, w.rhs)
        out["spmv_fine_s"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        mg.vcycle(H, w.rhs)
        out["vcycle_without_coarsest_s"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        _, it, _, _ = mg.fgmres(lambda v: mg.spmv(Lc, v), lambda v: mg.pbj_apply(Lc, v), self.rc, None, 1e-10, 100, coarse_its)
        out["coarse_gmres_iteration_s"] = (time.perf_counter() - t0) / max(1, it)
        out["coarse_gmres_iterations_timed"] = it
        if full:
            t0 = time.perf_counter()
            mg.chebyshev(L0, w.rhs, None, 1)
            out["chebyshev_sweep_fine_s"] = time.perf_counter() - t0
            # the single-thread figure of the fine-level SpMV: OpenMP threads of the oracle's C loops set to 1
            try:
                import ctypes
                omp = ctypes.CDLL("libgomp.so.1")
                nthr = omp.omp_get_max_threads()
                omp.omp_set_num_threads(1)
                t0 = time.perf_counter()
                mg.spmv(L0, w.rhs)
                out["spmv_fine_1_thread_s"] = time.perf_counter() - t0
                omp.omp_set_num_threads(nthr)
            except OSError:
                pass
            H.opt.coarse_fixed_sweeps = 8
            t0 = time.perf_counter()
            mg.vcycle(H, w.rhs)
            out["vcycle_pinned_coarse_mode_s"] = time.perf_counter() - t0
            H.opt.coarse_fixed_sweeps = 0
        return out

    @staticmethod
    def solve_estimate(u: dict, counts: dict) -> float:
        """Seconds of one solve from measured unit times x oracle-counted iterations (the Gram-Schmidt work of the outer
        FGMRES is left out: a lower bound)."""
        per_outer = u["vcycle_without_coarsest_s"] + u["spmv_fine_s"] + counts["coarse_per_cycle"] * u["coarse_gmres_iteration_s"]
        return counts["outer_iters"] * per_outer


def static_config(w, opt: dict, smoother: str = "chebyshev", world: int = 1) -> dict:
    """The part of ``config`` that names the workload and the method: identical in the CUDA and the reference arm."""
    return {"workload": w.name, "n_pol": w.n_pol, "n_phi": w.n_phi, "b": w.b, "levels": w.levels, "unknowns": w.n, "nnzb": w.nnzb,
            "rtol": RTOL,
            "cycle": f"V({opt['nu_pre']},{opt['nu_post']}) " + {"gmres": "PBJ-GMRES smoother (the paper's, PAPER.md:95)",
                                                                "line": "toroidal-line block-Jacobi Chebyshev (NEXT-4, PAPER.md:212-214)"
                                                                }.get(smoother, "PBJ-Chebyshev"),
            "coarsest": ("direct (block-tridiagonal Schur inverses)" if opt["coarse_mode"] == 2 else
                         f"PBJ-GMRES({opt['coarse_restart']}) to {opt['coarse_rtol']:g}"),
            "fgmres_restart": opt["restart"], "parallelism": "replicas only" if world > 1 else "1 GPU",
            "why_not_largest": WHY_NOT_LARGEST if w.name == "C1" else None}


def reference_arm(args):
    """The oracle alone on the host cores: each step is one bounded sample of the workload (fine-level SpMV, V-cycle without
    its coarsest-level solve, 40 coarsest-level PBJ-GMRES iterations); ``value`` is the solve time these unit times give with
    the oracle's own iteration counts -- an estimate, labelled so; nothing here comes from a GPU run."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2506_16676_b200.workloads import make_workload
    from oracle import mg as oracle_mg
    oracle_mg.build()
    w = make_workload(args.workload)
    units = OracleUnits(w)
    counts = golden_counts(args.workload)
    o = oracle_mg.Options()
    opt = dict(nu_pre=o.nu_pre, nu_post=o.nu_post, restart=o.restart, coarse_restart=o.coarse_restart, coarse_rtol=o.coarse_rtol,
               coarse_mode=0)
    for _ in range(args.warmup):
        units.sample(args.ref_coarse_its)
    vals, samples = [], []
    t0 = time.perf_counter()
    for _ in range(args.steps):
        u = units.sample(args.ref_coarse_its)
        samples.append(u)
        if counts:
            vals.append(units.solve_estimate(u, counts))
    wall = time.perf_counter() - t0
    value = sum(vals) / len(vals) if vals else None
    mean = {k: sum(u[k] for u in samples) / len(samples) for k in samples[0]}
    sample = (f"each step: 1 fine-level block SpMV + 1 V-cycle without its coarsest-level solve + "
              f"{int(mean['coarse_gmres_iterations_timed'])} coarsest-level PBJ-GMRES iterations of the oracle on {w.name} "
              f"({wall / max(1, args.steps):.1f} s of CPU work per step); value = ESTIMATE of one solve = oracle-counted iterations x "
              f"these measured unit times" + (f" [{counts['source']}: {counts['outer_iters']} outer, "
                                              f"{counts['coarse_per_cycle']:.0f} coarsest-level iterations per V-cycle]" if counts else
                                              " [no oracle iteration counts for this workload: no estimate]"))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": (1e3 * value) if value is not None else None,
            "sample_ms_per_step": 1e3 * wall / max(1, args.steps), "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": static_config(w, opt),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": units.threads, "kind": "oracle", "estimate": True,
                             "sample": sample, "measured": mean, "oracle_setup_s": units.setup_s},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def orth_bytes(iters, restart, vec_bytes):
    """Algorithmic CGS2 traffic of ``iters`` Arnoldi steps of GMRES(restart): step j must read V_0..V_j once (the fused
    kernel keeps the slices on chip for the second pass) plus a few passes over w."""
    full, rem = divmod(int(iters), int(restart))
    cyc = sum((j + 1) + 8 for j in range(restart))
    return (full * cyc + sum((j + 1) + 8 for j in range(rem))) * vec_bytes


def solve_bytes_from_counts(sizes, outer_iters, coarse_iters, opt, dram_true: bool = False, direct_bytes: int = 0):
    """Algorithmic bytes of one solve from its iteration counts.  dram_true: the fused coarse GMRES multiplies by the
    precomputed A D^-1 and never reads D^-1 (SURVEY's byte model charges it to every coarse iteration).  direct_bytes: bytes of
    one direct coarsest-level solve (coarse_mode 2)."""
    from paper_2506_16676_b200.traffic import vcycle_bytes
    L0, Lc = sizes[0], sizes[-1]
    outer = outer_iters * (vcycle_bytes(sizes, opt["nu_pre"], opt["nu_post"]) + L0.spmv() + direct_bytes) + \
        orth_bytes(outer_iters, opt["restart"], L0.vec_bytes)
    coarse = coarse_iters * (Lc.spmv() + (0 if dram_true else Lc.pbj())) + orth_bytes(coarse_iters, opt["coarse_restart"], Lc.vec_bytes)
    return outer + coarse


# ------------------------------------------------------------------------------------------------- CUDA arm
def cuda_arm(args):
    import numpy as np
    import torch
    from paper_2506_16676_b200 import binding, buildlib, replicas
    from paper_2506_16676_b200.workloads import make_workload

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(replicas.env_world()[1])     # before the process group: NCCL binds to the current device
    rank, local_rank, world = replicas.init("nccl")
    if world != args.gpus:
        log(f"note: --gpus {args.gpus} but WORLD_SIZE {world}; using WORLD_SIZE")
    dev = torch.device("cuda", local_rank)
    buildlib.build()

    t0 = time.perf_counter()
    w = make_workload(args.workload, **({"levels": args.levels} if args.levels > 0 else {}))
    gen_s = time.perf_counter() - t0
    rp, ci, va = binding.upload(w, dev)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    extra = {}
    if args.smoother == "gmres":
        extra["smoother"] = 1
    if args.smoother == "line":
        extra["smoother"] = 2
    if args.nu > 0:
        extra.update(nu_pre=args.nu, nu_post=args.nu)
    if args.coarse_mode >= 0:
        extra["coarse_mode"] = args.coarse_mode
    s = binding.Solver(rp, ci, va, w.b, w.n_pol, w.n_phi, w.levels, **extra)
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    # refresh cost (Table 4 reports setup per refresh): numeric-only rebuild of the hierarchy
    t0 = time.perf_counter()
    s.update_values(va)
    torch.cuda.synchronize()
    refresh_s = time.perf_counter() - t0
    if args.max_outer > 0:
        s.update_options(maxit=args.max_outer)
    opt = {k: getattr(s.opt, k) for k in ("nu_pre", "nu_post", "restart", "maxit", "coarse_restart", "coarse_rtol", "coarse_mode")}
    sizes = level_sizes(s)
    n = w.n
    rhs_h = torch.from_numpy(w.rhs.copy()).pin_memory()
    x_h = torch.empty(n, dtype=torch.float64).pin_memory()
    if rank == 0:
        log(f"[bench] workload {w.name}: n = {n}, nnzb = {w.nnzb}, levels = {w.levels}, generate {gen_s:.1f} s, "
            f"mg_setup {setup_s:.2f} s, hierarchy {s.device_bytes() / 1e9:.2f} GB (+ fine matrix {va.numel() * 8 / 1e9:.2f} GB)")

    info = None
    # Warm-up steps run the same call on the same inputs; by default each is cut after --warmup-outer outer FGMRES
    # iterations (every kernel, every level, the coarse-cycle CUDA graph and ~5,000 coarse iterations per outer
    # iteration are exercised; a full C1 solve takes minutes and three of them would only repeat that).  The timed
    # steps are always complete solves.  --warmup-outer 0 makes the warm-ups complete solves too.
    if args.warmup_outer > 0 and args.max_outer <= 0:
        s.update_options(maxit=args.warmup_outer)
    for i in range(args.warmup):
        _, info = s.solve_host(rhs_h, x_h, rtol=RTOL)
        if rank == 0:
            log(f"[bench] warm-up {i}: {info['solve_ms'] / 1e3:.2f} s, {info['iters']} its, rel_res {info['rel_res']:.2e}")
    if args.warmup_outer > 0 and args.max_outer <= 0:
        s.update_options(maxit=opt["maxit"])

    replicas.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    s.profile_reset()
    launches0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dev_ms = 0.0
    e0.record()
    for _ in range(args.steps):
        _, info = s.solve_host(rhs_h, x_h, rtol=RTOL)
        dev_ms += info["solve_ms"]
    e1.record()
    torch.cuda.synchronize()
    replicas.barrier()
    e2e_ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = s.launch_count() - launches0
    counts = s.profile_get()
    if args.max_outer <= 0 and (not info["converged"] or not (info["rel_res"] <= 1.05 * RTOL)):
        raise SystemExit(f"bench.py: solve did not reach rtol: {info}")
    x_dev_check = float(np.abs(x_h.numpy()).max())
    t_dev = replicas.max_over_ranks(dev_ms / args.steps / 1e3, dev)
    t_e2e = replicas.max_over_ranks(e2e_ms / args.steps / 1e3, dev)

    # ---- roofline: a short event-bracketed pass (same inputs, a few outer iterations) gives mean kernel durations
    peak, peak_src = measured_peaks()
    roof, detail, cpu, vcycle_roof, direct = None, [], None, None, None
    if rank == 0:
        dinfo = s.direct_info() if opt["coarse_mode"] == 2 else None
        direct_bytes = dinfo["bytes_per_solve"] if dinfo else 0
        # (launch-chain fallback of the direct solve: hundreds of launches per solve are booked under "direct", no per-launch size)
        direct_launch_bytes = direct_bytes if dinfo and dinfo["persistent"] else 0
        s.update_options(maxit=min(opt["maxit"], 2))
        s.profile_reset()
        s.profile_enable(True)
        s.solve_host(rhs_h, x_h, rtol=RTOL)
        s.profile_enable(False)
        timed = s.profile_get()
        s.update_options(maxit=opt["maxit"])
        restart_by_level = {s.levels - 1: opt["coarse_restart"]}
        for (level, kind), c in counts.items():
            t = timed.get((level, kind))
            if not t or not t["timed"]:
                continue
            mean_ms = t["ms"] / t["timed"]
            per_step_launches = c["launches"] / args.steps
            nbytes = class_bytes(sizes, level, kind, restart_by_level, direct_launch_bytes)
            share_ms = per_step_launches * mean_ms
            detail.append({"level": level, "kind": kind, "launches_per_step": per_step_launches, "mean_us": 1e3 * mean_ms,
                           "bytes_per_launch": nbytes, "GBps": (nbytes / mean_ms / 1e6) if nbytes else None,
                           "frac": (nbytes / mean_ms / 1e6 / peak) if nbytes else None, "ms_per_step": share_ms})
        detail.sort(key=lambda d: -d["ms_per_step"])
        for d in detail:
            d["share_of_step"] = d["ms_per_step"] / (1e3 * t_dev)
        top = next((d for d in detail if d["bytes_per_launch"]), None)
        if top:
            what = ("direct coarsest-level solve (direct_solve_persistent_kernel)" if top["kind"] == "direct" else
                    f"bsr kernel, kind {top['kind']}, level {top['level']}")
            roof = {"bound": "hbm", "kernel": what, "achieved": top["GBps"],
                    "peak": peak, "unit": "GB/s", "frac": top["frac"],
                    "traffic": measured_traffic(w.name, top["level"], top["kind"]), "peak_source": peak_src,
                    "bytes_per_launch": top["bytes_per_launch"], "mean_us": top["mean_us"],
                    "share_of_step": top["share_of_step"], "frac_of_8TBs_nominal": top["GBps"] / 8000.0}
        # ---- V-cycle roofline, reported twice: (i) one mg_vcycle in the pinned coarse mode (coarsest level = 8
        # Chebyshev-PBJ sweeps: every byte is a smoother/transfer byte), CUDA events around 5 calls; (ii) the complete
        # outer iteration of the timed solve (V-cycle with its measured coarse GMRES steps + SpMV + CGS2).
        from paper_2506_16676_b200.traffic import vcycle_bytes
        s.update_options(coarse_mode=1)
        rv = torch.from_numpy(w.rhs).to(dev)
        zv = s.new()
        for _ in range(2):
            s.vcycle(rv, zv)
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0.record()
        for _ in range(5):
            s.vcycle(rv, zv)
        v1.record()
        torch.cuda.synchronize()
        s.update_options(coarse_mode=opt["coarse_mode"])
        vc_ms = v0.elapsed_time(v1) / 5
        vc_bytes = vcycle_bytes(sizes, opt["nu_pre"], opt["nu_post"], coarse_sweeps=s.opt.coarse_fixed_sweeps)
        solve_bytes = solve_bytes_from_counts(sizes, info["iters"], info["coarse_iters_total"], opt, direct_bytes=direct_bytes)
        solve_bytes_dram = solve_bytes_from_counts(sizes, info["iters"], info["coarse_iters_total"], opt, dram_true=True,
                                                   direct_bytes=direct_bytes)
        vcycle_roof = None if args.smoother != "chebyshev" else {   # the byte model below is the PBJ-Chebyshev cycle's
            "pinned_coarse_mode": {"ms": vc_ms, "bytes": vc_bytes, "GBps": vc_bytes / vc_ms / 1e6,
                                   "frac_of_measured_peak": vc_bytes / vc_ms / 1e6 / peak, "frac_of_8TBs_nominal": vc_bytes / vc_ms / 1e6 / 8000.0},
            "complete_outer_iteration": {"ms": 1e3 * t_dev / max(1, info["iters"]), "bytes": solve_bytes / max(1, info["iters"]),
                                         "GBps": solve_bytes / t_dev / 1e9, "frac_of_measured_peak": solve_bytes / t_dev / 1e9 / peak,
                                         "frac_of_8TBs_nominal": solve_bytes / t_dev / 1e9 / 8000.0,
                                         "coarse_steps_per_cycle": info["coarse_iters_total"] / max(1, info["iters"]),
                                         "byte_model": "SURVEY 8d: every coarsest-level iteration charged A + D^-1"},
            # what DRAM really moves: the fused coarse GMRES multiplies by the precomputed A D^-1 and never reads D^-1
            "complete_outer_iteration_dram_true": {"bytes": solve_bytes_dram / max(1, info["iters"]), "GBps": solve_bytes_dram / t_dev / 1e9,
                                                   "frac_of_measured_peak": solve_bytes_dram / t_dev / 1e9 / peak,
                                                   "frac_of_8TBs_nominal": solve_bytes_dram / t_dev / 1e9 / 8000.0}}
        # ---- the same solve with the paper's kind of coarsest-level solver (direct, NEXT-2): reported beside the metric,
        # which keeps the configs' PBJ-GMRES coarse solve
        direct = None
        if opt["coarse_mode"] == 0 and args.max_outer <= 0 and not args.no_direct:
            try:
                s.update_options(coarse_mode=2)
                t0d = time.perf_counter()
                s.solve_host(rhs_h, x_h, rtol=RTOL)           # first call builds the dense Schur inverses
                torch.cuda.synchronize()
                first_s = time.perf_counter() - t0d
                _, info_d = s.solve_host(rhs_h, x_h, rtol=RTOL)
                di = s.direct_info()
                # the coarsest-level solve alone: CUDA events around 20 back-to-back calls
                rc = torch.rand(s.n(s.levels - 1), dtype=torch.float64, device=dev) * 2 - 1
                ec = s.new(s.levels - 1)
                for _ in range(3):
                    s.coarse_solve(rc, ec)
                c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                c0.record()
                for _ in range(20):
                    s.coarse_solve(rc, ec)
                c1.record()
                torch.cuda.synchronize()
                cs_ms = c0.elapsed_time(c1) / 20
                direct = {"value": info_d["solve_ms"] / 1e3, "unit": UNIT, "outer_iters": info_d["iters"], "rel_res": info_d["rel_res"],
                          "converged": info_d["converged"], "factorisation_s": max(0.0, first_s - info_d["solve_ms"] / 1e3),
                          "coarse_solve": {"us": 1e3 * cs_ms, "bytes": di["bytes_per_solve"], "GBps": di["bytes_per_solve"] / cs_ms / 1e6,
                                           "frac_of_measured_peak": di["bytes_per_solve"] / cs_ms / 1e6 / peak,
                                           "level_sets": di["level_sets"], "dense_GB": di["dense_bytes"] / 1e9,
                                           "persistent_kernel": di["persistent"]},
                          "what": "mg_options.coarse_mode = 2: block-tridiagonal direct solve of the coarsest level "
                                  "(the paper solves its coarsest level by LU, PAPER.md:374-381); not the metric's configuration"}
            except Exception as exc:   # e.g. not enough memory for the dense blocks
                direct = {"unavailable": str(exc)}
            finally:
                s.update_options(coarse_mode=opt["coarse_mode"])
        # ---- oracle timed beside it (rank 0, N = 1 only): bounded units of the same workload on the host cores
        if world == 1 and not args.no_cpu_baseline:
            units = OracleUnits(w)
            u = units.sample(args.ref_coarse_its, full=True)
            gc_ = golden_counts(w.name) if opt["coarse_mode"] == 0 and args.smoother == "chebyshev" and args.levels <= 0 else None
            est = units.solve_estimate(u, gc_) if gc_ else None
            cpu = {"value": est, "unit": UNIT, "cores": units.threads, "kind": "oracle", "estimate": True, "measured": u,
                   "oracle_setup_s": units.setup_s,
                   "sample": (f"oracle units timed on {w.name}: fine-level block SpMV, one Chebyshev-PBJ sweep, one V-cycle (pinned "
                              f"coarse mode and without the coarsest level), {u['coarse_gmres_iterations_timed']} coarsest-level "
                              f"PBJ-GMRES iterations; value = ESTIMATE of one solve = oracle-counted iterations x these unit times"
                              + (f" [{gc_['source']}: {gc_['outer_iters']} outer, {gc_['coarse_per_cycle']:.0f} coarsest-level "
                                 f"iterations per V-cycle]" if gc_ else " [no oracle iteration counts for this configuration: no estimate]"))}

    if rank == 0:
        cfg = static_config(w, opt, args.smoother, world)
        cfg["l2"] = ("inputs larger than L2 (every level's matrix >= 0.5 GB vs 126 MB L2)" if sizes[-1].matrix_bytes > 2.6e8
                     else "coarsest level fits L2: not an HBM-roofline workload")
        cfg["warmup_steps"] = (f"{args.warmup} x the first {args.warmup_outer} outer iterations of the same solve"
                               if args.warmup_outer > 0 and args.max_outer <= 0 else f"{args.warmup} x complete solves")
        line = {"metric": METRIC, "value": t_dev, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * t_dev, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": cfg,
                "solve": {"outer_iters": info["iters"], "coarse_iters": info["coarse_iters_total"], "rel_res": info["rel_res"],
                          "max_abs_x": x_dev_check, "setup_s": setup_s, "refresh_s": refresh_s,
                          "hierarchy_GB": s.device_bytes() / 1e9, "fine_matrix_GB": va.numel() * 8 / 1e9},
                "e2e": {"value": t_e2e, "unit": UNIT, "h2d_bytes_per_step": 8 * n, "d2h_bytes_per_step": 8 * n},
                "gpu_launches": launches, "clocks": clocks, "roofline": roof, "vcycle_roofline": vcycle_roof, "direct_coarse_solve": direct, "cpu_baseline": cpu,
                "throughput": {"value": world / t_dev, "unit": "solves/s"}, "truncated": args.max_outer > 0,
                "kernels": detail[:12]}
        print(json.dumps(line), flush=True)
    s.destroy()
    replicas.finalize()
    return 0


def kernel_sweep_arm(args):
    """configs[4] "Kernel sweep for the roofline": GB/s and fraction of the HBM peak per point."""
    import torch
    from paper_2506_16676_b200 import buildlib, kernel_sweep
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(0)
    buildlib.build()
    peak, peak_src = measured_peaks()
    for rep in kernel_sweep.run(peak, points=args.kernel_sweep or None, reps=max(3, args.steps),
                                shuffled=args.sweep_shuffled, max_gb=args.sweep_max_gb):
        rep.update(peak_GBps=peak, peak_source=peak_src, dtype="f64", data="synthetic")
        print(json.dumps(rep), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["cuda", "reference"], default="cuda")
    ap.add_argument("--workload", default="C1", help="C1 (the metric's config, default); C0, C2-16/32/64, C3, C3b for other configs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-coarse-its", type=int, default=40,
                    help="coarsest-level PBJ-GMRES iterations in one timed oracle sample (cpu_baseline / --impl reference)")
    ap.add_argument("--no-direct", action="store_true", help="skip the extra solve with the direct coarsest-level solver")
    ap.add_argument("--max-outer", type=int, default=0,
                    help="profiling aid (ncu launch lists): cap the outer FGMRES iterations of every solve; the line is then "
                         "marked \"truncated\": true and is NOT a bench value")
    ap.add_argument("--smoother", choices=["chebyshev", "gmres", "line"], default="chebyshev",
                    help="level smoother: PBJ-Chebyshev (default, the metric's configuration), the paper's PBJ-GMRES (NEXT-1) or "
                         "toroidal-line block-Jacobi Chebyshev (NEXT-4)")
    ap.add_argument("--levels", type=int, default=0,
                    help="override the number of MG levels of the workload (e.g. 5 on C1: coarsen to 1 plane as the paper does, "
                         "PAPER.md:181); not the metric's configuration")
    ap.add_argument("--coarse-mode", type=int, default=-1,
                    help="override the coarsest-level solver: 0 PBJ-GMRES to 1e-10 (the configs'; default), 2 direct "
                         "(block-tridiagonal Schur inverses, NEXT-2); not the metric's configuration")
    ap.add_argument("--nu", type=int, default=0, help="smoothing steps pre and post (default: the library's 2)")
    ap.add_argument("--warmup-outer", type=int, default=4,
                    help="outer FGMRES iterations of each warm-up step (default 4, about 2.5 s on C1); 0 = complete solves")
    ap.add_argument("--kernel-sweep", nargs="*", default=None, metavar="TOKEN",
                    help="configs[4]: time the block SpMV and one PBJ-Chebyshev sweep on the C4 points (all, or those whose "
                         "name contains a TOKEN, e.g. b36 n2000-p16) and print one JSON line per point instead of the solve line")
    ap.add_argument("--sweep-max-gb", type=float, default=50.0, help="skip C4 points whose matrix exceeds this size")
    ap.add_argument("--sweep-shuffled", action="store_true", help="C4 'shuffled' variant: permuted node numbering")
    args = ap.parse_args()
    if args.kernel_sweep is not None:
        return kernel_sweep_arm(args)
    if args.steps < 1 or args.warmup < 0:
        ap.error("--steps >= 1 and --warmup >= 0")
    return reference_arm(args) if args.impl == "reference" else cuda_arm(args)


if __name__ == "__main__":
    sys.exit(main())
