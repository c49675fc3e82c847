"""Kernel sweep for the roofline (BASELINE.json configs[4]): block-CSR SpMV and one
PBJ-Chebyshev sweep, FP64, b in {6, 12, 36} x poloidal nodes in {2,000, 8,000} x planes in {16, 64}.

Every point builds a one-level handle on the seeded C4 workload, launches the two kernels through the C ABI with
the library's per-launch CUDA-event profiling on, and reports algorithmic GB/s (traffic.py) and the fraction of
the measured HBM copy rate.  ``bench.py --kernel-sweep`` prints one JSON line per point.
"""
from __future__ import annotations

import gc

from .traffic import LevelSize

L2_BYTES = 126e6


def time_level_kernels(s, level: int, reps: int = 10, nu: int = 4):
    """Mean CUDA-event durations (ms) of the SpMV, full sweep, sweep without d-update and PBJ apply on one
    level of solver ``s``.  One warm-up pass, then ``reps`` event-bracketed passes."""
    import torch
    n = s.n(level)
    g = torch.Generator(device="cpu").manual_seed(1234 + level)
    x = (torch.rand(n, generator=g, dtype=torch.float64) * 2 - 1).to(s.device)
    rhs = (torch.rand(n, generator=g, dtype=torch.float64) * 2 - 1).to(s.device)
    y = s.new(level)
    z = s.new(level)
    out = {}
    for timed in (False, True):
        s.profile_reset()
        s.profile_enable(timed)
        for _ in range(reps if timed else 2):
            s.spmv(level, x, y)
            s.smooth(level, rhs, z, nu, True)      # pbj + (nu-1) full sweeps + 1 sweep without the d-update
        s.profile_enable(False)
        if timed:
            prof = s.profile_get()
            for kind in ("spmv", "sweep", "sweep_nod", "pbj"):
                t = prof.get((level, kind))
                if t and t["timed"]:
                    out[kind] = t["ms"] / t["timed"]
    torch.cuda.synchronize()
    return out


def point_report(name, size: LevelSize, times: dict, peak_gbs: float) -> dict:
    rep = {"point": name, "b": size.b, "n_brows": size.n_brows, "nnzb": size.nnzb,
           "matrix_GB": size.matrix_bytes / 1e9,
           "l2": "L2-resident (excluded from the HBM fraction)" if size.matrix_bytes < L2_BYTES else "larger than L2"}
    for kind, ms in times.items():
        nbytes = size.by_kind(kind)
        gbs = nbytes / ms / 1e6
        rep[kind] = {"us": 1e3 * ms, "bytes": nbytes, "GBps": gbs, "frac_of_measured_peak": gbs / peak_gbs,
                     "frac_of_8TBs_nominal": gbs / 8000.0}
    return rep


def run(peak_gbs: float, points=None, reps: int = 10, shuffled: bool = False, max_gb: float = 50.0):
    """Yield one report dict per C4 point (seeded synthetic matrices; levels = 1)."""
    import torch
    from . import binding
    from .workloads import c4_points, make_workload
    for p in c4_points():
        if points and not any(tok in p["name"] for tok in points):
            continue
        kw = dict(p)
        name = kw.pop("name")
        deg_blocks = 8.9                                    # blocks per row of the stated stencil
        if kw["mesh"][0] * kw["mesh"][1] * kw["n_phi"] * deg_blocks * kw["b"] ** 2 * 8 / 1e9 > max_gb:
            yield {"point": name, "skipped": f"matrix larger than --sweep-max-gb {max_gb:g}"}
            continue
        w = make_workload("C0", shuffle=shuffled, want_rhs=False, **kw)
        rp, ci, va = binding.upload(w)
        s = binding.Solver(rp, ci, va, w.b, w.n_pol, w.n_phi, 1, eig_iters=1)
        try:
            times = time_level_kernels(s, 0, reps=reps)
            size = LevelSize(n_brows=w.n_brows, nnzb=w.nnzb, b=w.b)
            yield point_report(name + ("-shuffled" if shuffled else ""), size, times, peak_gbs)
        finally:
            s.destroy()
            del s, rp, ci, va, w
            gc.collect()
            torch.cuda.empty_cache()


def run_levels(s, peak_gbs: float, reps: int = 10):
    """The same report for every level of an existing hierarchy (the kernels the solve actually runs)."""
    out = []
    for level in range(s.levels):
        g = s.get_level(level)
        size = LevelSize(n_brows=g["n_brows"], nnzb=g["nnzb"], b=s.b)
        out.append(point_report(f"level{level}", size, time_level_kernels(s, level, reps=reps), peak_gbs))
    return out
