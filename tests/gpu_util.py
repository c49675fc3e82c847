"""Shared helpers of the ``-m gpu`` parity tests: build the same seeded workload for the oracle (NumPy) and for
the CUDA library (through the C ABI binding), and compare in the max-norm."""
import numpy as np

from oracle import mg
from paper_2506_16676_b200.workloads import make_workload

# tolerances (BASELINE.json north_star)
TOL_KERNEL = 1e-12   # per-kernel outputs, relative max-norm
TOL_VCYCLE = 1e-10   # one V-cycle application (pinned coarse mode), relative max-norm


def relmax(a, b):
    """max|a - b| / max|b| (b = oracle)."""
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    den = np.abs(b).max() if b.size else 0.0
    if a.size == 0:
        return 0.0
    return float(np.abs(a - b).max() / (den if den > 0 else 1.0))


def small(name="C0", **kw):
    return make_workload(name, **kw)


GPU_ONLY_OPTIONS = ("use_graphs", "kernel_variant", "orth_eta")   # launch mechanics of the CUDA library; no arithmetic meaning


def oracle_hierarchy(w, **opt):
    opt = {k: v for k, v in opt.items() if k not in GPU_ONLY_OPTIONS}
    return mg.setup(w.row_ptr, w.col_idx, w.vals, w.b, w.n_pol, w.n_phi, w.levels, mg.Options(**opt))


def gpu_solver(w, inject_bounds_from=None, **opt):
    """Solver on cuda:0 for workload ``w``; optionally with the oracle hierarchy's Chebyshev bounds injected."""
    from paper_2506_16676_b200 import binding
    rp, ci, va = binding.upload(w)
    s = binding.Solver(rp, ci, va, w.b, w.n_pol, w.n_phi, w.levels, **opt)
    if inject_bounds_from is not None:
        for l, L in enumerate(inject_bounds_from.levels):
            s.set_cheb_bounds(l, L.lam_min, L.lam_max)
    return s


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def to_np(t):
    return t.detach().cpu().numpy()
