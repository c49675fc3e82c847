"""GPU parity of the lagged preconditioner ("the preconditioner is lagged",
refresh cost PAPER.md:185-192): mg_update_values (refresh values, keep patterns) and mg_set_operator (solve a new
matrix with the old hierarchy).

A "new Jacobian" is emulated by the generator with the same mesh/pattern and slightly different coefficients
(sigma, beta), as consecutive time steps of the application would give."""
import numpy as np
import pytest
import torch

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from gpu_util import TOL_KERNEL, relmax, small, oracle_hierarchy, gpu_solver, to_dev, to_np

pytestmark = pytest.mark.gpu

BASE = dict(mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77)


def two_steps(**kw):
    args = dict(BASE)
    args.update(kw)
    w0 = small("C0", **args)
    w1 = small("C0", sigma=2e-3, beta=0.12, **args)      # same seed => same mesh, pattern and noise; new coefficients
    assert np.array_equal(w0.row_ptr, w1.row_ptr) and np.array_equal(w0.col_idx, w1.col_idx)
    return w0, w1


@pytest.mark.parametrize("b", [12, 36])
def test_refresh_equals_a_fresh_setup(b):
    kw = dict(b=b, mesh=(3, 10)) if b == 36 else {}
    w0, w1 = two_steps(**kw)
    H1 = oracle_hierarchy(w1)
    s = gpu_solver(w0)
    fresh = gpu_solver(w1)
    try:
        v1 = torch.from_numpy(w1.vals.reshape(-1)).cuda()
        s.update_values(v1)
        for l, L in enumerate(H1.levels):
            g, f = s.level_arrays(l), fresh.level_arrays(l)
            assert np.array_equal(g["col_idx"], L.col_idx) and np.array_equal(g["row_ptr"], L.row_ptr)
            assert np.array_equal(g["vals"], f["vals"]) and np.array_equal(g["dinv"], f["dinv"])   # same kernels, same bits
            assert g["rho_est"] == f["rho_est"] and g["lam_max"] == f["lam_max"]
            assert relmax(g["vals"], L.vals) <= TOL_KERNEL and relmax(g["dinv"], L.dinv) <= 1e-11
        r = input_vector(w1.n, 5, 21)
        for sol in (s, fresh):
            sol.update_options(coarse_mode=1)
        assert np.array_equal(to_np(s.vcycle(to_dev(r))), to_np(fresh.vcycle(to_dev(r))))
        # default coarse mode after a refresh: the precomputed A D^-1 of the coarsest level was refreshed too
        s.update_options(coarse_mode=0)
        Lc = H1.levels[-1]
        rc = input_vector(Lc.n, 5, 23)
        e, it = s.coarse_solve(to_dev(rc))
        assert np.linalg.norm(rc - mg.spmv(Lc, to_np(e))) <= 1.01e-10 * np.linalg.norm(rc)
    finally:
        s.destroy()
        fresh.destroy()


def test_lagged_solve_matches_the_oracle():
    """Solve A_1 x = b with the hierarchy of A_0 (pinned coarse mode: a fixed linear preconditioner)."""
    w0, w1 = two_steps()
    H0 = oracle_hierarchy(w0, coarse_mode=1)
    L1 = mg.Level(n_phi=w1.n_phi, n_pol=w1.n_pol, b=w1.b, row_ptr=w1.row_ptr, col_idx=w1.col_idx, vals=w1.vals)
    x_or, it_or, conv_or, hist_or = mg.fgmres(lambda v: mg.spmv(L1, v), lambda v: mg.vcycle(H0, v), w1.rhs, None, 1e-8,
                                              H0.opt.restart, H0.opt.maxit)
    s = gpu_solver(w0, inject_bounds_from=H0, coarse_mode=1)
    try:
        v1 = torch.from_numpy(w1.vals.reshape(-1)).cuda()
        s.set_operator(v1)
        x, info = s.solve(to_dev(w1.rhs), rtol=1e-8, hist_cap=512)
        assert conv_or and info["converged"] and abs(info["iters"] - it_or) <= 1
        k = min(len(hist_or), len(info["hist"]))
        assert np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k]))).max() <= 0.05
        true_rel = np.linalg.norm(w1.rhs - mg.spmv(L1, to_np(x))) / np.linalg.norm(w1.rhs)      # residual of the NEW matrix
        assert true_rel <= 1.05e-8 and info["rel_res"] == pytest.approx(true_rel, rel=1e-3)
        # back to the hierarchy's own matrix
        s.set_operator(None)
        x0, info0 = s.solve(to_dev(w0.rhs), rtol=1e-8)
        L0 = H0.levels[0]
        assert np.linalg.norm(w0.rhs - mg.spmv(L0, to_np(x0))) <= 1.05e-8 * np.linalg.norm(w0.rhs)
    finally:
        s.destroy()


def test_refresh_with_one_level_rebuilds_the_captured_coarse_cycle():
    """levels = 1: the coarsest level IS level 0, whose values pointer is borrowed; mg_update_values with a NEW buffer must not
    leave the captured CUDA graph of the coarse GMRES cycle pointing at the old one."""
    import torch
    w = small("C0", mesh=(3, 8), n_phi=4, levels=1, b=6, seed=91)
    H = oracle_hierarchy(w)
    s = gpu_solver(w, inject_bounds_from=H)
    try:
        r = input_vector(w.n, 91, 24)
        z1 = to_np(s.vcycle(to_dev(r)))                       # captures the graph on the first buffer
        assert np.linalg.norm(r - mg.spmv(H.levels[0], z1)) <= 1.01e-10 * np.linalg.norm(r)
        vals2 = (s.vals * 2.0).clone()                        # a new buffer with A' = 2 A
        old = s.vals
        s.update_values(vals2)
        old.zero_()                                           # the old buffer must not be read any more
        z2 = to_np(s.vcycle(to_dev(r)))
        assert np.linalg.norm(r - 2.0 * mg.spmv(H.levels[0], z2)) <= 1.01e-10 * np.linalg.norm(r)
    finally:
        s.destroy()


def test_changing_restart_and_maxit_does_not_leak_device_memory():
    """Every change of restart / maxit used to allocate a new Krylov basis and keep the old one until mg_destroy."""
    w = small("C0", mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77)
    s = gpu_solver(w, coarse_mode=1)
    try:
        rhs = to_dev(w.rhs)
        s.update_options(restart=20, maxit=30)
        s.solve(rhs, rtol=1e-8)
        base = s.device_bytes()
        for restart, maxit in ((10, 15), (20, 30), (20, 40), (35, 40), (20, 30)):
            s.update_options(restart=restart, maxit=maxit)
            s.solve(rhs, rtol=1e-8)
        assert s.device_bytes() == base
    finally:
        s.destroy()


def test_misaligned_and_wrong_size_vectors_are_rejected():
    import torch
    from paper_2506_16676_b200 import binding
    w = small("C0", mesh=(3, 8), n_phi=4, levels=2, b=6, seed=92)
    s = gpu_solver(w)
    try:
        buf = torch.zeros(w.n + 1, dtype=torch.float64, device="cuda")
        good = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        with pytest.raises(binding.MgError) as e:
            s.spmv(0, buf[1:], good)                          # 8-byte, not 16-byte aligned
        assert e.value.code == binding.MG_EINVAL
        with pytest.raises((binding.MgError, ValueError, TypeError)):
            s.spmv(0, buf[: w.n - 2], good)                    # too short
    finally:
        s.destroy()
