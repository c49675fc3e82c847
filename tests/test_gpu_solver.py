"""GPU parity of the iterations: V-cycle, coarsest-level solve, FGMRES solve (through the C ABI) vs the oracle.

Bars (BASELINE.json north_star): one V-cycle application within 1e-10 relative
(max-norm) in the pinned coarse mode (a fixed polynomial), and in the default mode in the residual sense;
FGMRES iteration counts to rtol 1e-8 equal or within +-1, residual histories within a 0.05-decade band."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from gpu_util import TOL_VCYCLE, relmax, small, oracle_hierarchy, gpu_solver, to_dev, to_np

pytestmark = pytest.mark.gpu

CASES = {
    "C0-b36": dict(name="C0"),
    "b12-3lev": dict(name="C0", mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77),
    "b6-4lev": dict(name="C0", mesh=(6, 20), n_phi=16, levels=4, b=6, seed=78),
    "b5-generic-to-1-plane": dict(name="C0", mesh=(3, 8), n_phi=4, levels=3, b=5, seed=79),
    # b = 36 at small size: the TMA-ring kernel, GMRES on the precomputed A D^-1 and the fused CGS2 (the bench path)
    "b36-3lev": dict(name="C0", mesh=(3, 10), n_phi=8, levels=3, seed=85),
}


def make(case, **opt):
    kw = dict(CASES[case])
    w = small(kw.pop("name"), **kw)
    H = oracle_hierarchy(w, **opt)
    s = gpu_solver(w, inject_bounds_from=H, **opt)
    return w, H, s


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("nu", [(2, 2), (1, 1), (0, 1), (3, 0)])
def test_vcycle_pinned_coarse_mode(case, nu):
    """coarse_mode = 1: the coarsest level is 8 Chebyshev-PBJ sweeps, so M is a fixed linear operator."""
    w, H, s = make(case, coarse_mode=1, nu_pre=nu[0], nu_post=nu[1])
    try:
        r = input_vector(w.n, w.seed, 21)
        z_or = mg.vcycle(H, r)
        z = to_np(s.vcycle(to_dev(r)))
        assert relmax(z, z_or) <= TOL_VCYCLE
    finally:
        s.destroy()


@pytest.mark.parametrize("case", ["b12-3lev", "b6-4lev", "b5-generic-to-1-plane", "b36-3lev"])
def test_vcycle_default_mode_residual_sense(case):
    """PBJ-GMRES coarse solve on both sides, coarse_rtol tightened to 1e-13: the cycles agree in the residual
    sense ||A (z_gpu - z_or)||_inf / ||r||_inf <= 1e-8 (the coarse corrections agree only to cond * rtol)."""
    w, H, s = make(case, coarse_rtol=1e-13)
    try:
        r = input_vector(w.n, w.seed, 22)
        z_or = mg.vcycle(H, r)
        z = to_np(s.vcycle(to_dev(r)))
        diff = mg.spmv(H.levels[0], z - z_or)
        assert np.abs(diff).max() / np.abs(r).max() <= 1e-8
    finally:
        s.destroy()


@pytest.mark.parametrize("case", ["b12-3lev", "b6-4lev", "b5-generic-to-1-plane", "b36-3lev"])
@pytest.mark.parametrize("graphs,eta", [(1, 0.25), (0, 0.25), (1, 0.0)])
def test_coarse_solve(case, graphs, eta):
    """PBJ-GMRES(100) to 1e-10 on the coarsest level: both reach the tolerance; the solutions agree to
    cond * rtol.  The inner iteration COUNT is not a north_star parity quantity (its +-1 is for the outer FGMRES) and a
    restarted GMRES near stagnation amplifies rounding differences between Gram-Schmidt variants (CPU and
    GPU counts of the same solver differ), so it is held to a 5 % band -- measured in round 2 with classical Gram-Schmidt
    + reorthogonalisation on every step (orth_eta = 0) and with selective reorthogonalisation (0.25) alike: 2959 / 2960 vs
    2958 (oracle, MGS), 1944 vs 1944, 69 vs 69, 3865 / 3881 vs 3894.  (Round 1 had widened the band to 15 % after a
    3296 vs 3076 mismatch of an earlier kernel; the 5 % band is restored.)"""
    w, H, s = make(case, use_graphs=graphs, orth_eta=eta)
    try:
        Lc = H.levels[-1]
        r = input_vector(Lc.n, w.seed, 23)
        e_or = mg.coarse_solve(H, r)
        it_or = H.coarse_iters_last
        e, it = s.coarse_solve(to_dev(r))
        e = to_np(e)
        rn = np.linalg.norm(r)
        assert np.linalg.norm(r - mg.spmv(Lc, e)) <= 1.01e-10 * rn       # the device solve met its tolerance
        assert np.linalg.norm(r - mg.spmv(Lc, e_or)) <= 1.01e-10 * rn
        assert np.linalg.norm(mg.spmv(Lc, e - e_or)) <= 2.1e-10 * rn
        print(f"coarse iterations: device {it} (orth_eta {eta}), oracle {it_or}")
        assert abs(it - it_or) <= max(2, int(0.05 * it_or))
    finally:
        s.destroy()


@pytest.mark.parametrize("case", ["b12-3lev", "b6-4lev", "b5-generic-to-1-plane", "b36-3lev"])
def test_solve_iteration_count_and_history(case):
    w, H, s = make(case)
    try:
        x_or, it_or, conv_or, hist_or = mg.solve(H, w.rhs, 1e-8)
        x, info = s.solve(to_dev(w.rhs), rtol=1e-8, hist_cap=512)
        x = to_np(x)
        assert conv_or and info["converged"]
        assert abs(info["iters"] - it_or) <= 1
        # the estimate equals the true residual (right preconditioning) and the true residual met rtol
        true_rel = np.linalg.norm(w.rhs - mg.spmv(H.levels[0], x)) / np.linalg.norm(w.rhs)
        assert true_rel <= 1.05e-8
        assert info["rel_res"] == pytest.approx(true_rel, rel=1e-3)
        assert info["hist"][-1] == pytest.approx(true_rel, rel=1e-3)
        k = min(len(hist_or), len(info["hist"]))
        band = np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k])))
        assert band.max() <= 0.05
        # both approximate A^-1 b to rtol: the solutions agree to cond-scaled rtol in the residual sense
        assert np.linalg.norm(mg.spmv(H.levels[0], x - x_or)) <= 2.1e-8 * np.linalg.norm(w.rhs)
    finally:
        s.destroy()


def test_solve_pinned_mode_C0_full_size():
    """Config 0 at full size, pinned coarse mode (fixed polynomial cycle => linear preconditioner)."""
    w, H, s = make("C0-b36", coarse_mode=1)
    try:
        x_or, it_or, conv_or, hist_or = mg.solve(H, w.rhs, 1e-8)
        x, info = s.solve(to_dev(w.rhs), rtol=1e-8, hist_cap=512)
        assert conv_or == info["converged"]
        assert abs(info["iters"] - it_or) <= 1
        k = min(len(hist_or), len(info["hist"]))
        assert np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k]))).max() <= 0.05
    finally:
        s.destroy()


def test_solve_host_buffers_and_initial_guess():
    import torch
    w, H, s = make("b6-4lev")
    try:
        rhs_h = torch.from_numpy(w.rhs.copy()).pin_memory()
        x_h = torch.empty_like(rhs_h).pin_memory()
        _, info = s.solve_host(rhs_h, x_h, rtol=1e-8)
        assert info["converged"]
        x = x_h.numpy()
        assert np.linalg.norm(w.rhs - mg.spmv(H.levels[0], x)) <= 1.05e-8 * np.linalg.norm(w.rhs)
        # restart from the converged solution: zero further iterations
        xg = to_dev(x)
        _, info2 = s.solve(to_dev(w.rhs), xg, rtol=1e-7, x_is_initial_guess=True)
        assert info2["converged"] and info2["iters"] == 0
        # zero right-hand side
        z = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        xz, info3 = s.solve(z, rtol=1e-8)
        assert info3["converged"] and info3["iters"] == 0 and float(xz.abs().max()) == 0.0
    finally:
        s.destroy()


def test_restart_and_maxit_are_honoured():
    w, H, s = make("b6-4lev", restart=5, maxit=12)
    try:
        x_or, it_or, conv_or, hist_or = mg.solve(H, w.rhs, 1e-8)
        x, info = s.solve(to_dev(w.rhs), rtol=1e-8, hist_cap=64)
        assert info["iters"] <= 12 and abs(info["iters"] - it_or) <= 1
        assert info["converged"] == conv_or
        k = min(len(hist_or), len(info["hist"]))
        assert np.abs(np.log10(np.array(info["hist"][:k]) / np.array(hist_or[:k]))).max() <= 0.05
    finally:
        s.destroy()


def test_levels_1_is_the_coarse_solver_on_the_fine_matrix():
    w = small("C0", mesh=(3, 8), n_phi=4, levels=1, b=6, seed=91)
    H = oracle_hierarchy(w)
    s = gpu_solver(w, inject_bounds_from=H)
    try:
        r = input_vector(w.n, 91, 24)
        z = to_np(s.vcycle(to_dev(r)))
        assert np.linalg.norm(r - mg.spmv(H.levels[0], z)) <= 1.01e-10 * np.linalg.norm(r)
    finally:
        s.destroy()


def test_error_codes():
    import torch
    from paper_2506_16676_b200 import binding
    w = small("C0", mesh=(3, 8), n_phi=4, levels=2, b=6, seed=92)
    rp, ci, va = binding.upload(w)
    with pytest.raises(binding.MgError) as e:   # n_phi not divisible by 2^(levels-1)
        binding.Solver(rp, ci, va, w.b, w.n_pol, w.n_phi, 4)
    assert e.value.code == binding.MG_EINVAL
    with pytest.raises(binding.MgError) as e:   # unsupported block size
        binding.Solver(rp, ci, va, 65, w.n_pol, w.n_phi, 1)
    assert e.value.code == binding.MG_EINVAL
    ci_bad = ci.clone()
    ci_bad[1], ci_bad[2] = ci[2].item(), ci[1].item()   # unsorted columns
    with pytest.raises(binding.MgError) as e:
        binding.Solver(rp, ci_bad, va, w.b, w.n_pol, w.n_phi, w.levels)
    assert e.value.code == binding.MG_EINVAL
    va_bad = va.clone()
    bb = w.b * w.b
    dpos = int(np.nonzero(w.col_idx[w.row_ptr[5]:w.row_ptr[6]] == 5)[0][0] + w.row_ptr[5])
    va_bad[dpos * bb:(dpos + 1) * bb] = 0.0      # singular diagonal block
    with pytest.raises(binding.MgError) as e:
        binding.Solver(rp, ci, va_bad, w.b, w.n_pol, w.n_phi, w.levels)
    assert e.value.code == binding.MG_ESINGULAR
    s = binding.Solver(rp, ci, va, w.b, w.n_pol, w.n_phi, w.levels)
    try:
        v = s.new()
        with pytest.raises(binding.MgError):
            s.vcycle(v, v)                        # aliased in/out
        with pytest.raises(binding.MgError):
            s.spmv(7, v)                          # bad level
        assert s.launch_count() > 0 and s.device_bytes() > 0
    finally:
        s.destroy()
