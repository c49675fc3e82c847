"""GPU parity, per kernel: the CUDA library (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs (BASELINE.json north_star: per-kernel outputs within 1e-12 relative, max-norm).

Sizes: reduced instances of the configs' recipe that the oracle finishes in seconds yet span many CTAs and a
ragged last CTA (b=6: 14 block rows per CTA, b=12: 3, b=36: 1), plus config 0 at full size."""
import numpy as np
import pytest

from oracle import mg
from paper_2506_16676_b200.workloads import input_vector
from gpu_util import TOL_KERNEL, relmax, small, oracle_hierarchy, gpu_solver, to_dev, to_np

pytestmark = pytest.mark.gpu

CASES = {
    "C0-b36": dict(name="C0"),
    "b12-3lev": dict(name="C0", mesh=(5, 16), n_phi=8, levels=3, b=12, seed=77),
    "b6-4lev": dict(name="C0", mesh=(6, 20), n_phi=16, levels=4, b=6, seed=78),
    "b5-generic-to-1-plane": dict(name="C0", mesh=(3, 8), n_phi=4, levels=3, b=5, seed=79),
    "b1": dict(name="C0", mesh=(3, 7), n_phi=6, levels=2, b=1, seed=80),
    "b36-nonaxi": dict(name="C3", mesh=(3, 10), n_phi=8, levels=3, seed=81),
    # C3b recipe (21-block prism stencil on the fine level, plane-modulated), reduced
    "b36-prism": dict(name="C3b", mesh=(3, 10), n_phi=8, levels=3, seed=88),
    # largest supported block (generic kernel; the batched inverse needs > 48 KB of shared memory) and a tiny one
    "b64-max-block": dict(name="C0", mesh=(2, 6), n_phi=4, levels=2, b=64, seed=86),
    "b2": dict(name="C0", mesh=(2, 5), n_phi=4, levels=3, b=2, seed=87),
    # TMA-ring kernel: ~120 blocks per persistent CTA (the 20-stage ring wraps six times), ragged row ranges
    "b36-ring-wraps": dict(name="C0", mesh=(8, 30), n_phi=8, levels=3, seed=82),
    # fewer block rows than SMs on the coarsest level (CTAs with a single row, idle consumer groups)
    "b36-few-rows": dict(name="C0", mesh=(3, 5), n_phi=8, levels=3, seed=83),
    # the one-CTA-per-row 128-bit-load kernel at b = 36 (kernel_variant = 1)
    "b36-ldg-variant": dict(name="C0", mesh=(4, 12), n_phi=8, levels=2, seed=84, opt=dict(kernel_variant=1)),
}


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    kw = dict(CASES[request.param])
    opt = kw.pop("opt", {})
    w = small(kw.pop("name"), **kw)
    H = oracle_hierarchy(w)
    s = gpu_solver(w, inject_bounds_from=H, **opt)
    yield w, H, s
    s.destroy()


def test_hierarchy_pattern_is_bit_exact_and_values_match(case):
    """mg_setup: Galerkin coarse operators A_{l+1} = P^T A_l P and PBJ inverses."""
    w, H, s = case
    for l, L in enumerate(H.levels):
        g = s.level_arrays(l)
        assert g["n_brows"] == L.n_brows and g["nnzb"] == L.nnzb
        assert np.array_equal(g["row_ptr"], L.row_ptr)          # index work: bit-exact
        assert np.array_equal(g["col_idx"], L.col_idx)
        assert relmax(g["vals"], L.vals) <= TOL_KERNEL
        # both sides run Gauss-Jordan with partial pivoting: differences are rounding amplified by cond(D) ~ 1e2..1e3
        assert relmax(g["dinv"], L.dinv) <= 1e-11
        assert abs(g["rho_est"] - L.rho_est) <= 1e-9 * L.rho_est


def test_library_bounds_follow_the_estimate(case):
    w, H, s = case
    s2 = gpu_solver(w)
    try:
        for l, L in enumerate(H.levels):
            g = s2.get_level(l)
            assert g["lam_min"] == pytest.approx(0.1 * g["rho_est"], rel=1e-14)
            assert g["lam_max"] == pytest.approx(1.1 * g["rho_est"], rel=1e-14)
            assert g["lam_max"] == pytest.approx(L.lam_max, rel=1e-9)
    finally:
        s2.destroy()


def test_spmv_residual_pbj(case):
    w, H, s = case
    for l, L in enumerate(H.levels):
        x = input_vector(L.n, w.seed + l, 11)
        rhs = input_vector(L.n, w.seed + l, 12)
        y_or = mg.spmv(L, x)
        assert relmax(to_np(s.spmv(l, to_dev(x))), y_or) <= TOL_KERNEL
        assert relmax(to_np(s.residual(l, to_dev(rhs), to_dev(x))), rhs - y_or) <= TOL_KERNEL
        assert relmax(to_np(s.pbj_apply(l, to_dev(rhs))), mg.pbj_apply(L, rhs)) <= TOL_KERNEL


@pytest.mark.parametrize("nu", [0, 1, 2, 3, 5])
@pytest.mark.parametrize("zero_guess", [True, False])
def test_chebyshev_pbj_smoother(case, nu, zero_guess):
    """Fused sweep kernel vs the three-term recurrence written out in the oracle (reading Q2/Q3)."""
    w, H, s = case
    for l, L in enumerate(H.levels):
        rhs = input_vector(L.n, w.seed + l, 13)
        x0 = None if zero_guess else input_vector(L.n, w.seed + l, 14)
        x_or = mg.chebyshev(L, rhs, x0, nu)
        xg = to_dev(np.full(L.n, 123.0) if zero_guess else x0)  # a zero guess must overwrite garbage
        s.smooth(l, to_dev(rhs), xg, nu, zero_guess)
        assert relmax(to_np(xg), x_or) <= TOL_KERNEL


def test_restrict_prolong(case):
    w, H, s = case
    for l in range(len(H.levels) - 1):
        Lf, Lc = H.levels[l], H.levels[l + 1]
        r = input_vector(Lf.n, w.seed + l, 15)
        e = input_vector(Lc.n, w.seed + l, 16)
        x = input_vector(Lf.n, w.seed + l, 17)
        assert relmax(to_np(s.restrict(l, to_dev(r))), mg.restrict(Lc.pphi, r)) <= TOL_KERNEL
        xg = to_dev(x)
        s.prolong_add(l, to_dev(e), xg)
        assert relmax(to_np(xg), x + mg.prolong(Lc.pphi, e)) <= TOL_KERNEL


def test_prolongation_of_plane_constant_field_is_exact(case):
    """north_star invariant: P 1 = 1 plane-wise (row sums of the [1/2 1 1/2] stencil)."""
    w, H, s = case
    import torch
    for l in range(len(H.levels) - 1):
        Lf, Lc = H.levels[l], H.levels[l + 1]
        plane = input_vector(Lf.n_pol * Lf.b, w.seed, 18)
        e = np.tile(plane, Lc.n_phi)
        xg = torch.zeros(Lf.n, dtype=torch.float64, device="cuda")
        s.prolong_add(l, to_dev(e), xg)
        assert np.array_equal(to_np(xg), np.tile(plane, Lf.n_phi))


@pytest.mark.parametrize("b", [12, 36])
def test_shuffled_numbering_spmv(b):
    """configs[4] 'shuffled' variant: col_idx is arbitrary within a plane."""
    w = small("C0", mesh=(6, 20), n_phi=4, levels=1, b=b, seed=90, shuffle=True)
    H = oracle_hierarchy(w)
    s = gpu_solver(w, inject_bounds_from=H)
    try:
        x = input_vector(w.n, 90, 11)
        assert relmax(to_np(s.spmv(0, to_dev(x))), mg.spmv(H.levels[0], x)) <= TOL_KERNEL
        rhs = input_vector(w.n, 90, 12)
        xg = s.new()
        s.smooth(0, to_dev(rhs), xg, 1, True)
        assert relmax(to_np(xg), mg.chebyshev(H.levels[0], rhs, None, 1)) <= TOL_KERNEL
    finally:
        s.destroy()
