"""Thin ctypes binding of ``libmgtoroidal.so`` -- same names as ``include/mg_toroidal.h``.

Argument marshalling only: torch tensors give device memory (``data_ptr()``) and the current CUDA
stream; every step of the path runs in the library's kernels.  There is no CPU fallback: importing
works anywhere (so that symbol tests can run without a GPU), but any compute call without the
library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

from . import buildlib

MG_OK, MG_EINVAL, MG_ENOMEM, MG_ESINGULAR, MG_ECUDA, MG_ETOOLARGE = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_N = 1 << 26
KIND_NAMES = ("spmv", "resid", "sweep", "sweep_nod", "pbj", "restrict", "prolong", "orth", "other", "cycle", "direct", "line")

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class mg_options(C.Structure):
    _fields_ = [("nu_pre", C.c_int), ("nu_post", C.c_int), ("cheb_lo", C.c_double), ("cheb_hi", C.c_double),
                ("eig_iters", C.c_int), ("coarse_mode", C.c_int), ("coarse_rtol", C.c_double),
                ("coarse_restart", C.c_int), ("coarse_maxit", C.c_int), ("coarse_fixed_sweeps", C.c_int),
                ("restart", C.c_int), ("maxit", C.c_int), ("use_graphs", C.c_int), ("kernel_variant", C.c_int), ("smoother", C.c_int), ("orth_eta", C.c_double),
                ("alloc", ALLOC_FN), ("free", FREE_FN), ("alloc_ctx", C.c_void_p)]


class mg_solve_info(C.Structure):
    _fields_ = [("iters", C.c_int), ("converged", C.c_int), ("solve_ms", C.c_double), ("rel_res", C.c_double), ("coarse_iters_total", C.c_int),
                ("hist_len", C.c_int), ("hist", C.POINTER(C.c_double))]


# name -> (restype, argtypes); one row per symbol declared in include/mg_toroidal.h
_VP, _I, _D, _I64 = C.c_void_p, C.c_int, C.c_double, C.c_int64
SYMBOLS = {
    "mg_options_default": (_I, [C.POINTER(mg_options)]),
    "mg_sizeof_options": (C.c_size_t, []),
    "mg_sizeof_solve_info": (C.c_size_t, []),
    "mg_setup": (_I, [C.POINTER(_VP), _VP, _VP, _VP, _I, _I, _I, _I, C.POINTER(mg_options), _VP]),
    "mg_update_options": (_I, [_VP, C.POINTER(mg_options)]),
    "mg_update_values": (_I, [_VP, _VP]),
    "mg_set_operator": (_I, [_VP, _VP]),
    "mg_vcycle": (_I, [_VP, _VP, _VP]),
    "mg_solve": (_I, [_VP, _VP, _VP, _D, _I, C.POINTER(mg_solve_info)]),
    "mg_solve_host": (_I, [_VP, _VP, _VP, _D, _I, C.POINTER(mg_solve_info)]),
    "mg_destroy": (_I, [_VP]),
    "mg_spmv": (_I, [_VP, _I, _VP, _VP]),
    "mg_residual": (_I, [_VP, _I, _VP, _VP, _VP]),
    "mg_pbj_apply": (_I, [_VP, _I, _VP, _VP]),
    "mg_smooth": (_I, [_VP, _I, _VP, _VP, _I, _I]),
    "mg_restrict": (_I, [_VP, _I, _VP, _VP]),
    "mg_prolong_add": (_I, [_VP, _I, _VP, _VP]),
    "mg_coarse_solve": (_I, [_VP, _VP, _VP, C.POINTER(_I)]),
    "mg_direct_info": (_I, [_VP, C.POINTER(_I), C.POINTER(_I64), C.POINTER(_I64), C.POINTER(_I), C.POINTER(_I)]),
    "mg_dot": (_I, [_VP, _I, _VP, _VP, _VP]),
    "mg_dot_noalloc": (_I, [_VP, _VP, _I64, _VP, _VP]),
    "mg_get_level": (_I, [_VP, _I, C.POINTER(_I64), C.POINTER(_I64), C.POINTER(_VP), C.POINTER(_VP), C.POINTER(_VP),
                          C.POINTER(_VP), C.POINTER(_D), C.POINTER(_D), C.POINTER(_D)]),
    "mg_copy_level_to_host": (_I, [_VP, _I, _VP, _VP, _VP, _VP]),
    "mg_set_cheb_bounds": (_I, [_VP, _I, _D, _D]),
    "mg_profile_enable": (_I, [_VP, _I]),
    "mg_profile_reset": (_I, [_VP]),
    "mg_profile_get": (_I, [_VP, _I, _I, C.POINTER(_I64), C.POINTER(_I64), C.POINTER(_D)]),
    "mg_launch_count": (_I64, [_VP]),
    "mg_device_bytes": (_I64, [_VP]),
    "mg_strerror": (C.c_char_p, [_I]),
    "mg_version": (C.c_char_p, []),
}

_lib = None


class MgError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__(f"{what}: {strerror(code)} (code {code})")


def lib():
    """Load ``libmgtoroidal.so`` (never builds silently on import; ``buildlib.build()`` does that)."""
    global _lib
    if _lib is None:
        if not os.path.exists(buildlib.LIB_PATH):
            raise RuntimeError(f"{buildlib.LIB_PATH} is missing: run paper_2506_16676_b200.buildlib.build(); "
                               "there is no CPU fallback")
        L = C.CDLL(buildlib.LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        if L.mg_sizeof_options() != C.sizeof(mg_options) or L.mg_sizeof_solve_info() != C.sizeof(mg_solve_info):
            raise RuntimeError("binding.py and libmgtoroidal.so disagree on the layout of mg_options / mg_solve_info: "
                               "rebuild with paper_2506_16676_b200.buildlib.build(force=True)")
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().mg_strerror(code).decode()


def version() -> str:
    return lib().mg_version().decode()


def _chk(code, what):
    if code != MG_OK:
        raise MgError(code, what)


def options_default(**kw) -> mg_options:
    o = mg_options()
    _chk(lib().mg_options_default(C.byref(o)), "mg_options_default")
    for k, v in kw.items():
        if not hasattr(o, k):
            raise AttributeError(k)
        setattr(o, k, v)
    return o


def _ptr(t, dtype=None, numel=None):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"expected {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


class Solver:
    """Owner of one ``mg_handle``.  Methods carry the C names without the ``mg_`` prefix."""

    def __init__(self, row_ptr, col_idx, vals, b: int, n_pol: int, n_phi: int, levels: int, opt: mg_options = None,
                 **opt_kw):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libmgtoroidal has no CPU fallback")
        self._h = C.c_void_p()
        self.b, self.n_pol, self.n_phi, self.levels = int(b), int(n_pol), int(n_phi), int(levels)
        # the library borrows these for the life of the handle: keep them alive here
        self.row_ptr, self.col_idx, self.vals = row_ptr, col_idx, vals
        self.opt = opt if opt is not None else options_default(**opt_kw)
        self.stream = torch.cuda.current_stream().cuda_stream
        _chk(lib().mg_setup(C.byref(self._h), _ptr(row_ptr, torch.int64), _ptr(col_idx, torch.int32),
                            _ptr(vals, torch.float64), self.b, self.n_pol, self.n_phi, self.levels, C.byref(self.opt),
                            C.c_void_p(self.stream)), "mg_setup")
        self.device = vals.device

    # ---- lifetime ------------------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().mg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    # ---- helpers -------------------------------------------------------------------------------------------
    def n(self, level: int = 0):
        """Vector length of a level (None for a level that does not exist: the library rejects it with MG_EINVAL)."""
        if not 0 <= level < self.levels:
            return None
        return (self.n_phi >> level) * self.n_pol * self.b

    def new(self, level: int = 0):
        import torch
        return torch.empty(self.n(level) or 0, dtype=torch.float64, device=self.device)

    def update_options(self, **kw):
        for k, v in kw.items():
            if not hasattr(self.opt, k):
                raise AttributeError(k)
            setattr(self.opt, k, v)
        _chk(lib().mg_update_options(self._h, C.byref(self.opt)), "mg_update_options")

    # ---- the C ABI -----------------------------------------------------------------------------------------
    def update_values(self, vals):
        """Refresh: new fine values (same pattern); the library borrows ``vals`` from now on."""
        import torch
        _chk(lib().mg_update_values(self._h, _ptr(vals, torch.float64)), "mg_update_values")
        self.vals = vals
        self._op_vals = None

    def set_operator(self, vals=None):
        """Lag: solve with (pattern, ``vals``) while the V-cycle keeps the old hierarchy; None = hierarchy's matrix."""
        import torch
        _chk(lib().mg_set_operator(self._h, _ptr(vals, torch.float64) if vals is not None else None), "mg_set_operator")
        self._op_vals = vals

    def vcycle(self, r, z=None):
        import torch
        z = self.new() if z is None else z
        _chk(lib().mg_vcycle(self._h, _ptr(r, torch.float64, self.n()), _ptr(z, torch.float64, self.n())), "mg_vcycle")
        return z

    def solve(self, rhs, x=None, rtol: float = 1e-8, x_is_initial_guess: bool = False, hist_cap: int = 0):
        import torch
        x = self.new() if x is None else x
        info = mg_solve_info()
        hist = (C.c_double * hist_cap)() if hist_cap > 0 else None
        info.hist_len = hist_cap
        info.hist = C.cast(hist, C.POINTER(C.c_double)) if hist is not None else None
        _chk(lib().mg_solve(self._h, _ptr(rhs, torch.float64, self.n()), _ptr(x, torch.float64, self.n()), float(rtol),
                            int(bool(x_is_initial_guess)), C.byref(info)), "mg_solve")
        return x, _info_dict(info, hist)

    def solve_host(self, rhs_host, x_host, rtol: float = 1e-8, x_is_initial_guess: bool = False, hist_cap: int = 0):
        """HOST buffers (torch CPU tensors, ideally pinned, or NumPy float64 arrays)."""
        info = mg_solve_info()
        hist = (C.c_double * hist_cap)() if hist_cap > 0 else None
        info.hist_len = hist_cap
        info.hist = C.cast(hist, C.POINTER(C.c_double)) if hist is not None else None
        _chk(lib().mg_solve_host(self._h, _host_ptr(rhs_host, self.n()), _host_ptr(x_host, self.n()), float(rtol),
                                 int(bool(x_is_initial_guess)), C.byref(info)), "mg_solve_host")
        return x_host, _info_dict(info, hist)

    def spmv(self, level, x, y=None):
        import torch
        y = self.new(level) if y is None else y
        _chk(lib().mg_spmv(self._h, level, _ptr(x, torch.float64, self.n(level)), _ptr(y, torch.float64, self.n(level))), "mg_spmv")
        return y

    def residual(self, level, rhs, x, r=None):
        import torch
        r = self.new(level) if r is None else r
        _chk(lib().mg_residual(self._h, level, _ptr(rhs, torch.float64, self.n(level)), _ptr(x, torch.float64, self.n(level)),
                               _ptr(r, torch.float64, self.n(level))), "mg_residual")
        return r

    def pbj_apply(self, level, r, z=None):
        import torch
        z = self.new(level) if z is None else z
        _chk(lib().mg_pbj_apply(self._h, level, _ptr(r, torch.float64, self.n(level)), _ptr(z, torch.float64, self.n(level))), "mg_pbj_apply")
        return z

    def smooth(self, level, rhs, x, nu: int, zero_guess: bool):
        import torch
        _chk(lib().mg_smooth(self._h, level, _ptr(rhs, torch.float64, self.n(level)), _ptr(x, torch.float64, self.n(level)), int(nu),
                             int(bool(zero_guess))), "mg_smooth")
        return x

    def restrict(self, level, r_fine, r_coarse=None):
        import torch
        r_coarse = self.new(level + 1) if r_coarse is None else r_coarse
        _chk(lib().mg_restrict(self._h, level, _ptr(r_fine, torch.float64, self.n(level)), _ptr(r_coarse, torch.float64, self.n(level + 1))),
             "mg_restrict")
        return r_coarse

    def prolong_add(self, level, e_coarse, x_fine):
        import torch
        _chk(lib().mg_prolong_add(self._h, level, _ptr(e_coarse, torch.float64, self.n(level + 1)), _ptr(x_fine, torch.float64, self.n(level))),
             "mg_prolong_add")
        return x_fine

    def coarse_solve(self, r, e=None):
        import torch
        e = self.new(self.levels - 1) if e is None else e
        it = C.c_int(0)
        _chk(lib().mg_coarse_solve(self._h, _ptr(r, torch.float64, self.n(self.levels - 1)), _ptr(e, torch.float64, self.n(self.levels - 1)), C.byref(it)),
             "mg_coarse_solve")
        return e, it.value

    def direct_info(self) -> dict:
        """Sizes of the direct coarsest-level solve (after its first use)."""
        ls, mx, pers = C.c_int(), C.c_int(), C.c_int()
        dense, od = C.c_int64(), C.c_int64()
        _chk(lib().mg_direct_info(self._h, C.byref(ls), C.byref(dense), C.byref(od), C.byref(mx), C.byref(pers)), "mg_direct_info")
        return dict(level_sets=ls.value, dense_bytes=dense.value, offdiag_bytes=od.value, max_n=mx.value,
                    persistent=bool(pers.value), bytes_per_solve=2 * dense.value + od.value)

    def dot(self, level, a, b, out=None):
        """<a, b> of two level vectors into a 1-element device tensor (the handle's own scratch)."""
        import torch
        out = torch.empty(1, dtype=torch.float64, device=self.device) if out is None else out
        _chk(lib().mg_dot(self._h, level, _ptr(a, torch.float64, self.n(level)), _ptr(b, torch.float64, self.n(level)),
                          _ptr(out, torch.float64, 1)), "mg_dot")
        return out

    def get_level(self, level: int) -> dict:
        """Sizes, Chebyshev bounds and (as torch views of the library's device memory) the level's arrays."""
        nb, nz = C.c_int64(), C.c_int64()
        rp, ci, va, di = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
        rho, lo, hi = C.c_double(), C.c_double(), C.c_double()
        _chk(lib().mg_get_level(self._h, level, C.byref(nb), C.byref(nz), C.byref(rp), C.byref(ci), C.byref(va),
                                C.byref(di), C.byref(rho), C.byref(lo), C.byref(hi)), "mg_get_level")
        return dict(n_brows=nb.value, nnzb=nz.value, row_ptr=rp.value, col_idx=ci.value, vals=va.value, dinv=di.value,
                    rho_est=rho.value, lam_min=lo.value, lam_max=hi.value)

    def level_arrays(self, level: int) -> dict:
        """Copies of one level's arrays as NumPy (tests compare them with the oracle's hierarchy)."""
        g = self.get_level(level)
        b = self.b
        out = dict(g)
        import numpy as np
        out["row_ptr"] = np.empty(g["n_brows"] + 1, np.int64)
        out["col_idx"] = np.empty(g["nnzb"], np.int32)
        out["vals"] = np.empty((g["nnzb"], b, b), np.float64)
        out["dinv"] = np.empty((g["n_brows"], b, b), np.float64)
        _chk(lib().mg_copy_level_to_host(self._h, level, *(C.c_void_p(out[k].ctypes.data) for k in
                                                            ("row_ptr", "col_idx", "vals", "dinv"))),
             "mg_copy_level_to_host")
        return out

    def set_cheb_bounds(self, level, lam_min, lam_max):
        _chk(lib().mg_set_cheb_bounds(self._h, level, float(lam_min), float(lam_max)), "mg_set_cheb_bounds")

    def profile_enable(self, on: bool = True):
        _chk(lib().mg_profile_enable(self._h, int(bool(on))), "mg_profile_enable")

    def profile_reset(self):
        _chk(lib().mg_profile_reset(self._h), "mg_profile_reset")

    def profile_get(self) -> dict:
        """{(level, kind_name): dict(launches, timed, ms)} of every class that launched since the last reset."""
        out = {}
        for level in range(self.levels):
            for kind, name in enumerate(KIND_NAMES):
                n, nt, ms = C.c_int64(), C.c_int64(), C.c_double()
                _chk(lib().mg_profile_get(self._h, level, kind, C.byref(n), C.byref(nt), C.byref(ms)),
                     "mg_profile_get")
                if n.value:
                    out[(level, name)] = dict(launches=n.value, timed=nt.value, ms=ms.value)
        return out

    def launch_count(self) -> int:
        return int(lib().mg_launch_count(self._h))

    def device_bytes(self) -> int:
        return int(lib().mg_device_bytes(self._h))


def dot_noalloc(a, b, out):
    """mg_dot_noalloc: <a, b> into the caller's 1-element device tensor ``out``; the library allocates nothing (its scratch is
    a fixed device array; at most NOALLOC_MAX_N elements; calls that overlap on the GPU race on that array)."""
    import torch
    if a.numel() != b.numel():
        raise ValueError("a and b differ in length")
    stream = torch.cuda.current_stream().cuda_stream
    _chk(lib().mg_dot_noalloc(_ptr(a, torch.float64), _ptr(b, torch.float64), a.numel(), _ptr(out, torch.float64, 1),
                              C.c_void_p(stream)), "mg_dot_noalloc")
    return out


def _info_dict(info, hist):
    return dict(iters=info.iters, converged=bool(info.converged), solve_ms=info.solve_ms, rel_res=info.rel_res,
                coarse_iters_total=info.coarse_iters_total,
                hist=[hist[i] for i in range(info.hist_len)] if hist is not None else [])


def _host_ptr(a, n):
    import numpy as np
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n:
            raise TypeError("expected a contiguous float64 CPU tensor of the level-0 vector length")
        return C.c_void_p(a.data_ptr())
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags.c_contiguous or a.size != n:
            raise TypeError("expected a contiguous float64 array of the level-0 vector length")
        return C.c_void_p(a.ctypes.data)
    raise TypeError("expected a torch CPU tensor or a NumPy array")


def upload(w, device="cuda"):
    """Workload (NumPy arrays from ``workloads.make_workload``) -> the three device tensors mg_setup borrows."""
    import torch
    return (torch.from_numpy(w.row_ptr).to(device), torch.from_numpy(w.col_idx).to(device),
            torch.from_numpy(w.vals.reshape(-1)).to(device))
