"""mg_dot_noalloc: the deterministic dot product of the orthogonalisation for callers that must not allocate
(CUDA graph capture, serving loops).  Its scratch is a file-scope device array of the library instead of the handle's
cudaMalloc'd buffers; same kernel, same launch shape.  Checked against the existing path (mg_dot, the handle's scratch) within
the kernel tolerance 1e-12, on two calls in a row (the shared array keeps the previous call's contents).

Collected last on purpose (pytest -x): the file name sorts after every other test file."""
import numpy as np
import pytest

from gpu_util import TOL_KERNEL, small, gpu_solver, to_dev
from paper_2506_16676_b200.workloads import input_vector

pytestmark = pytest.mark.gpu


def test_dot_noalloc_matches_the_handle_path_twice_in_a_row():
    import torch
    from paper_2506_16676_b200 import binding
    w = small("C0", mesh=(5, 16), n_phi=8, levels=2, b=12, seed=77)       # 7,680 / 3,840 unknowns per level
    s = gpu_solver(w, coarse_mode=1)
    try:
        out = torch.full((1,), 123.0, dtype=torch.float64, device="cuda")  # caller-owned result, pre-filled with garbage
        for call, level in enumerate((0, 1, 0)):                           # different lengths: stale partials must not leak
            n = s.n(level)
            a = to_dev(input_vector(n, 100 + call, 31))
            b = to_dev(input_vector(n, 200 + call, 32))
            ref = float(s.dot(level, a, b).cpu()[0])                        # existing path: the handle's scratch
            got = float(binding.dot_noalloc(a, b, out).cpu()[0])
            exact = float(np.dot(a.cpu().numpy(), b.cpu().numpy()))
            scale = float(np.abs(a.cpu().numpy() * b.cpu().numpy()).sum())
            assert abs(got - ref) <= TOL_KERNEL * scale, (call, got, ref)
            assert got == ref                                               # same kernel and launch shape: the same bits
            assert abs(got - exact) <= TOL_KERNEL * scale
    finally:
        s.destroy()


def test_dot_noalloc_needs_no_handle_and_rejects_oversize():
    import torch
    from paper_2506_16676_b200 import binding
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    a = torch.arange(1, 1001, dtype=torch.float64, device="cuda")
    assert float(binding.dot_noalloc(a, a, out).cpu()[0]) == float((np.arange(1, 1001, dtype=np.float64) ** 2).sum())
    odd = a[:999]                                                           # odd length: the scalar tail element
    assert float(binding.dot_noalloc(odd, odd, out).cpu()[0]) == float((np.arange(1, 1000, dtype=np.float64) ** 2).sum())
    # beyond the fixed maximum: a clear error, nothing launched (the check needs only the size, so no 512 MiB buffers here)
    import ctypes as C
    rc = binding.lib().mg_dot_noalloc(C.c_void_p(a.data_ptr()), C.c_void_p(a.data_ptr()), binding.NOALLOC_MAX_N + 1,
                                      C.c_void_p(out.data_ptr()), None)
    assert rc == binding.MG_ETOOLARGE and "MG_NOALLOC_MAX_N" in binding.strerror(rc)
