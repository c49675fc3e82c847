"""B200-native toroidal semi-coarsening multigrid / FGMRES solve path (arXiv 2506.16676).

The package holds only what the hot path needs:

* ``csrc/``      -- hand-written CUDA (sm_100a) kernels and the C-ABI library ``libmgtoroidal.so``
                    (boundary declared in ``include/mg_toroidal.h``);
* ``binding``    -- thin ctypes binding with the same names as the C ABI (argument marshalling only);
* ``workloads``  -- the seeded synthetic input generator shared by the oracle tests and the GPU
                    tests (holds none of the method's arithmetic);
* ``buildlib``   -- the in-tree nvcc build step.

Nothing here imports ``oracle/`` (test infrastructure) and there is no CPU fallback: every product
entry point fails loudly if the CUDA library is missing.

Submodules are imported lazily so that ``paper_2506_16676_b200.workloads`` can be used on a box with
no GPU and no built library.
"""

__all__ = ["binding", "workloads", "buildlib"]
__version__ = "0.1.0"
