"""Algorithmic-bytes model of the solve path.

Pure arithmetic on level sizes: what each step of the method MUST move through HBM if every array is read or
written exactly once per use (gathered ``x_J`` re-reads that the L2 serves are not counted).  ``bench.py`` and
the roofline report divide these by measured kernel durations.  Nothing here touches the GPU or the oracle.
"""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class LevelSize:
    n_brows: int   # block rows  n
    nnzb: int      # stored blocks
    b: int         # block size

    @property
    def nvec(self) -> int:
        return self.n_brows * self.b

    # ---- building blocks ------------------------------------------------------------------------------------
    @property
    def vec_bytes(self) -> int:          # one FP64 vector
        return 8 * self.nvec

    @property
    def matrix_bytes(self) -> int:       # values + col_idx (int32) + row_ptr (int64)
        return self.nnzb * (8 * self.b * self.b + 4) + 8 * (self.n_brows + 1)

    @property
    def dinv_bytes(self) -> int:         # explicit dense inverses of the diagonal blocks
        return 8 * self.n_brows * self.b * self.b

    # ---- per-kernel algorithmic bytes (one launch) --------------------------------------------------------------
    def spmv(self) -> int:               # read A, x; write y
        return self.matrix_bytes + 2 * self.vec_bytes

    def resid(self) -> int:              # read A, x, rhs; write r
        return self.matrix_bytes + 3 * self.vec_bytes

    def sweep(self) -> int:              # read A, D^-1, d, r, x; write r, x, d'
        return self.matrix_bytes + self.dinv_bytes + 6 * self.vec_bytes

    def sweep_nod(self) -> int:          # read A, d, r, x; write r, x
        return self.matrix_bytes + 5 * self.vec_bytes

    def pbj(self) -> int:                # read D^-1, r; write z
        return self.dinv_bytes + 2 * self.vec_bytes

    def restrict(self) -> int:           # read fine r; write coarse r (half as long)
        return self.vec_bytes + self.vec_bytes // 2

    def prolong(self) -> int:            # read coarse e (half), read+write fine x, write P e
        return self.vec_bytes // 2 + 3 * self.vec_bytes

    def gmres_iteration(self, j: int) -> int:
        """One right-PBJ-preconditioned GMRES step with j previous basis vectors, CGS2: A, D^-1 once; the basis
        V_0..V_j read once (what the method must move: the second Gram-Schmidt pass can run from on-chip copies);
        w and the work vectors read/written a few times."""
        return self.matrix_bytes + self.dinv_bytes + ((j + 1) + 8) * self.vec_bytes

    def by_kind(self, kind: str) -> int:
        return getattr(self, kind)()


def vcycle_bytes(levels, nu_pre: int, nu_post: int, coarse_sweeps: int | None = None) -> int:
    """One V(nu_pre, nu_post) cycle over ``levels`` (list of LevelSize, finest first), excluding the coarsest
    solve unless ``coarse_sweeps`` (pinned coarse mode: that many Chebyshev-PBJ sweeps) is given."""
    total = 0
    for L in levels[:-1]:
        if nu_pre > 0:
            total += L.pbj() + (nu_pre - 1) * L.sweep() + L.sweep_nod()
        total += L.restrict() + L.prolong()
        total += nu_post * L.sweep()
    if coarse_sweeps:
        Lc = levels[-1]
        total += Lc.pbj() + (coarse_sweeps - 1) * Lc.sweep() + Lc.sweep_nod()
    return total
