"""Seeded synthetic workload generator (test/bench infrastructure; none of the method's arithmetic).

Stands in for the paper's M3D-C1 matrices (SPARC / stellarator), which are not
available.  It keeps their *shape and structure*: block size b = 36 = 12 x 3 DoF per
vertex, a 2-D unstructured-style poloidal mesh extruded over periodic toroidal planes
(PAPER.md:27, 45), 4-64 planes, nearly symmetric elliptic blocks with weak nonsymmetry
(PAPER.md:47, 328-330), and a non-axisymmetric variant.  The numeric recipe is the one
``BASELINE.json:configs`` states, made concrete in DESIGN.md "Input recipe":

    A = sigma*I + sum_ij w_ij (S_i - S_ij) + beta * L_tor (x) T + delta * N

* D1 mesh: annulus of n_r rings x n_theta nodes, node (a,t) -> i = a*n_theta + t, lattice units,
  quads split along (a,t)-(a+1,t+1), coordinates jittered by 0.2*h_loc*U(-1,1); w_ij = 1/|p_i - p_j|.
* D2 S, T: Q diag(lambda) Q^T with lambda log-spaced in [0.1, 10] (condition number 1e2).
* D3 blocks: diag = sigma I + (sum_j w_ij) S + 2 beta T; in-plane = -w_ij S; toroidal = -beta T;
  noise N block-skew-symmetric: N_IJ = c G / sqrt(b), N_JI = -c G^T / sqrt(b), c = w_ij or beta.
* D4 non-axisymmetric: per-plane modulation of w_ij and of the spectrum of S.
* D5 RHS: U[-1, 1].

Output layout (what both the oracle and the CUDA library consume): square block-CSR, block rows
ordered plane-major (I = k*n_pol + i), ``row_ptr`` int64[n+1], ``col_idx`` int32[nnzb] sorted
ascending within a row, ``vals`` float64[nnzb, b, b] row-major blocks, ``rhs`` float64[n*b].
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

BASE_SEED = 20250616


@dataclass
class Workload:
    name: str
    b: int
    n_r: int
    n_theta: int
    n_phi: int
    levels: int
    sigma: float
    beta: float
    delta: float
    seed: int
    row_ptr: np.ndarray = field(repr=False, default=None)
    col_idx: np.ndarray = field(repr=False, default=None)
    vals: np.ndarray = field(repr=False, default=None)
    rhs: np.ndarray = field(repr=False, default=None)
    S: np.ndarray = field(repr=False, default=None)
    T: np.ndarray = field(repr=False, default=None)
    adj_w: object = field(repr=False, default=None)  # (edges int64[E,2], w float64[E]) of one plane

    @property
    def n_pol(self) -> int:
        return self.n_r * self.n_theta

    @property
    def n_brows(self) -> int:
        return self.n_pol * self.n_phi

    @property
    def nnzb(self) -> int:
        return int(self.col_idx.shape[0])

    @property
    def n(self) -> int:
        return self.n_brows * self.b


# name -> parameters (BASELINE.json configs[0..4])
CONFIGS = {
    "C0": dict(mesh=(4, 24), n_phi=8, levels=2, sigma=1e-3, beta=0.1, delta=0.05, b=36, seed=BASE_SEED + 0),
    "C1": dict(mesh=(20, 100), n_phi=16, levels=4, sigma=1e-3, beta=0.1, delta=0.05, b=36, seed=BASE_SEED + 1),
    "C2-16": dict(mesh=(20, 100), n_phi=16, levels=4, sigma=1e-4, beta=1.0, delta=0.05, b=36, seed=BASE_SEED + 2),
    "C2-32": dict(mesh=(20, 100), n_phi=32, levels=5, sigma=1e-4, beta=1.0, delta=0.05, b=36, seed=BASE_SEED + 2),
    "C2-64": dict(mesh=(20, 100), n_phi=64, levels=6, sigma=1e-4, beta=1.0, delta=0.05, b=36, seed=BASE_SEED + 2),
    "C3": dict(mesh=(40, 200), n_phi=32, levels=5, sigma=1e-4, beta=0.5, delta=0.15, b=36, seed=BASE_SEED + 3,
               nonaxisymmetric=True),
    # C3b (Q16): config 3 with the 21-block prism stencil on the FINE level -- the density of
    # the paper's matrices (~750 nnz/row) and the "~55 GB" that configs[3] states (54.9 GB).
    "C3b": dict(mesh=(40, 200), n_phi=32, levels=5, sigma=1e-4, beta=0.5, delta=0.15, b=36, seed=BASE_SEED + 3,
                nonaxisymmetric=True, prism=True),
}


def c4_points():
    """The 12 kernel-sweep points of configs[4]: b in {6,12,36} x nodes in {2000, 8000} x planes in {16, 64}."""
    pts = []
    idx = 0
    for b in (6, 12, 36):
        for mesh in ((20, 100), (40, 200)):
            for n_phi in (16, 64):
                pts.append(dict(name=f"C4-b{b}-n{mesh[0] * mesh[1]}-p{n_phi}", mesh=mesh, n_phi=n_phi, levels=1,
                                sigma=1e-3, beta=0.1, delta=0.05, b=b, seed=BASE_SEED + 4 + idx))
                idx += 1
    return pts


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(np.random.SeedSequence([seed, stream])))


def _spd(rng: np.random.Generator, b: int):
    """Q diag(lambda) Q^T, lambda_c = 10^(-1 + 2c/(b-1)); returns (Q, lambda)."""
    G = rng.standard_normal((b, b))
    Q, R = np.linalg.qr(G)
    Q = Q * np.sign(np.diag(R))[None, :]
    lam = np.ones(1) if b == 1 else 10.0 ** (-1.0 + 2.0 * np.arange(b) / (b - 1))
    return Q, lam


def poloidal_mesh(n_r: int, n_theta: int, rng: np.random.Generator):
    """D1: jittered triangulated annulus. Returns (edges int64[E,2] with i<j, w float64[E], xy float64[n,2])."""
    a = np.repeat(np.arange(n_r), n_theta)
    t = np.tile(np.arange(n_theta), n_r)
    r_a = n_theta / (2 * np.pi) - (n_r - 1) / 2.0 + a
    ang = 2 * np.pi * t / n_theta
    xy = np.stack([r_a * np.cos(ang), r_a * np.sin(ang)], axis=1)
    h_loc = np.minimum(1.0, 2 * np.pi * r_a / n_theta)
    xy = xy + 0.2 * h_loc[:, None] * rng.uniform(-1.0, 1.0, size=xy.shape)

    def idx(aa, tt):
        return aa * n_theta + (tt % n_theta)

    e = [np.stack([idx(a, t), idx(a, t + 1)], axis=1)]
    inner = a + 1 < n_r
    e.append(np.stack([idx(a[inner], t[inner]), idx(a[inner] + 1, t[inner])], axis=1))
    e.append(np.stack([idx(a[inner], t[inner]), idx(a[inner] + 1, t[inner] + 1)], axis=1))
    edges = np.concatenate(e, axis=0).astype(np.int64)
    edges = np.sort(edges, axis=1)
    # n_theta == 2 would duplicate azimuthal edges; configs never go there
    edges = np.unique(edges, axis=0)
    w = 1.0 / np.linalg.norm(xy[edges[:, 0]] - xy[edges[:, 1]], axis=1)
    return edges, w, xy


def make_workload(name: str = "C0", *, mesh=None, n_phi=None, levels=None, sigma=None, beta=None, delta=None,
                  b=None, seed=None, nonaxisymmetric=None, shuffle: bool = False, noise_chunk: int = 4096,
                  want_rhs: bool = True, prism=None) -> Workload:
    """Build one workload.  ``name`` selects a row of CONFIGS; keyword arguments override single fields
    (used by the tests for reduced-size variants of the same recipe)."""
    cfg = dict(CONFIGS[name]) if name in CONFIGS else {}
    for k, v in dict(mesh=mesh, n_phi=n_phi, levels=levels, sigma=sigma, beta=beta, delta=delta, b=b, seed=seed,
                     nonaxisymmetric=nonaxisymmetric, prism=prism).items():
        if v is not None:
            cfg[k] = v
    cfg.setdefault("nonaxisymmetric", False)
    cfg.setdefault("prism", False)
    n_r, n_theta = cfg["mesh"]
    n_phi_, b_ = int(cfg["n_phi"]), int(cfg["b"])
    sigma_, beta_, delta_ = float(cfg["sigma"]), float(cfg["beta"]), float(cfg["delta"])
    seed_ = int(cfg["seed"])
    if n_phi_ < 3:
        raise ValueError("generator needs n_phi >= 3 on the fine level (planes k-1 and k+1 must differ)")
    n_pol = n_r * n_theta
    n = n_pol * n_phi_

    edges, w, _ = poloidal_mesh(n_r, n_theta, _rng(seed_, 1))
    if shuffle:  # C4 "shuffled" variant: same permutation of node numbers in every plane
        perm = _rng(seed_, 7).permutation(n_pol)
        edges = np.sort(perm[edges], axis=1)
    QS, lamS = _spd(_rng(seed_, 2), b_)
    QT, lamT = _spd(_rng(seed_, 3), b_)
    S = (QS * lamS[None, :]) @ QS.T
    T = (QT * lamT[None, :]) @ QT.T
    S = 0.5 * (S + S.T)
    T = 0.5 * (T + T.T)

    nonaxi = bool(cfg["nonaxisymmetric"])
    planes = np.arange(n_phi_)
    if nonaxi:  # D4
        r4 = _rng(seed_, 4)
        theta_node = r4.uniform(0.0, 2 * np.pi, size=n_pol)
        psi_c = r4.uniform(0.0, 2 * np.pi, size=b_)
        m_node = 1.0 + 0.3 * np.sin(2 * np.pi * planes[:, None] / n_phi_ + theta_node[None, :])  # [k, i]
        w_k = w[None, :] * 0.5 * (m_node[:, edges[:, 0]] + m_node[:, edges[:, 1]])  # [k, E]
        lam_k = lamS[None, :] * (1.0 + 0.3 * np.sin(2 * np.pi * planes[:, None] / n_phi_ + psi_c[None, :]))
    else:
        w_k = np.broadcast_to(w[None, :], (n_phi_, w.shape[0]))
        lam_k = None

    # ---- pattern: COO of all blocks, then sort by (row, col) -------------------------------------------------
    E = edges.shape[0]
    i_all = np.arange(n_pol, dtype=np.int64)
    rows, cols, kind, ref, dpl = [], [], [], [], []   # dpl: plane offset of the column (-1, 0, +1)
    prism_ = bool(cfg["prism"])
    if prism_ and n_phi_ < 3:
        raise ValueError("the prism stencil needs n_phi >= 3")
    for k in range(n_phi_):
        base = k * n_pol
        rows += [base + i_all, base + edges[:, 0], base + edges[:, 1], base + i_all, base + i_all]
        cols += [base + i_all, base + edges[:, 1], base + edges[:, 0],
                 ((k - 1) % n_phi_) * n_pol + i_all, ((k + 1) % n_phi_) * n_pol + i_all]
        kind += [np.full(n_pol, 0, np.int8), np.full(E, 1, np.int8), np.full(E, 1, np.int8),
                 np.full(n_pol, 2, np.int8), np.full(n_pol, 2, np.int8)]
        ref += [i_all, np.arange(E, dtype=np.int64), np.arange(E, dtype=np.int64), i_all, i_all]
        dpl += [np.zeros(n_pol, np.int8), np.zeros(E, np.int8), np.zeros(E, np.int8),
                np.full(n_pol, -1, np.int8), np.full(n_pol, 1, np.int8)]
        if prism_:  # edge blocks to the neighbouring planes: (i,k)-(j,k+-1)
            for dk in (-1, 1):
                nb = ((k + dk) % n_phi_) * n_pol
                rows += [base + edges[:, 0], base + edges[:, 1]]
                cols += [nb + edges[:, 1], nb + edges[:, 0]]
                kind += [np.full(E, 3, np.int8), np.full(E, 3, np.int8)]
                ref += [np.arange(E, dtype=np.int64), np.arange(E, dtype=np.int64)]
                dpl += [np.full(E, dk, np.int8), np.full(E, dk, np.int8)]
    rows = np.concatenate(rows)
    cols = np.concatenate(cols)
    kind = np.concatenate(kind)
    ref = np.concatenate(ref)
    dpl = np.concatenate(dpl)
    order = np.lexsort((cols, rows))
    rows, cols, kind, ref, dpl = rows[order], cols[order], kind[order], ref[order], dpl[order]
    nnzb = rows.shape[0]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(row_ptr, rows + 1, 1)
    row_ptr = np.cumsum(row_ptr)
    col_idx = cols.astype(np.int32)
    plane_of_row = rows // n_pol

    # ---- deterministic part of the values ---------------------------------------------------------------------
    vals = np.empty((nnzb, b_, b_), dtype=np.float64)
    eye = np.eye(b_)
    def S_of(k):
        if lam_k is None:
            return S
        Sk_ = (QS * lam_k[k][None, :]) @ QS.T
        return 0.5 * (Sk_ + Sk_.T)

    def wsum_of(k):
        ws_ = np.zeros(n_pol)
        np.add.at(ws_, edges[:, 0], w_k[k])
        np.add.at(ws_, edges[:, 1], w_k[k])
        return ws_

    if prism_:
        # A = sigma I + sum over toroidal intervals (k, k+1) of W_{k+1/2} (x) [[1/3, 1/6], [1/6, 1/3]] + beta circ(-1,2,-1) (x) I (x) T,
        # W_k = L_w^(k) (x) S^(k), W_{k+1/2} = (W_k + W_{k+1}) / 2: a sum of positive semi-definite Kronecker products (linear
        # finite-element mass coupling along the torus).  Axisymmetric case: (L_w (x) S) (x) circ(1/6, 2/3, 1/6).
        for k in range(n_phi_):
            km, kp = (k - 1) % n_phi_, (k + 1) % n_phi_
            Sm, S0, Sp = S_of(km), S_of(k), S_of(kp)
            wm, w0, wp = wsum_of(km), wsum_of(k), wsum_of(kp)
            sel = np.nonzero(plane_of_row == k)[0]
            kd, rf, dp_ = kind[sel], ref[sel], dpl[sel]
            m = kd == 0
            vals[sel[m]] = sigma_ * eye[None] + (2.0 * beta_) * T[None] + (1.0 / 3.0) * (
                0.5 * wm[rf[m]][:, None, None] * Sm[None] + w0[rf[m]][:, None, None] * S0[None] + 0.5 * wp[rf[m]][:, None, None] * Sp[None])
            m = kd == 1
            vals[sel[m]] = (-1.0 / 3.0) * (0.5 * w_k[km][rf[m]][:, None, None] * Sm[None] + w_k[k][rf[m]][:, None, None] * S0[None]
                                           + 0.5 * w_k[kp][rf[m]][:, None, None] * Sp[None])
            for dk, Sn, wn, kn in ((-1, Sm, wm, km), (1, Sp, wp, kp)):
                m = (kd == 2) & (dp_ == dk)
                vals[sel[m]] = (1.0 / 12.0) * (w0[rf[m]][:, None, None] * S0[None] + wn[rf[m]][:, None, None] * Sn[None]) - beta_ * T[None]
                m = (kd == 3) & (dp_ == dk)
                vals[sel[m]] = (-1.0 / 12.0) * (w_k[k][rf[m]][:, None, None] * S0[None] + w_k[kn][rf[m]][:, None, None] * Sn[None])
    for k in range(n_phi_ if not prism_ else 0):
        Sk = S_of(k)
        wsum = wsum_of(k)
        sel = np.nonzero(plane_of_row == k)[0]
        kd, rf = kind[sel], ref[sel]
        d = sel[kd == 0]
        vals[d] = sigma_ * eye[None] + wsum[rf[kd == 0]][:, None, None] * Sk[None] + (2.0 * beta_) * T[None]
        o = sel[kd == 1]
        vals[o] = (-w_k[k][rf[kd == 1]])[:, None, None] * Sk[None]
        t_ = sel[kd == 2]
        vals[t_] = (-beta_) * T[None]

    # ---- D3 noise: one Gaussian block per undirected stored pair, skew-symmetric placement -----------------------
    if delta_ != 0.0:
        up = np.nonzero(rows < cols)[0]
        key = rows * n + cols  # strictly increasing in CSR order
        mate = np.searchsorted(key, cols[up] * n + rows[up])
        assert np.array_equal(key[mate], cols[up] * n + rows[up]), "pattern is not structurally symmetric"
        coef = np.where(kind[up] == 1, w_k[plane_of_row[up], ref[up]], beta_)
        if prism_:
            coef = np.where(kind[up] == 3, w_k[plane_of_row[up], ref[up]] / 6.0, coef)
        rng_n = _rng(seed_, 5)
        scale = delta_ / np.sqrt(b_)
        for s in range(0, up.shape[0], noise_chunk):
            sl = slice(s, min(s + noise_chunk, up.shape[0]))
            G = rng_n.standard_normal((sl.stop - sl.start, b_, b_))
            G *= (scale * coef[sl])[:, None, None]
            vals[up[sl]] += G
            vals[mate[sl]] -= np.transpose(G, (0, 2, 1))

    rhs = _rng(seed_, 6).uniform(-1.0, 1.0, size=n * b_) if want_rhs else None
    return Workload(name=name, b=b_, n_r=n_r, n_theta=n_theta, n_phi=n_phi_, levels=int(cfg["levels"]),
                    sigma=sigma_, beta=beta_, delta=delta_, seed=seed_, row_ptr=row_ptr, col_idx=col_idx,
                    vals=vals, rhs=rhs, S=S, T=T, adj_w=(edges, np.array(w_k[0])))


def input_vector(n: int, seed: int, stream: int = 11) -> np.ndarray:
    """D5: U[-1,1] input vector for kernel tests."""
    return _rng(seed, stream).uniform(-1.0, 1.0, size=n)
