"""CPU ORACLE for one parallel-transport Crank-Nicolson (PT-CN) time step with a model Hamiltonian (TEST INFRASTRUCTURE, not
the product; only tests/ may import it; it shares no code with paper_1905_01348_b200/).

Follows PAPER.md:74-90 (Sec. 2, Algorithm 1) line by line, in the paper's notation, with plain numpy and the C oracle's
own routines (oracle.fft3d, oracle.apply, oracle.overlap / rotate / residual / density / orthonormalize):

    H[Psi] psi = -1/2 Laplacian psi + (v_ext + g rho[Psi]) psi + V_X[Psi] psi           (model; reading Q17)
    1  R_n = H_n Psi_n - Psi_n (Psi_n^* H_n Psi_n)                                       (signs: Eq. (4)/(5))
    2  Psi_{n+1/2} = Psi_n - (i dt / 2) R_n,  Psi_f = Psi_{n+1/2}
    3  rho_f
    4-10  repeat: H_f from Psi_f;  R_f = Psi_f + (i dt/2)(H_f Psi_f - Psi_f (Psi_f^* H_f Psi_f)) - Psi_{n+1/2};
          Anderson mixing of Psi_f (one least-squares problem PER WAVEFUNCTION); rho_f;
          stop when the density change is small
    11 orthogonalise Psi_f -> Psi_{n+1} (Cholesky + triangular solve)

Anderson mixing (reference [2] of the paper; fixed point of x -> x - R(x)), per wavefunction j, history depth <= m:
    gamma_j = argmin || R_k - dR gamma ||,  x_{k+1} = x_k - beta R_k - (dX - beta dR) gamma_j,
    dX = [x_k - x_{k-1}, ..., x_{k-m+1} - x_{k-m}],  dR likewise.

Pins: tests/test_oracle_ptcn_pins.py (stationary eigenstates, third-order agreement of the gauge-invariant density matrix
with the exact propagator of a linear H, the converged un-orthogonalised Psi_f satisfies Eq. (5) with H_f rebuilt from
Psi_f to 1e-9, orthonormal output, kinetic operator on plane waves, H[Psi] against a dense matrix built point by point on
4^3, the Anderson update solving per-wavefunction linear systems of dimension d in d + 1 iterations).
"""
from __future__ import annotations

import numpy as np

import oracle


def g2_table(cell, n) -> np.ndarray:
    """|G|^2 on the FFT grid, frequencies m_d in [-n_d/2, n_d/2), G = m0 b0 + m1 b1 + m2 b2, b_d rows of 2 pi inv(A)^T."""
    a = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    b = 2.0 * np.pi * np.linalg.inv(a).T
    ms = [np.where(np.arange(k) < (k + 1) // 2, np.arange(k), np.arange(k) - k) for k in n]
    m0, m1, m2 = np.meshgrid(ms[0], ms[1], ms[2], indexing="ij")
    g = m0[..., None] * b[0] + m1[..., None] * b[1] + m2[..., None] * b[2]
    return np.sum(g * g, axis=-1)


def kinetic_apply(cell, n, psi: np.ndarray) -> np.ndarray:
    """-1/2 Laplacian psi_j through the oracle's own FFT: IFFT[ |G|^2/2 FFT psi_j ]."""
    g2 = g2_table(cell, n)
    N = int(np.prod(n))
    out = np.empty_like(psi)
    for j in range(psi.shape[0]):
        f = oracle.fft3d(np.ascontiguousarray(psi[j]), -1)
        out[j] = oracle.fft3d(np.ascontiguousarray(0.5 * g2 * f), +1) / N
    return out


class Model:
    """cell (9), grid n (3), exchange kernel / omega / alpha (alpha = 0: no exchange), v_ext (real grid), density coupling g."""

    def __init__(self, cell, n, kernel=1, omega=0.106, alpha=0.25, v_ext=None, g=0.0):
        self.cell, self.n = list(cell), tuple(int(x) for x in n)
        self.kernel, self.omega, self.alpha, self.g = kernel, omega, alpha, g
        self.N = int(np.prod(self.n))
        self.volume = abs(float(np.linalg.det(np.asarray(cell, dtype=np.float64).reshape(3, 3))))
        self.w = self.volume / self.N
        self.v_ext = np.zeros(self.n) if v_ext is None else np.asarray(v_ext, dtype=np.float64)

    def h_apply(self, psi: np.ndarray) -> np.ndarray:
        """H[Psi] Psi: the density and the exchange operator are built from Psi itself."""
        v = self.v_ext + self.g * oracle.density(psi)
        out = kinetic_apply(self.cell, self.n, psi) + v[None] * psi
        if self.alpha != 0.0:
            out = out + oracle.apply(self.cell, self.n, self.kernel, self.omega, self.alpha, np.ascontiguousarray(psi))
        return np.ascontiguousarray(out)


def anderson_update(xs, rs, beta: float, w: float = 1.0) -> np.ndarray:
    """Line 7 of Algorithm 1: the next iterate from the stored iterates xs[0..m] and their residuals rs[0..m] (newest last),
    one least-squares problem PER WAVEFUNCTION j (the formula is the module header's):
        gamma_j = argmin || r_m[j] - dR_j gamma ||,   x_new[j] = x_m[j] - beta r_m[j] - (dX_j - beta dR_j) gamma_j.
    xs[k], rs[k]: arrays [n_e, ...]; w: weight of the inner product (a common factor, it cancels in gamma)."""
    m = len(xs) - 1
    x, r = xs[m], rs[m]
    new = x - beta * r
    if m > 0:
        for j in range(x.shape[0]):
            dx = np.array([(xs[m - a][j] - xs[m - a - 1][j]).ravel() for a in range(m)])
            dr = np.array([(rs[m - a][j] - rs[m - a - 1][j]).ravel() for a in range(m)])
            gram = w * (dr.conj() @ dr.T)
            rhs = w * (dr.conj() @ r[j].ravel())
            gram = gram + 1e-14 * np.trace(gram).real / m * np.eye(m)
            gamma = np.linalg.solve(gram, rhs)
            new[j] = new[j] - ((dx - beta * dr).T @ gamma).reshape(x[j].shape)
    return np.ascontiguousarray(new)


def ptcn_step(model: Model, psi_n: np.ndarray, dt: float, tol: float = 1e-10, max_iter: int = 60, beta: float = 1.0,
              depth: int = 20):
    """One PT-CN step (Algorithm 1).  Returns (psi_{n+1}, info)."""
    w = model.w
    n_e = psi_n.shape[0]
    h = model.h_apply(psi_n)
    r_n = oracle.residual(psi_n, h, w)                                   # line 1
    psi_half = psi_n - 0.5j * dt * r_n                                   # line 2
    psi_f = psi_half.copy()
    rho = oracle.density(psi_f)                                          # line 3
    xs, rs = [], []
    info = {"iterations": 0, "rho_change": None, "residual": None}
    for it in range(max_iter):                                           # lines 4-10
        h = model.h_apply(psi_f)                                         # line 5
        r_f = oracle.residual(psi_f, h, w, dt=dt, psi_half=np.ascontiguousarray(psi_half))      # line 6
        info["residual"] = float(np.sqrt(w * np.sum(np.abs(r_f) ** 2) / n_e))
        if info["residual"] < tol:                                       # "when the residual is sufficiently small"
            break
        xs.append(psi_f.copy())
        rs.append(r_f.copy())
        if len(xs) > depth + 1:
            xs.pop(0)
            rs.pop(0)
        psi_f = anderson_update(xs, rs, beta, w)                         # line 7: Anderson mixing, per wavefunction
        rho_new = oracle.density(psi_f)                                  # line 8
        change = float(np.abs(rho_new - rho).sum() * w / n_e)
        rho = rho_new
        info.update(iterations=it + 1, rho_change=change)                # line 9: the density change is reported; the
        #                                                                  residual (checked above) decides
    info["psi_f"] = psi_f.copy()                                         # the fixed point of Eq. (5) before line 11 (for the pins)
    return oracle.orthonormalize(psi_f, w), info                         # line 11
