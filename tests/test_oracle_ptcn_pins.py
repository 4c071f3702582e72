"""Pins for the PT-CN oracle (oracle/ptcn_ref.py; Eq. (4)-(5), Algorithm 1).  CPU only.

  P1 stationary states: for a linear H (no exchange, no density coupling) and Psi_n = eigenvectors of H, R_n = 0 and
     Psi_{n+1} = Psi_n -- the parallel-transport gauge removes the phase dynamics entirely ("residual type term").
  P2 exact propagator: for a linear H the gauge-invariant density matrix P = Psi Psi^* after one step agrees with
     U P U^*, U = exp(-i H dt), to third order in dt (Crank-Nicolson): halving dt divides the error by ~8.  A wrong sign of i,
     a missing 1/2 or a wrong projector term changes the order.  H is built as a dense matrix with explicit exponentials
     (no FFT), U from numpy's eigendecomposition.
  P3 the converged Psi_f satisfies Eq. (5) with the full model (exchange + density coupling), evaluated here from the
     definition; the output is orthonormal.
  P5 kinetic operator: plane waves are eigenfunctions with eigenvalue |G|^2 / 2.
"""
import math

import numpy as np

import oracle
from oracle import ptcn_ref


def _dense_h(cell_edges, n, v):
    """H = -1/2 Laplacian + diag(v) as a dense N x N matrix from explicit plane-wave sums (orthorhombic cell)."""
    n0, n1, n2 = n
    N = n0 * n1 * n2
    idx = np.array([(a, b, c) for a in range(n0) for b in range(n1) for c in range(n2)])
    fr = [np.array([k if k < (m + 1) // 2 else k - m for k in range(m)]) for m in n]
    T = np.zeros((N, N), dtype=complex)
    for k0 in range(n0):
        for k1 in range(n1):
            for k2 in range(n2):
                g = 2 * np.pi * np.array([fr[0][k0] / cell_edges[0], fr[1][k1] / cell_edges[1], fr[2][k2] / cell_edges[2]])
                ph = np.exp(2j * np.pi * (k0 * idx[:, 0] / n0 + k1 * idx[:, 1] / n1 + k2 * idx[:, 2] / n2))
                T += 0.5 * g.dot(g) / N * np.outer(ph, ph.conj())
    return T + np.diag(v.ravel())


def _setup(n=(4, 4, 4), edges=(5.0, 6.0, 7.0)):
    rng = np.random.default_rng(11)
    v = 0.3 * rng.standard_normal(n)
    cell = [edges[0], 0, 0, 0, edges[1], 0, 0, 0, edges[2]]
    model = ptcn_ref.Model(cell, n, alpha=0.0, v_ext=v, g=0.0)
    return model, _dense_h(edges, n, v), rng


def test_P5_kinetic_plane_wave():
    n, edges = (6, 4, 8), (5.0, 6.0, 7.0)
    cell = [edges[0], 0, 0, 0, edges[1], 0, 0, 0, edges[2]]
    x = np.meshgrid(*[np.arange(k) / k for k in n], indexing="ij")
    for m in [(1, 0, 0), (-2, 1, 3), (0, -1, -3)]:
        pw = np.exp(2j * np.pi * (m[0] * x[0] + m[1] * x[1] + m[2] * x[2]))[None]
        g2 = sum((2 * np.pi * m[d] / edges[d]) ** 2 for d in range(3))
        t = ptcn_ref.kinetic_apply(cell, n, np.ascontiguousarray(pw))
        assert np.abs(t - 0.5 * g2 * pw).max() <= 1e-12 * max(1.0, g2)


def test_P1_eigenstates_are_stationary_in_the_PT_gauge():
    model, H, _ = _setup()
    assert np.abs(H - H.conj().T).max() < 1e-12
    evals, evecs = np.linalg.eigh(H)
    psi = np.ascontiguousarray((evecs[:, :3].T / math.sqrt(model.w)).reshape((3,) + model.n))
    hp = model.h_apply(psi)
    assert np.abs(hp.reshape(3, -1) - (H @ psi.reshape(3, -1).T).T).max() <= 1e-11        # model H == dense H
    assert np.abs(oracle.residual(psi, hp, model.w)).max() <= 1e-11
    out, info = ptcn_ref.ptcn_step(model, psi, dt=0.8, tol=1e-12)
    assert np.abs(out - psi).max() <= 1e-10 and info["iterations"] <= 2


def test_P2_density_matrix_matches_the_exact_propagator_to_third_order():
    model, H, rng = _setup()
    N = model.N
    a = rng.standard_normal((2, N)) + 1j * rng.standard_normal((2, N))
    psi0 = oracle.orthonormalize(np.ascontiguousarray(a.reshape((2,) + model.n)), model.w)
    evals, V = np.linalg.eigh(H)
    errs = []
    for dt in (0.2, 0.1):
        out, info = ptcn_ref.ptcn_step(model, psi0, dt=dt, tol=1e-13, max_iter=200)
        U = (V * np.exp(-1j * evals * dt)) @ V.conj().T
        x0, x1 = psi0.reshape(2, N).T, out.reshape(2, N).T
        P_exact = U @ (x0 @ x0.conj().T) @ U.conj().T
        errs.append(np.abs(x1 @ x1.conj().T - P_exact).max() / np.abs(P_exact).max())
    assert errs[0] < 2e-2 and 6.0 < errs[0] / errs[1] < 10.5, errs


def test_P3_fixed_point_satisfies_eq5_and_output_is_orthonormal():
    n, edges = (8, 8, 8), (9.0, 10.0, 11.0)
    cell = [edges[0], 0, 0, 0, edges[1], 0, 0, 0, edges[2]]
    x = np.meshgrid(*[np.arange(k) / k for k in n], indexing="ij")
    v = 0.2 * np.cos(2 * np.pi * x[0]) + 0.1 * np.sin(2 * np.pi * (x[1] + x[2]))
    model = ptcn_ref.Model(cell, n, kernel=1, omega=0.106, alpha=0.25, v_ext=v, g=0.5)
    rng = np.random.default_rng(12)
    a = rng.standard_normal((3,) + n) + 1j * rng.standard_normal((3,) + n)
    sm = np.exp(-2.0 * ptcn_ref.g2_table(cell, n))                          # smooth the noise: low kinetic energy
    a = np.array([oracle.fft3d(np.ascontiguousarray(sm * oracle.fft3d(np.ascontiguousarray(z), -1)), +1) for z in a])
    psi0 = oracle.orthonormalize(np.ascontiguousarray(a), model.w)
    dt = 0.5
    out, info = ptcn_ref.ptcn_step(model, psi0, dt=dt, tol=1e-11, max_iter=100)
    assert info["residual"] < 1e-11 and info["iterations"] < 60
    assert np.abs(oracle.overlap(out, out, model.w) - np.eye(3)).max() <= 1e-12
    # Eq. (5) from its definition, at the un-orthogonalised fixed point: redo the iteration's last state by hand.
    # The orthonormalised output spans the same space; Eq. (5) is covariant under unitary mixing only, so the check
    # uses the residual the oracle reports AND an independent evaluation for a rotated copy of the fixed point.
    def eq5_residual(pf, pn):
        def hres(p):
            hp = model.h_apply(p)
            s = model.w * np.einsum("mr,nr->mn", p.reshape(3, -1).conj(), hp.reshape(3, -1))
            return hp - np.einsum("mr,mn->nr", p.reshape(3, -1), s).reshape(p.shape)
        return pf + 0.5j * dt * hres(pf) - (pn - 0.5j * dt * hres(pn))
    # the PT-CN solution stays orthonormal to O(dt^3) even before line 11, so `out` is within that of the fixed point
    r = eq5_residual(out, psi0)
    nrm = math.sqrt(model.w * np.sum(np.abs(r) ** 2) / 3)
    assert nrm < 5e-3 * dt
    # and its density matrix is gauge invariant: mixing Psi_n by a unitary first gives the same P_{n+1}
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3)))
    out2, _ = ptcn_ref.ptcn_step(model, np.ascontiguousarray(np.einsum("mr,mn->nr", psi0.reshape(3, -1), q).reshape(psi0.shape)),
                                 dt=dt, tol=1e-11, max_iter=100)
    p1 = out.reshape(3, -1).T @ out.reshape(3, -1).conj()
    p2 = out2.reshape(3, -1).T @ out2.reshape(3, -1).conj()
    assert np.abs(p1 - p2).max() <= 1e-8 * np.abs(p1).max()
