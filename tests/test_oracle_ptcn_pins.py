"""Pins for the PT-CN oracle (oracle/ptcn_ref.py; Eq. (4)-(5), Algorithm 1).  CPU only.

  P1 stationary states: for a linear H (no exchange, no density coupling) and Psi_n = eigenvectors of H, R_n = 0 and
     Psi_{n+1} = Psi_n -- the parallel-transport gauge removes the phase dynamics entirely ("residual type term").
  P2 exact propagator: for a linear H the gauge-invariant density matrix P = Psi Psi^* after one step agrees with
     U P U^*, U = exp(-i H dt), to third order in dt (Crank-Nicolson): halving dt divides the error by ~8.  A wrong sign of i,
     a missing 1/2 or a wrong projector term changes the order.  H is built as a dense matrix with explicit exponentials
     (no FFT), U from numpy's eigendecomposition.
  P3 the converged Psi_f satisfies Eq. (5) with the full model (exchange + density coupling), evaluated here from the
     definition; the output is orthonormal.
     The residual of Eq. (5) is evaluated at the un-orthogonalised fixed point with H_f rebuilt from Psi_f (bar 1e-9).
  P5 kinetic operator: plane waves are eigenfunctions with eigenvalue |G|^2 / 2.
  P6 H[Psi] Psi with exchange AND density coupling against a dense N x N matrix assembled point by point on 4^3 (explicit
     exponentials, v(G) typed out here, no FFT): sign and weight of every term of the model Hamiltonian (Alg. 1 line 5).
  P7 the Anderson update (Alg. 1 line 7): on linear residuals R_j(x) = A_j x - b_j of dimension d, one system
     per wavefunction, full-depth mixing with beta = 1 reaches the exact solutions within d + 1 iterations (Krylov
     property of Anderson's method); plain mixing does not, and neither would one least-squares problem shared by the
     wavefunctions.
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
    # Eq. (5) from its definition (Alg. 1 lines 5-6), at the un-orthogonalised fixed point Psi_f the oracle
    # hands out: H_f is REBUILT here from Psi_f (density and exchange operator), so an oracle that froze the Hamiltonian at
    # Psi_n during the iteration (residual 1.8e-3 in that mutant) or dropped a term of line 6 fails the 1e-9 bar.
    def eq5_residual(pf, pn):
        def hres(p):
            hp = model.h_apply(p)
            s = model.w * np.einsum("mr,nr->mn", p.reshape(3, -1).conj(), hp.reshape(3, -1))
            return hp - np.einsum("mr,mn->nr", p.reshape(3, -1), s).reshape(p.shape)
        return pf + 0.5j * dt * hres(pf) - (pn - 0.5j * dt * hres(pn))
    r = eq5_residual(info["psi_f"], psi0)
    nrm = math.sqrt(model.w * np.sum(np.abs(r) ** 2) / 3)
    assert nrm <= 1e-9, nrm
    # the step is not trivial: the fixed point is far (on the 1e-9 scale) from both Psi_n and the explicit half step
    assert np.abs(info["psi_f"] - psi0).max() > 1e-3 * np.abs(psi0).max()
    # the orthonormalised output spans the same space (line 11 only mixes the columns of Psi_f)
    pf = info["psi_f"].reshape(3, -1)
    proj = out.reshape(3, -1).T @ (model.w * (out.reshape(3, -1).conj() @ pf.T))       # P_out Psi_f
    assert np.abs(proj - pf.T).max() <= 1e-11 * np.abs(pf).max()
    # and its density matrix is gauge invariant: mixing Psi_n by a unitary first gives the same P_{n+1}
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3)))
    out2, _ = ptcn_ref.ptcn_step(model, np.ascontiguousarray(np.einsum("mr,mn->nr", psi0.reshape(3, -1), q).reshape(psi0.shape)),
                                 dt=dt, tol=1e-11, max_iter=100)
    p1 = out.reshape(3, -1).T @ out.reshape(3, -1).conj()
    p2 = out2.reshape(3, -1).T @ out2.reshape(3, -1).conj()
    assert np.abs(p1 - p2).max() <= 1e-8 * np.abs(p1).max()


def test_P6_h_apply_with_exchange_and_density_coupling_matches_a_dense_matrix():
    n, edges = (4, 4, 4), (5.0, 6.0, 7.0)
    N = 64
    cell = [edges[0], 0, 0, 0, edges[1], 0, 0, 0, edges[2]]
    rng = np.random.default_rng(21)
    v = 0.3 * rng.standard_normal(n)
    alpha, g, omega = 0.25, 0.7, 0.106
    psi = rng.standard_normal((3,) + n) + 1j * rng.standard_normal((3,) + n)
    model = ptcn_ref.Model(cell, n, kernel=1, omega=omega, alpha=alpha, v_ext=v, g=g)
    got = model.h_apply(np.ascontiguousarray(psi)).reshape(3, N)
    # dense H[Psi] = T + diag(v + g rho) + V_X[Psi], V_X(r, r') = -alpha sum_i psi_i(r) K(r - r') conj(psi_i(r')),
    # K(d) = (1/N) sum_G v(G) exp(i G d) (include/ptfock.h: unnormalised forward DFT, 1/N on the inverse, no volume factor)
    P = psi.reshape(3, N)
    rho = (np.abs(P) ** 2).sum(0)
    H = _dense_h(edges, n, v + g * rho.reshape(n))
    idx = np.array([(a, b, c) for a in range(4) for b in range(4) for c in range(4)])
    K = np.zeros((N, N), dtype=complex)
    for k0 in range(4):
        for k1 in range(4):
            for k2 in range(4):
                m = [k if k < 2 else k - 4 for k in (k0, k1, k2)]
                G2 = sum((2 * np.pi * m[d] / edges[d]) ** 2 for d in range(3))
                vg = np.pi / omega ** 2 if G2 == 0 else 4 * np.pi / G2 * (1.0 - math.exp(-G2 / (4 * omega ** 2)))
                ph = np.exp(2j * np.pi * (k0 * idx[:, 0] + k1 * idx[:, 1] + k2 * idx[:, 2]) / 4)
                K += vg / N * np.outer(ph, ph.conj())
    VX = -alpha * sum(np.outer(P[i], P[i].conj()) for i in range(3)) * K
    ref = (H + VX) @ P.T                                               # [r, j]
    assert np.abs(got.T - ref).max() <= 1e-12 * np.abs(ref).max()
    # each term matters at this bar
    assert np.abs(VX @ P.T).max() > 1e-3 * np.abs(ref).max() and np.abs(g * rho[:, None] * P.T).max() > 1e-3 * np.abs(ref).max()


def test_P7_anderson_update_solves_linear_systems_in_d_plus_1_iterations():
    d, n_e = 5, 3
    rng = np.random.default_rng(33)
    A = [np.eye(d) + 0.35 * (rng.standard_normal((d, d)) + 1j * rng.standard_normal((d, d))) / math.sqrt(d) for _ in range(n_e)]
    b = rng.standard_normal((n_e, d)) + 1j * rng.standard_normal((n_e, d))
    exact = np.array([np.linalg.solve(A[j], b[j]) for j in range(n_e)])
    res = lambda x: np.array([A[j] @ x[j] - b[j] for j in range(n_e)])

    def iterate(update, iters):
        x = np.zeros((n_e, d, 1, 1), dtype=complex)                     # [n_e, grid]: the layout ptcn_step uses
        xs, rs = [], []
        for _ in range(iters):
            xs.append(x.copy())
            rs.append(res(x.reshape(n_e, d)).reshape(x.shape))
            x = update(xs, rs)
        return x.reshape(n_e, d)

    x = iterate(lambda xs, rs: ptcn_ref.anderson_update(xs, rs, 1.0, 0.37), d + 1)
    assert np.abs(x - exact).max() <= 1e-9 * np.abs(exact).max()
    # plain mixing x - R(x) is nowhere near after the same number of steps: the history term does the work
    y = iterate(lambda xs, rs: xs[-1] - rs[-1], d + 1)
    assert np.abs(y - exact).max() > 1e-4 * np.abs(exact).max()
    # with d iterations (history one short) the solution is not reached yet: it is the Krylov dimension that counts
    z = iterate(lambda xs, rs: ptcn_ref.anderson_update(xs, rs, 1.0, 0.37), d - 1)
    assert np.abs(z - exact).max() > 1e-6 * np.abs(exact).max()
