"""Pins for the dense-algebra oracle (oracle/ptdense_ref.c; Alg. 3, Sec. 3.4) against what the
paper and the mathematics fix: plane-wave closed forms, invariants, a hand-worked Cholesky factor, and classical
Gram-Schmidt written with scalar Python loops.  CPU only; nothing here calls the CUDA path.

  D1 plane waves phi_m = exp(i G_m r) / sqrt(Omega): S = I; with H = -1/2 Laplacian (H phi_m = |G_m|^2/2 phi_m):
     Psi^* H Psi = diag(|G_m|^2 / 2), R_n = 0, rho = n / Omega, R_f = Psi_f - Psi_half.
  D2 seeded orthonormal orbitals (made by a different code: Loewdin in torch): S = I; sum_r rho Omega/N = n.
  D3 R_n is orthogonal to Psi for orthonormal Psi and ANY H Psi; R_f by hand from the definition on a tiny case.
  D4 rotate: identity, associativity with overlap (Psi^* (Psi S) = (Psi^* Psi) S), a scalar-loop brute force.
  D5 Cholesky: the 2 x 2 factor worked by hand, L L^H = S, lower triangular with positive real diagonal, failure on an
     indefinite matrix.
  D6 orthonormalize = classical Gram-Schmidt (scalar loops), gives S = I, keeps the span (projector), leaves an
     orthonormal set alone, first column only normalised.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1905_01348_b200 import synth

TOL = 1e-12


def _planewaves(n, edges, ms):
    n0, n1, n2 = n
    vol = edges[0] * edges[1] * edges[2]
    x = np.meshgrid(np.arange(n0) / n0, np.arange(n1) / n1, np.arange(n2) / n2, indexing="ij")
    out, g2 = [], []
    for m in ms:
        out.append(np.exp(2j * np.pi * (m[0] * x[0] + m[1] * x[1] + m[2] * x[2])) / math.sqrt(vol))
        g2.append(sum((2 * np.pi * m[d] / edges[d]) ** 2 for d in range(3)))
    return np.ascontiguousarray(np.array(out)), np.array(g2), vol


def test_D1_plane_wave_closed_forms():
    n, edges = (8, 6, 4), (7.0, 5.0, 3.0)
    ms = [(0, 0, 0), (1, 0, 0), (0, -2, 1), (3, 1, -1), (-2, 2, 1)]
    psi, g2, vol = _planewaves(n, edges, ms)
    N = n[0] * n[1] * n[2]
    w = vol / N
    s = oracle.overlap(psi, psi, w)
    assert np.abs(s - np.eye(len(ms))).max() <= TOL
    hpsi = np.ascontiguousarray(psi * (0.5 * g2)[:, None, None, None])
    sh = oracle.overlap(psi, hpsi, w)
    assert np.abs(sh - np.diag(0.5 * g2)).max() <= TOL * max(1.0, g2.max())
    assert np.abs(oracle.residual(psi, hpsi, w)).max() <= 1e-12 * np.abs(hpsi).max()
    rho = oracle.density(psi)
    assert np.abs(rho - len(ms) / vol).max() <= TOL
    half = np.ascontiguousarray(0.5 * psi[::-1])
    rf = oracle.residual(psi, hpsi, w, dt=0.37, psi_half=half)
    assert np.abs(rf - (psi - half)).max() <= 1e-12


def test_D1_wrong_conjugate_or_weight_would_fail():
    """conj on the wrong factor turns S[m, n] for distinct plane waves into delta(G_m + G_n): not the identity."""
    n, edges = (8, 6, 4), (7.0, 5.0, 3.0)
    psi, _, vol = _planewaves(n, edges, [(1, 0, 0), (-1, 0, 0)])
    w = vol / (8 * 6 * 4)
    s = oracle.overlap(psi, psi, w)
    wrong = w * np.einsum("mr,nr->mn", psi.reshape(2, -1), psi.reshape(2, -1))
    assert np.abs(s - np.eye(2)).max() <= TOL and abs(wrong[0, 1] - 1.0) <= TOL and abs(wrong[0, 0]) <= TOL


def test_D2_seeded_orbitals_are_orthonormal_and_density_counts_electrons():
    cfg = synth.Config("d2", (9.0, 10.0, 11.0), (16, 16, 16), 7, synth.KERNEL_HSE)
    psi = synth.orbitals(cfg, device="cpu").numpy()
    w = cfg.volume / cfg.N
    s = oracle.overlap(psi, psi, w)
    assert np.abs(s - np.eye(7)).max() <= 1e-12
    assert np.abs(s - s.conj().T).max() <= 1e-15
    rho = oracle.density(psi)
    assert rho.min() >= 0.0 and abs(rho.sum() * w - 7.0) <= 1e-12


def test_D3_residual_is_orthogonal_to_psi_and_matches_the_definition():
    cfg = synth.Config("d3", (9.0, 10.0, 11.0), (8, 8, 8), 4, synth.KERNEL_HSE, ecut=4.0)
    psi = synth.orbitals(cfg, device="cpu").numpy()
    rng = np.random.default_rng(3)
    hpsi = rng.standard_normal(psi.shape) + 1j * rng.standard_normal(psi.shape)
    half = rng.standard_normal(psi.shape) + 1j * rng.standard_normal(psi.shape)
    w = cfg.volume / cfg.N
    rn = oracle.residual(psi, hpsi, w)
    assert np.abs(oracle.overlap(psi, rn, w)).max() <= 1e-12 * np.abs(hpsi).max()        # Psi^* R_n = S - S = 0
    # definition with scalar loops on a few points
    N = cfg.N
    P, H = psi.reshape(4, N), hpsi.reshape(4, N)
    S = np.zeros((4, 4), dtype=complex)
    for m in range(4):
        for k in range(4):
            S[m, k] = w * sum(P[m, r].conjugate() * H[k, r] for r in range(N))
    dt = 0.21
    rf = oracle.residual(psi, hpsi, w, dt=dt, psi_half=half).reshape(4, N)
    for k in range(4):
        for r in (0, 17, N - 1):
            t = sum(P[m, r] * S[m, k] for m in range(4))
            assert abs(rn.reshape(4, N)[k, r] - (H[k, r] - t)) <= 1e-12
            assert abs(rf[k, r] - (P[k, r] + 0.5j * dt * (H[k, r] - t) - half.reshape(4, N)[k, r])) <= 1e-12


def test_D4_rotate():
    rng = np.random.default_rng(4)
    a = rng.standard_normal((5, 4, 3, 2)) + 1j * rng.standard_normal((5, 4, 3, 2))
    s = rng.standard_normal((5, 3)) + 1j * rng.standard_normal((5, 3))
    out = oracle.rotate(a, s)
    assert out.shape == (3, 4, 3, 2)
    for k in range(3):
        for idx in ((0, 0, 0), (3, 2, 1), (1, 1, 0)):
            assert abs(out[(k,) + idx] - sum(a[(m,) + idx] * s[m, k] for m in range(5))) <= 1e-13
    assert np.abs(oracle.rotate(a, np.eye(5, dtype=complex)) - a).max() == 0.0
    w = 0.3
    lhs = oracle.overlap(a, out, w)
    rhs = oracle.overlap(a, a, w) @ s
    assert np.abs(lhs - rhs).max() <= 1e-12 * np.abs(rhs).max()


def test_D5_cholesky():
    # hand-worked: S = [[4, 2 - 2i], [2 + 2i, 11]] -> L = [[2, 0], [1 + i, 3]]  (|1 + i|^2 + 9 = 11)
    s = np.array([[4.0, 2.0 - 2.0j], [2.0 + 2.0j, 11.0]], dtype=complex)
    l = oracle.cholesky(s)
    assert np.abs(l - np.array([[2.0, 0.0], [1.0 + 1.0j, 3.0]])).max() <= 1e-15
    rng = np.random.default_rng(5)
    for n in (1, 3, 17, 64):
        m = rng.standard_normal((n, n + 3)) + 1j * rng.standard_normal((n, n + 3))
        s = m @ m.conj().T + 0.1 * np.eye(n)
        l = oracle.cholesky(np.ascontiguousarray(s))
        assert np.abs(np.triu(l, 1)).max() == 0.0 and np.abs(np.diag(l).imag).max() == 0.0 and np.diag(l).real.min() > 0.0
        assert np.abs(l @ l.conj().T - s).max() <= 1e-13 * np.abs(s).max()
    with pytest.raises(RuntimeError):
        oracle.cholesky(np.array([[1.0, 2.0], [2.0, 1.0]], dtype=complex))


def test_D6_orthonormalize_is_gram_schmidt():
    rng = np.random.default_rng(6)
    n, shape = 5, (4, 3, 5)
    N = 60
    psi = rng.standard_normal((n,) + shape) + 1j * rng.standard_normal((n,) + shape)
    w = 0.7
    out = oracle.orthonormalize(psi, w)
    assert np.abs(oracle.overlap(out, out, w) - np.eye(n)).max() <= 1e-12
    # classical Gram-Schmidt, scalar loops, columns in order
    P = psi.reshape(n, N)
    Q = np.zeros_like(P)
    for c in range(n):
        v = P[c].copy()
        for m in range(c):
            proj = w * sum(Q[m, r].conjugate() * P[c, r] for r in range(N))
            v = v - proj * Q[m]
        Q[c] = v / math.sqrt(w * sum(abs(v[r]) ** 2 for r in range(N)))
    assert np.abs(out.reshape(n, N) - Q).max() <= 1e-12
    # same span: the projector Psi S^-1 Psi^* is unchanged
    s = oracle.overlap(psi, psi, w)
    proj_in = P.T @ np.linalg.inv(s) @ P.conj()
    proj_out = out.reshape(n, N).T @ out.reshape(n, N).conj()
    assert np.abs(proj_in - proj_out).max() <= 1e-12
    # an orthonormal set is a fixed point; the first column is only normalised
    again = oracle.orthonormalize(out, w)
    assert np.abs(again - out).max() <= 1e-13
    assert np.abs(out[0] - psi[0] / math.sqrt(w * np.sum(np.abs(psi[0]) ** 2))).max() <= 1e-14
