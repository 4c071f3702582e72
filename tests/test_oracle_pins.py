"""Pins for the CPU oracle (oracle/ptfock_ref.c) against things OTHER than itself.

The paper prints no value of V_X Psi, E_x or any intermediate, so the oracle is
pinned by what the mathematics fixes (BASELINE.json north_star):

T1 plane-wave closed form            -> Omega/N normalisation, sign, conj placement, v table incl. G = 0, index->G map
T2 O(N^2) real-space brute force      -> convolution theorem + the oracle's FFT (no FFT anywhere in the check)
T3 Hermiticity                        -> the x phi_i multiply and the i-sum
T4 unitary invariance                 -> V_X depends on Phi only through P = Phi Phi^*
T5 E_x real and <= 0                  -> energy formula
T6 FFT vs O(n^2) DFT, round trip, Parseval, delta, single mode
T7 periodic Poisson textbook case
T8 structure: W_ji = conj(W_ij), column subsets, linearity, real orbitals, grid shift

All CPU, all small: the whole file runs in well under a minute.
"""
import math
import os

import numpy as np
import pytest

import oracle

COUL, HSE = oracle.KERNEL_COULOMB, oracle.KERNEL_HSE
OMEGA = 0.106


def _v_of_g2(g2, kernel, omega):
    """The kernel formulas of BASELINE.json north_star, typed here independently of the oracle."""
    g2 = np.asarray(g2, dtype=np.float64)
    out = np.empty_like(g2)
    z = g2 == 0.0
    nz = ~z
    if kernel == COUL:
        out[z] = 0.0
        out[nz] = 4.0 * math.pi / g2[nz]
    else:
        out[z] = math.pi / omega ** 2
        out[nz] = 4.0 * math.pi / g2[nz] * (1.0 - np.exp(-g2[nz] / (4.0 * omega ** 2)))
    return out


def _recip(cell):
    a = np.asarray(cell, dtype=np.float64).reshape(3, 3)
    return 2.0 * math.pi * np.linalg.inv(a).T          # rows b_d, b_d . a_e = 2 pi delta


def _points_frac(n):
    x0, x1, x2 = np.meshgrid(*[np.arange(nd) / nd for nd in n], indexing="ij")
    return np.stack([x0, x1, x2], axis=-1)             # fractional coordinates, [n0,n1,n2,3]


def _plane_wave(n, m, volume):
    f = _points_frac(n)
    return np.exp(2j * math.pi * (f @ np.asarray(m, dtype=np.float64))) / math.sqrt(volume)


def _rng(seed):
    return np.random.default_rng(seed)


def _randc(rng, shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex128)


CELLS = {
    "ortho": [7.3, 0, 0, 0, 5.9, 0, 0, 0, 4.4],
    "skew": [7.3, 0.4, 0.0, -0.7, 5.9, 0.3, 0.2, -0.5, 4.4],
}


# --------------------------------------------------------------------------------------- T1
@pytest.mark.parametrize("kernel", [COUL, HSE])
@pytest.mark.parametrize("cellname", ["ortho", "skew"])
def test_T1_plane_wave_closed_form(kernel, cellname):
    """phi_i = exp(i G_i r)/sqrt(Omega)  =>  V_X phi_j = -(1/Omega) sum_i v(G_j - G_i) phi_j and
    E_x = -(1/(2 Omega)) sum_ij v(G_i - G_j)  (BASELINE.json north_star)."""
    n = (8, 6, 4)
    cell = CELLS[cellname]
    vol = abs(np.linalg.det(np.asarray(cell).reshape(3, 3)))
    b = _recip(cell)
    # distinct m_i whose pairwise differences stay inside [-n/2, n/2) on every axis
    ms = np.array([[0, 0, 0], [1, 0, 0], [-1, 1, 0], [2, -1, -1], [0, 1, -1], [1, 1, 0]])
    diffs = ms[:, None, :] - ms[None, :, :]
    for d in range(3):
        assert diffs[..., d].min() >= -(n[d] // 2) and diffs[..., d].max() < n[d] // 2
    phi = np.stack([_plane_wave(n, m, vol) for m in ms])
    alpha = 0.75 if kernel == HSE else 1.0
    out = oracle.apply(cell, n, kernel, OMEGA, alpha, phi)
    g = diffs.astype(np.float64) @ b                    # G_j - G_i, [j, i, 3]
    vji = _v_of_g2((g ** 2).sum(-1), kernel, OMEGA)
    coeff = -alpha / vol * vji.sum(axis=1)               # per j
    expect = coeff[:, None, None, None] * phi
    scale = np.abs(expect).max()
    assert scale > 0
    assert np.abs(out - expect).max() <= 1e-13 * scale
    e = oracle.exchange_energy(cell, n, phi, out)
    e_expect = -alpha / (2.0 * vol) * vji.sum()
    assert abs(e.real - e_expect) <= 1e-13 * abs(e_expect)
    assert abs(e.imag) <= 1e-13 * abs(e_expect)


def test_T1_wrong_conjugate_would_fail():
    """The closed form distinguishes conj(phi_i) psi_j from phi_i conj(psi_j) (reading Q8)."""
    n = (8, 6, 4)
    cell = CELLS["ortho"]
    vol = 7.3 * 5.9 * 4.4
    phi = np.stack([_plane_wave(n, m, vol) for m in ([1, 0, 0], [0, 1, 0])])
    psi = _plane_wave(n, [1, 1, 1], vol)[None]
    out = oracle.apply(cell, n, COUL, OMEGA, 1.0, phi, psi)
    # out must be proportional to psi itself (phi_i conj(phi_i) psi); the wrong conjugate gives exp(i(2G_i - G_j) r)
    ratio = out[0] / psi[0]
    assert np.abs(ratio - ratio.flat[0]).max() <= 1e-13 * abs(ratio.flat[0])


def test_T1_hse_g0_value_is_the_limit():
    """Reading Q2: v_HSE(G=0) = pi/omega^2 = 279.6006 bohr^2; bare v(0) = 0."""
    n = (4, 4, 4)
    v = oracle.vtable(CELLS["ortho"], n, HSE, OMEGA)
    assert v[0, 0, 0] == pytest.approx(math.pi / OMEGA ** 2, rel=1e-15)
    assert v[0, 0, 0] == pytest.approx(279.6006, rel=1e-6)
    assert oracle.vtable(CELLS["ortho"], n, COUL, OMEGA)[0, 0, 0] == 0.0
    # the limit is continuous: tiny G in a huge cell approaches it
    big = [4000.0, 0, 0, 0, 4000.0, 0, 0, 0, 4000.0]
    vb = oracle.vtable(big, n, HSE, OMEGA)
    assert vb[0, 0, 1] == pytest.approx(math.pi / OMEGA ** 2, rel=1e-3)


# --------------------------------------------------------------------------------------- T2
def _brute_force_apply(cell, n, kernel, omega, alpha, phi, psi):
    """Direct O(N^2) sums, no FFT: K(r) = (1/N) sum_k v(G_k) exp(+i G_k r), W = K (*) rho (circular)."""
    n = tuple(n)
    N = n[0] * n[1] * n[2]
    b = _recip(cell)
    idx = np.stack(np.meshgrid(*[np.arange(nd) for nd in n], indexing="ij"), axis=-1).reshape(N, 3)
    m = idx.copy()
    for d in range(3):
        m[:, d] = np.where(idx[:, d] < (n[d] + 1) // 2, idx[:, d], idx[:, d] - n[d])
    g2 = ((m.astype(np.float64) @ b) ** 2).sum(-1)
    v = _v_of_g2(g2, kernel, omega)
    frac = idx / np.asarray(n, dtype=np.float64)
    phase = np.exp(2j * math.pi * (frac @ idx.T.astype(np.float64)))    # [r, k] exp(+2 pi i sum k_d x_d / n_d)
    K = (phase @ v) / N                                                    # K(r), [N]
    # shift table: index of (r - r') mod n
    diff = (idx[:, None, :] - idx[None, :, :]) % np.asarray(n)
    lin = (diff[..., 0] * n[1] + diff[..., 1]) * n[2] + diff[..., 2]      # [r, r']
    Kmat = K[lin]
    out = np.zeros((psi.shape[0], N), dtype=np.complex128)
    for j in range(psi.shape[0]):
        for i in range(phi.shape[0]):
            rho = np.conj(phi[i].reshape(N)) * psi[j].reshape(N)
            W = Kmat @ rho
            out[j] -= alpha * phi[i].reshape(N) * W
    return out.reshape((psi.shape[0],) + n)


@pytest.mark.parametrize("n,kernel", [((8, 8, 8), HSE), ((8, 8, 8), COUL), ((4, 6, 8), HSE)])
def test_T2_brute_force_convolution(n, kernel):
    rng = _rng(11 + kernel)
    cell = CELLS["ortho"] if n[0] == n[1] else CELLS["skew"]
    phi = _randc(rng, (3,) + n)
    psi = _randc(rng, (2,) + n)
    got = oracle.apply(cell, n, kernel, OMEGA, 1.0, phi, psi)
    ref = _brute_force_apply(cell, n, kernel, OMEGA, 1.0, phi, psi)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()


# --------------------------------------------------------------------------------------- T3
@pytest.mark.parametrize("kernel", [COUL, HSE])
def test_T3_hermiticity(kernel):
    n = (6, 8, 4)
    rng = _rng(3)
    phi = _randc(rng, (4,) + n)            # random, not orthonormal
    vx = oracle.apply(CELLS["skew"], n, kernel, OMEGA, 1.0, phi)
    M = np.einsum("axyz,bxyz->ab", phi.conj(), vx)
    assert np.abs(M - M.conj().T).max() <= 1e-13 * np.abs(M).max()


# --------------------------------------------------------------------------------------- T4
def test_T4_unitary_invariance():
    n = (8, 4, 6)
    rng = _rng(4)
    phi = _randc(rng, (5,) + n)
    psi = _randc(rng, (2,) + n)
    q, _ = np.linalg.qr(_randc(rng, (5, 5)))
    phi_rot = np.ascontiguousarray(np.einsum("ab,bxyz->axyz", q, phi))
    a = oracle.apply(CELLS["ortho"], n, HSE, OMEGA, 1.0, phi, psi)
    b = oracle.apply(CELLS["ortho"], n, HSE, OMEGA, 1.0, phi_rot, psi)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()
    # self case: V_X[U Phi](U Phi) = U V_X[Phi] Phi
    s = oracle.apply(CELLS["ortho"], n, COUL, OMEGA, 1.0, phi)
    s_rot = oracle.apply(CELLS["ortho"], n, COUL, OMEGA, 1.0, phi_rot)
    assert np.abs(s_rot - np.einsum("ab,bxyz->axyz", q, s)).max() <= 1e-13 * np.abs(s).max()


# --------------------------------------------------------------------------------------- T5
@pytest.mark.parametrize("kernel", [COUL, HSE])
def test_T5_energy_real_and_nonpositive(kernel):
    n = (8, 8, 4)
    rng = _rng(5)
    phi = _randc(rng, (4,) + n)
    vx = oracle.apply(CELLS["ortho"], n, kernel, OMEGA, 1.0, phi)
    e = oracle.exchange_energy(CELLS["ortho"], n, phi, vx)
    assert e.real < 0.0
    assert abs(e.imag) <= 1e-13 * abs(e.real)
    # independent evaluation of the energy formula (reading Q11)
    vol = 7.3 * 5.9 * 4.4
    e2 = 0.5 * vol / (n[0] * n[1] * n[2]) * np.vdot(phi, vx)
    assert abs(e - e2) <= 1e-13 * abs(e2)


# --------------------------------------------------------------------------------------- T6
@pytest.mark.parametrize("nlen", [1, 2, 3, 4, 6, 8, 9, 12, 16, 32, 48, 64, 128, 5, 10, 15, 60, 90, 120])
def test_T6_fft1d_matches_definition(nlen):
    rng = _rng(nlen)
    x = _randc(rng, (nlen,))
    for sign in (-1, 1):
        ref = oracle.dft1d_naive(x, sign)
        got = oracle.fft1d(x, sign)
        assert np.abs(got - ref).max() <= 2e-14 * max(1.0, np.abs(ref).max())
    # delta at position p -> pure phase; single mode -> delta
    p = nlen // 3
    d = np.zeros(nlen, dtype=np.complex128)
    d[p] = 1.0
    pk = (p * np.arange(nlen)) % nlen                                  # exact argument reduction
    expect = np.exp(-2j * math.pi * pk / nlen)
    assert np.abs(oracle.fft1d(d, -1) - expect).max() <= 1e-14
    mode = np.exp(2j * math.pi * pk / nlen)
    spec = oracle.fft1d(mode, -1)
    e = np.zeros(nlen, dtype=np.complex128)
    e[p] = nlen
    assert np.abs(spec - e).max() <= 1e-13 * nlen


@pytest.mark.parametrize("n", [(4, 6, 8), (16, 16, 16), (12, 8, 3), (10, 15, 6)])
def test_T6_fft3d_roundtrip_parseval_and_definition(n):
    rng = _rng(sum(n))
    x = _randc(rng, n)
    f = oracle.fft3d(x, -1)
    N = n[0] * n[1] * n[2]
    assert np.vdot(f, f).real == pytest.approx(N * np.vdot(x, x).real, rel=1e-13)      # Parseval
    back = oracle.fft3d(f, +1) / N
    assert np.abs(back - x).max() <= 1e-14 * np.abs(x).max() * math.log2(N)
    # a few output points straight from the definition (3-D sum)
    fr = _points_frac(n)
    for k in [(0, 0, 0), (1, 2, 1), (n[0] - 1, n[1] - 1, n[2] - 1), (2, 0, n[2] // 2)]:
        ph = np.exp(-2j * math.pi * (fr @ np.asarray(k, dtype=np.float64)))
        assert abs(f[k] - (x * ph).sum()) <= 1e-12 * np.abs(f).max()


# --------------------------------------------------------------------------------------- T7
@pytest.mark.parametrize("kernel", [COUL, HSE])
def test_T7_periodic_poisson_textbook(kernel):
    """One constant orbital phi = 1/sqrt(Omega), psi = cos(G0 r): V_X psi = -(1/Omega) v(G0) cos(G0 r)."""
    n = (8, 6, 4)
    cell = CELLS["ortho"]
    vol = 7.3 * 5.9 * 4.4
    phi = np.full((1,) + n, 1.0 / math.sqrt(vol), dtype=np.complex128)
    m0 = np.array([2.0, -1.0, 1.0])
    fr = _points_frac(n)
    psi = np.cos(2.0 * math.pi * (fr @ m0)).astype(np.complex128)[None]
    g0 = m0 @ _recip(cell)
    expect = -(1.0 / vol) * _v_of_g2(np.array([(g0 ** 2).sum()]), kernel, OMEGA)[0] * psi
    got = oracle.apply(cell, n, kernel, OMEGA, 1.0, phi, psi)
    assert np.abs(got - expect).max() <= 1e-13 * np.abs(expect).max()


# --------------------------------------------------------------------------------------- T8
def test_T8_pair_symmetry_W_ji_is_conj_W_ij():
    n = (6, 4, 8)
    rng = _rng(8)
    a, b = _randc(rng, n), _randc(rng, n)
    # needs v(-G) = v(G) on the grid: true for orthorhombic cells; in a skew cell the Nyquist planes
    # (m = -n/2 only, reading Q5) break it, which the second half of the test shows.
    for kernel in (COUL, HSE):
        w_ab = oracle.pair_w(CELLS["ortho"], n, kernel, OMEGA, a, b)
        w_ba = oracle.pair_w(CELLS["ortho"], n, kernel, OMEGA, b, a)
        assert np.abs(w_ba - np.conj(w_ab)).max() <= 1e-13 * np.abs(w_ab).max()
    w_ab = oracle.pair_w(CELLS["skew"], n, HSE, OMEGA, a, b)
    w_ba = oracle.pair_w(CELLS["skew"], n, HSE, OMEGA, b, a)
    assert np.abs(w_ba - np.conj(w_ab)).max() > 1e-6 * np.abs(w_ab).max()


def test_T8_column_subset_linearity_real_shift():
    n = (4, 6, 8)
    cell = CELLS["ortho"]
    rng = _rng(80)
    phi = _randc(rng, (3,) + n)
    psi = _randc(rng, (4,) + n)
    full = oracle.apply(cell, n, HSE, OMEGA, 1.0, phi, psi)
    sub = oracle.apply(cell, n, HSE, OMEGA, 1.0, phi, psi, cols=[3, 1])
    assert np.array_equal(sub[0], full[3]) and np.array_equal(sub[1], full[1])
    # linearity in Psi
    c1, c2 = 0.3 - 1.1j, -2.0 + 0.5j
    comb = np.ascontiguousarray((c1 * psi[0] + c2 * psi[2])[None])
    lin = oracle.apply(cell, n, HSE, OMEGA, 1.0, phi, comb)[0]
    assert np.abs(lin - (c1 * full[0] + c2 * full[2])).max() <= 1e-13 * np.abs(full).max()
    # quadratic in Phi
    dbl = oracle.apply(cell, n, HSE, OMEGA, 1.0, np.ascontiguousarray(2.0 * phi), psi)
    assert np.abs(dbl - 4.0 * full).max() <= 1e-13 * np.abs(full).max()
    # alpha is a plain prefactor (reading Q1)
    half = oracle.apply(cell, n, HSE, OMEGA, 0.25, phi, psi)
    assert np.abs(half - 0.25 * full).max() <= 1e-14 * np.abs(full).max()
    # real orbitals -> real output
    pr = np.ascontiguousarray(phi.real.astype(np.complex128))
    qr = np.ascontiguousarray(psi.real.astype(np.complex128))
    re = oracle.apply(cell, n, COUL, OMEGA, 1.0, pr, qr)
    assert np.abs(re.imag).max() <= 1e-13 * np.abs(re.real).max()
    # translating every orbital by a grid vector translates the output
    sh = (1, 2, 3)
    rolled = oracle.apply(cell, n, HSE, OMEGA, 1.0, np.ascontiguousarray(np.roll(phi, sh, axis=(1, 2, 3))),
                          np.ascontiguousarray(np.roll(psi, sh, axis=(1, 2, 3))))
    assert np.abs(rolled - np.roll(full, sh, axis=(1, 2, 3))).max() <= 1e-13 * np.abs(full).max()


def test_oracle_rejects_bad_arguments():
    n = (4, 4, 4)
    phi = np.zeros((1,) + n, dtype=np.complex128)
    with pytest.raises(RuntimeError):
        oracle.apply(CELLS["ortho"], n, 7, OMEGA, 1.0, phi)
    with pytest.raises(RuntimeError):
        oracle.apply(CELLS["ortho"], n, HSE, 0.0, 1.0, phi)
    with pytest.raises(RuntimeError):
        oracle.apply(CELLS["ortho"], n, HSE, OMEGA, 1.0, phi, cols=[1])
    with pytest.raises(TypeError):
        oracle.apply(CELLS["ortho"], n, HSE, OMEGA, 1.0, phi.astype(np.complex64))


# --------------------------------------------------------------------------------------- golden table
def test_golden_vg_table_pins_the_oracle_kernel():
    """tests/golden/vg_table.txt: v(G) in 40-digit decimal arithmetic (written by tests/golden/make_vg_table.py from the
    BASELINE.json north_star formulas), including both G = 0 conventions (readings Q2, Q3).  The
    oracle's table must agree to a few ulp at every listed (cell, m), for both kernels."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "vg_table.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 2 * 3 * 10
    n = (32, 32, 32)
    cache = {}
    for kernel, _cell, l0, l1, l2, m0, m1, m2, val in rows:
        key = (kernel, l0, l1, l2)
        if key not in cache:
            cell = [float(l0), 0, 0, 0, float(l1), 0, 0, 0, float(l2)]
            cache[key] = oracle.vtable(cell, n, COUL if kernel == "coulomb" else HSE, 0.106)
        got = cache[key][int(m0) % n[0], int(m1) % n[1], int(m2) % n[2]]
        want = float(val)
        assert abs(got - want) <= 1e-14 * max(abs(want), 1e-300), (kernel, l0, m0, m1, m2, got, want)
