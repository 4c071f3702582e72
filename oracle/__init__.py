"""CPU oracle for the plane-wave Fock exchange path (TEST INFRASTRUCTURE, not the product).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It loads ``oracle/ptfock_ref.c`` (plain C, own FFT) through ctypes and
shares nothing with ``paper_1905_01348_b200`` (no common code, tables or helpers).

Citations: PAPER.md:57-61 (Sec. 2, Eq. 3), PAPER.md:116-144 (Sec. 3.2, Alg. 2); see the header of
``ptfock_ref.c`` for the exact definition and the list of pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ptfock_ref.c")
_SRC_DENSE = os.path.join(_HERE, "ptdense_ref.c")       # dense-algebra neighbours (Alg. 3, Sec. 3.4)
_LIB = os.path.join(_HERE, "libptfock_ref.so")

KERNEL_COULOMB = 0
KERNEL_HSE = 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp, no fast-math).  Returns the path of the .so."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_DENSE))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c99", "-o", _LIB, _SRC, _SRC_DENSE, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        dp = ctypes.c_void_p
        _lib.ptfock_ref_apply.argtypes = [dp, dp, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int32, dp,
                                          ctypes.c_int32, dp, dp, ctypes.c_int32, dp, dp]
        _lib.ptfock_ref_apply.restype = ctypes.c_int
        _lib.ptfock_ref_exchange_energy.argtypes = [dp, dp, dp, dp, ctypes.c_int32, dp, dp]
        _lib.ptfock_ref_exchange_energy.restype = ctypes.c_int
        _lib.ptfock_ref_vtable.argtypes = [dp, dp, ctypes.c_int, ctypes.c_double, dp]
        _lib.ptfock_ref_vtable.restype = ctypes.c_int
        _lib.ptfock_ref_pair_w.argtypes = [dp, dp, ctypes.c_int, ctypes.c_double, dp, dp, dp]
        _lib.ptfock_ref_pair_w.restype = ctypes.c_int
        _lib.ptfock_ref_fft3d.argtypes = [dp, ctypes.c_int, dp]
        _lib.ptfock_ref_fft3d.restype = ctypes.c_int
        _lib.ptfock_ref_fft1d.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
        _lib.ptfock_ref_fft1d.restype = ctypes.c_int
        _lib.ptfock_ref_dft1d_naive.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
        _lib.ptfock_ref_dft1d_naive.restype = None
        _lib.ptfock_ref_num_threads.restype = ctypes.c_int
        i64, i32, f64 = ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        _lib.ptdense_ref_overlap.argtypes = [i64, f64, dp, i32, dp, i32, dp]
        _lib.ptdense_ref_rotate.argtypes = [i64, dp, i32, dp, i32, dp]
        _lib.ptdense_ref_residual.argtypes = [i64, f64, i32, f64, dp, dp, dp, dp]
        _lib.ptdense_ref_density.argtypes = [i64, dp, i32, dp]
        _lib.ptdense_ref_cholesky.argtypes = [i32, dp, dp]
        _lib.ptdense_ref_orthonormalize.argtypes = [i64, f64, dp, i32, dp]
        for f in ("overlap", "rotate", "residual", "density", "cholesky", "orthonormalize"):
            getattr(_lib, "ptdense_ref_" + f).restype = ctypes.c_int
    return _lib


def _ptr(a: np.ndarray) -> ctypes.c_void_p:
    return ctypes.c_void_p(a.ctypes.data)


def _cell(cell) -> np.ndarray:
    c = np.ascontiguousarray(np.asarray(cell, dtype=np.float64).reshape(9))
    return c


def _grid(n) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(n, dtype=np.int32).reshape(3))


def _c128(a, what: str) -> np.ndarray:
    a = np.asarray(a)
    if a.dtype != np.complex128 or not a.flags.c_contiguous:
        raise TypeError(f"{what} must be a C-contiguous complex128 array")
    return a


def num_threads() -> int:
    return int(lib().ptfock_ref_num_threads())


def apply(cell, n, kernel: int, omega: float, alpha: float, phi: np.ndarray, psi: np.ndarray | None = None,
          cols=None) -> np.ndarray:
    """V_X[Phi] psi_j for j in ``cols`` (default: all targets).  phi: [n_occ, n0, n1, n2] complex128;
    psi: [n_targets, ...] or None meaning Psi = Phi.  Returns [len(cols), n0, n1, n2] complex128."""
    n = _grid(n)
    phi = _c128(phi, "phi")
    psi = phi if psi is None else _c128(psi, "psi")
    N = int(n[0]) * int(n[1]) * int(n[2])
    if phi.size % N or psi.size % N:
        raise ValueError("orbital arrays do not match the grid")
    n_occ, n_t = phi.size // N, psi.size // N
    if cols is None:
        cols_a, n_cols, cols_p = None, n_t, ctypes.c_void_p(0)
    else:
        cols_a = np.ascontiguousarray(np.asarray(cols, dtype=np.int32))
        n_cols, cols_p = int(cols_a.size), _ptr(cols_a)
    out = np.empty((n_cols, int(n[0]), int(n[1]), int(n[2])), dtype=np.complex128)
    c = _cell(cell)
    rc = lib().ptfock_ref_apply(_ptr(c), _ptr(n), int(kernel), float(omega), float(alpha), n_occ, _ptr(phi), n_t,
                                _ptr(psi), cols_p, n_cols, _ptr(out), ctypes.c_void_p(0))
    if rc != 0:
        raise RuntimeError(f"ptfock_ref_apply failed: {rc}")
    return out


def exchange_energy(cell, n, psi: np.ndarray, vx: np.ndarray, cols=None) -> complex:
    """E_x = 1/2 (Omega/N) sum_j <psi_j | vx_j>; returned as complex (imaginary part should vanish)."""
    n = _grid(n)
    psi, vx = _c128(psi, "psi"), _c128(vx, "vx")
    N = int(n[0]) * int(n[1]) * int(n[2])
    n_cols = vx.size // N
    if cols is None:
        cols_p = ctypes.c_void_p(0)
        if psi.size // N != n_cols:
            raise ValueError("psi and vx column counts differ")
    else:
        cols_a = np.ascontiguousarray(np.asarray(cols, dtype=np.int32))
        cols_p = _ptr(cols_a)
    e = np.zeros(2, dtype=np.float64)
    c = _cell(cell)
    rc = lib().ptfock_ref_exchange_energy(_ptr(c), _ptr(n), _ptr(psi), cols_p, n_cols, _ptr(vx), _ptr(e))
    if rc != 0:
        raise RuntimeError(f"ptfock_ref_exchange_energy failed: {rc}")
    return complex(e[0], e[1])


def vtable(cell, n, kernel: int, omega: float) -> np.ndarray:
    n = _grid(n)
    v = np.empty((int(n[0]), int(n[1]), int(n[2])), dtype=np.float64)
    c = _cell(cell)
    rc = lib().ptfock_ref_vtable(_ptr(c), _ptr(n), int(kernel), float(omega), _ptr(v))
    if rc != 0:
        raise RuntimeError(f"ptfock_ref_vtable failed: {rc}")
    return v


def pair_w(cell, n, kernel: int, omega: float, phi_i: np.ndarray, psi_j: np.ndarray) -> np.ndarray:
    n = _grid(n)
    phi_i, psi_j = _c128(phi_i, "phi_i"), _c128(psi_j, "psi_j")
    w = np.empty((int(n[0]), int(n[1]), int(n[2])), dtype=np.complex128)
    c = _cell(cell)
    rc = lib().ptfock_ref_pair_w(_ptr(c), _ptr(n), int(kernel), float(omega), _ptr(phi_i), _ptr(psi_j), _ptr(w))
    if rc != 0:
        raise RuntimeError(f"ptfock_ref_pair_w failed: {rc}")
    return w


def fft3d(grid: np.ndarray, sign: int) -> np.ndarray:
    g = np.array(_c128(grid, "grid"), copy=True)
    n = _grid(g.shape)
    rc = lib().ptfock_ref_fft3d(_ptr(n), int(sign), _ptr(g))
    if rc != 0:
        raise RuntimeError(f"ptfock_ref_fft3d failed: {rc}")
    return g


def fft1d(x: np.ndarray, sign: int) -> np.ndarray:
    x = _c128(x, "x")
    y = np.empty_like(x)
    rc = lib().ptfock_ref_fft1d(int(x.size), int(sign), _ptr(x), _ptr(y))
    if rc != 0:
        raise RuntimeError(f"ptfock_ref_fft1d failed: {rc}")
    return y


def dft1d_naive(x: np.ndarray, sign: int) -> np.ndarray:
    x = _c128(x, "x")
    y = np.empty_like(x)
    lib().ptfock_ref_dft1d_naive(int(x.size), int(sign), _ptr(x), _ptr(y))
    return y


# ---- dense-algebra neighbours (oracle/ptdense_ref.c; Alg. 3, Sec. 3.4) ---------------
def _orbs(a, what: str):
    a = _c128(a, what)
    if a.ndim < 2:
        raise ValueError(f"{what} must be [n_orbitals, points...]")
    return a, a.shape[0], a.size // max(1, a.shape[0])


def overlap(a: np.ndarray, b: np.ndarray, weight: float) -> np.ndarray:
    """S[m, n] = weight * sum_r conj(a_m(r)) b_n(r)."""
    a, n_a, N = _orbs(a, "a")
    b, n_b, Nb = _orbs(b, "b")
    if N != Nb:
        raise ValueError("a and b live on different grids")
    s = np.empty((n_a, n_b), dtype=np.complex128)
    rc = lib().ptdense_ref_overlap(N, float(weight), _ptr(a), n_a, _ptr(b), n_b, _ptr(s))
    if rc != 0:
        raise RuntimeError(f"ptdense_ref_overlap failed: {rc}")
    return s


def rotate(a: np.ndarray, s: np.ndarray) -> np.ndarray:
    """out_n(r) = sum_m a_m(r) S[m, n]."""
    a, n_a, N = _orbs(a, "a")
    s = _c128(s, "s")
    if s.ndim != 2 or s.shape[0] != n_a:
        raise ValueError("S must be [n_a, n_out]")
    out = np.empty((s.shape[1],) + a.shape[1:], dtype=np.complex128)
    rc = lib().ptdense_ref_rotate(N, _ptr(a), n_a, _ptr(s), s.shape[1], _ptr(out))
    if rc != 0:
        raise RuntimeError(f"ptdense_ref_rotate failed: {rc}")
    return out


def residual(psi: np.ndarray, hpsi: np.ndarray, weight: float, dt: float = 0.0, psi_half: np.ndarray | None = None) -> np.ndarray:
    """psi_half None: R_n = H Psi - Psi (Psi^* H Psi); else R_f = Psi + (i dt/2)(H Psi - Psi (Psi^* H Psi)) - Psi_half."""
    psi, n, N = _orbs(psi, "psi")
    hpsi = _c128(hpsi, "hpsi")
    if hpsi.shape != psi.shape:
        raise ValueError("hpsi must have psi's shape")
    half_p = ctypes.c_void_p(0)
    if psi_half is not None:
        psi_half = _c128(psi_half, "psi_half")
        if psi_half.shape != psi.shape:
            raise ValueError("psi_half must have psi's shape")
        half_p = _ptr(psi_half)
    r = np.empty_like(psi)
    rc = lib().ptdense_ref_residual(N, float(weight), n, float(dt), _ptr(psi), _ptr(hpsi), half_p, _ptr(r))
    if rc != 0:
        raise RuntimeError(f"ptdense_ref_residual failed: {rc}")
    return r


def density(psi: np.ndarray) -> np.ndarray:
    """rho(r) = sum_i |psi_i(r)|^2 (shape of one grid)."""
    psi, n, N = _orbs(psi, "psi")
    rho = np.empty(psi.shape[1:], dtype=np.float64)
    rc = lib().ptdense_ref_density(N, _ptr(psi), n, _ptr(rho))
    if rc != 0:
        raise RuntimeError(f"ptdense_ref_density failed: {rc}")
    return rho


def cholesky(s: np.ndarray) -> np.ndarray:
    """Lower-triangular L with S = L L^H (S Hermitian positive definite)."""
    s = _c128(s, "s")
    if s.ndim != 2 or s.shape[0] != s.shape[1]:
        raise ValueError("S must be square")
    l = np.empty_like(s)
    rc = lib().ptdense_ref_cholesky(s.shape[0], _ptr(s), _ptr(l))
    if rc != 0:
        raise RuntimeError(f"ptdense_ref_cholesky failed: {rc}")
    return l


def orthonormalize(psi: np.ndarray, weight: float) -> np.ndarray:
    """Psi L^{-H} with L L^H = Psi^* Psi (Cholesky + triangular solve)."""
    psi, n, N = _orbs(psi, "psi")
    out = np.empty_like(psi)
    rc = lib().ptdense_ref_orthonormalize(N, float(weight), _ptr(psi), n, _ptr(out))
    if rc != 0:
        raise RuntimeError(f"ptdense_ref_orthonormalize failed: {rc}")
    return out
