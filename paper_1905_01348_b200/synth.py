"""Seeded synthetic inputs: Si-like supercells and random plane-wave orbitals.

This module holds NONE of the method's arithmetic (no pair product, no kernel v(G), no exchange
sum); it only makes inputs, and serves both the CUDA path and the CPU oracle so that the two are
handed identical bytes.  It stands in for the paper's workload -- converged HSE06 Kohn-Sham
orbitals of bulk-silicon supercells, E_cut = 10 Ha (Sec. 4) -- which cannot be
produced here (no pseudopotentials, no DFT code).  The recipe is BASELINE.json ``configs`` /
SURVEY.md Sec. 8(d):

1. sphere: all integer m with |m_d| < n_d/2 and |G(m)|^2/2 <= 10 Ha, G = 2 pi m_d / L_d;
2. raw coefficients c_i(m) = (g_re + i g_im) exp(-|G|^2/8), g standard normals from a
   counter-based generator (splitmix64 keyed by seed, counter = 2 (i N + k_lin) + {0, 1},
   53-bit uniforms, Box-Muller), so the numbers do not depend on generation order or device;
3. Loewdin orthonormalisation C <- (C C^H)^(-1/2) C in fp64;
4. phi_i(r) = (N / sqrt(Omega)) ifftn(c_i on the grid), so sum_r |phi_i|^2 Omega/N = 1.

``torch`` is used for memory, eigh/matmul and the library inverse FFT of step 4 (input generation
only; the hot path has its own FFT).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import torch

KERNEL_COULOMB = 0
KERNEL_HSE = 1

A_SI = 10.26          # bohr, simple-cubic 8-atom silicon cell edge (BASELINE.json configs[0])
ECUT_HA = 10.0        # PAPER.md:206 "kinetic energy cutoff is set to 10 Hartree"
OMEGA_HSE = 0.106     # bohr^-1 (BASELINE.json)
SEED_PHI = 190501348
SEED_PSI = 190501349


@dataclass(frozen=True)
class Config:
    name: str
    edges: tuple            # orthorhombic cell edges in bohr
    n: tuple                # real-space grid
    n_occ: int              # number of Phi orbitals
    kernel: int
    omega: float = OMEGA_HSE
    alpha: float = 1.0
    separate_psi: bool = False   # Psi is an independent seeded set (no pair symmetry)
    j_block: int = 0             # > 0: Psi = Phi streamed in j-blocks of this many columns
    seed_phi: int = SEED_PHI
    seed_psi: int = SEED_PSI
    ecut: float = ECUT_HA

    @property
    def N(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    @property
    def volume(self) -> float:
        return self.edges[0] * self.edges[1] * self.edges[2]

    @property
    def cell(self) -> list:
        return [self.edges[0], 0.0, 0.0, 0.0, self.edges[1], 0.0, 0.0, 0.0, self.edges[2]]


CONFIGS = {
    "Si8": Config("Si8", (A_SI,) * 3, (16, 16, 16), 16, KERNEL_HSE),
    "Si64": Config("Si64", (2 * A_SI,) * 3, (32, 32, 32), 128, KERNEL_COULOMB),
    "Si216": Config("Si216", (3 * A_SI,) * 3, (48, 48, 48), 432, KERNEL_HSE),
    "Si512": Config("Si512", (4 * A_SI,) * 3, (64, 64, 64), 1024, KERNEL_HSE, separate_psi=True),
    "Si1536": Config("Si1536", (8 * A_SI, 8 * A_SI, 3 * A_SI), (128, 128, 48), 3072, KERNEL_HSE, j_block=96),
    # the paper's own 1536-atom workload (4 x 6 x 8 cell, wavefunction grid
    # 60 x 90 x 120 = 648 000 points, 3072 orbitals), axes ordered so that the 120-point edge is x0 (the pencil axis)
    "Si1536p": Config("Si1536p", (8 * A_SI, 6 * A_SI, 4 * A_SI), (120, 90, 60), 3072, KERNEL_HSE, j_block=96),
}

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Two's-complement view of a 64-bit unsigned constant (torch has no uint64 arithmetic)."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of int64 bit patterns."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _splitmix64(z: torch.Tensor) -> torch.Tensor:
    z = z + _s64(0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def _splitmix64_int(z: int) -> int:
    z = (z + 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def _normals(seed: int, counters: torch.Tensor) -> tuple:
    """Two independent standard normals per counter (Box-Muller on two 53-bit uniforms)."""
    key = _s64(_splitmix64_int(seed & _M64))
    a = _splitmix64((counters * 2) ^ key)
    b = _splitmix64((counters * 2 + 1) ^ key)
    u1 = (_lsr(a, 11).to(torch.float64) + 1.0) * (2.0 ** -53)     # (0, 1]
    u2 = _lsr(b, 11).to(torch.float64) * (2.0 ** -53)             # [0, 1)
    r = torch.sqrt(-2.0 * torch.log(u1))
    t = (2.0 * math.pi) * u2
    return r * torch.cos(t), r * torch.sin(t)


def sphere(cfg: Config, device="cpu"):
    """Plane waves inside the cutoff sphere.  Returns (k_lin [P] int64 C-order grid index of m mod n,
    g2 [P] float64 = |G|^2)."""
    ms = []
    for d in range(3):
        nd = cfg.n[d]
        m = torch.arange(-(nd // 2) + (1 if nd % 2 == 0 else 0), (nd - 1) // 2 + 1, dtype=torch.int64, device=device)
        ms.append(m)                                               # |m| < n/2 strictly
    m0, m1, m2 = torch.meshgrid(*ms, indexing="ij")
    g2 = sum(((2.0 * math.pi / cfg.edges[d]) * mm.to(torch.float64)) ** 2 for d, mm in enumerate((m0, m1, m2)))
    keep = (0.5 * g2) <= cfg.ecut
    k0 = torch.remainder(m0[keep], cfg.n[0])
    k1 = torch.remainder(m1[keep], cfg.n[1])
    k2 = torch.remainder(m2[keep], cfg.n[2])
    k_lin = (k0 * cfg.n[1] + k1) * cfg.n[2] + k2
    order = torch.argsort(k_lin)
    return k_lin[order], g2[keep][order]


def coefficients(cfg: Config, seed: int, n_orb: int, device="cpu", chunk: int = 64) -> torch.Tensor:
    """Loewdin-orthonormal sphere coefficients C [n_orb, P] complex128 (steps 1-3)."""
    k_lin, g2 = sphere(cfg, device)
    P = k_lin.numel()
    if n_orb > P:
        raise ValueError(f"{n_orb} orbitals do not fit {P} plane waves")
    damp = torch.exp(-g2 / 8.0)
    C = torch.empty((n_orb, P), dtype=torch.complex128, device=device)
    for i0 in range(0, n_orb, chunk):
        i1 = min(n_orb, i0 + chunk)
        idx = torch.arange(i0, i1, dtype=torch.int64, device=device)[:, None] * cfg.N + k_lin[None, :]
        gr, gi = _normals(seed, idx)
        C[i0:i1] = torch.complex(gr * damp, gi * damp)
    S = C @ C.conj().T
    w, U = torch.linalg.eigh(S)
    if float(w.min()) <= 0.0:
        raise RuntimeError("overlap matrix is not positive definite")
    S_mhalf = (U * (w ** -0.5).to(U.dtype)[None, :]) @ U.conj().T
    return S_mhalf @ C


def orbitals(cfg: Config, seed: int | None = None, n_orb: int | None = None, device="cpu", chunk: int = 32,
             out: torch.Tensor | None = None) -> torch.Tensor:
    """Grid orbitals [n_orb, n0, n1, n2] complex128 with sum_r |phi|^2 Omega/N = 1 (steps 1-4)."""
    seed = cfg.seed_phi if seed is None else seed
    n_orb = cfg.n_occ if n_orb is None else n_orb
    C = coefficients(cfg, seed, n_orb, device)
    k_lin, _ = sphere(cfg, device)
    if out is None:
        out = torch.empty((n_orb,) + tuple(cfg.n), dtype=torch.complex128, device=device)
    scale = cfg.N / math.sqrt(cfg.volume)
    for i0 in range(0, n_orb, chunk):
        i1 = min(n_orb, i0 + chunk)
        g = torch.zeros((i1 - i0, cfg.N), dtype=torch.complex128, device=device)
        g[:, k_lin] = C[i0:i1]
        out[i0:i1] = torch.fft.ifftn(g.view((i1 - i0,) + tuple(cfg.n)), dim=(1, 2, 3)) * scale
    return out


def random_orbitals(cfg: Config, seed: int, n_orb: int, device="cpu") -> torch.Tensor:
    """Plain complex normal noise on the grid (NOT orthonormal, not band-limited): for invariant
    and edge-case tests that should not lean on smooth inputs."""
    idx = torch.arange(n_orb * cfg.N, dtype=torch.int64, device=device)
    gr, gi = _normals(seed, idx)
    return torch.complex(gr, gi).view((n_orb,) + tuple(cfg.n)).contiguous()


def make_case(cfg: Config, device="cpu"):
    """(phi, psi) for a config: psi is None when Psi = Phi."""
    phi = orbitals(cfg, cfg.seed_phi, cfg.n_occ, device)
    psi = orbitals(cfg, cfg.seed_psi, cfg.n_occ, device) if cfg.separate_psi else None
    return phi, psi
