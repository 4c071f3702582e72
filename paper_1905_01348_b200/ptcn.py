"""One parallel-transport Crank-Nicolson (PT-CN) time step with a MODEL Hamiltonian, driving the C-ABI library
(Eq. (4)-(5), Algorithm 1; PAPER.md:194-200 Anderson mixing, re-orthogonalisation).

    H[Psi] psi = -1/2 Laplacian psi + (v_ext + g rho[Psi]) psi + V_X[Psi] psi

A real Hamiltonian needs the pseudopotentials the paper uses, which are not available; the model keeps
the structure of the step.  This module only SEQUENCES library calls: every operation on grids runs in the kernels of
libptfock.so (ptfock_apply, ptfock_hloc_apply, ptfock_residual, ptfock_density, ptfock_vloc_update, ptfock_density_change,
ptfock_axpby, ptfock_banddot, ptfock_banddot_many, ptfock_orthonormalize); the host solves the (<= 20 x 20) per-wavefunction least-squares problems of the Anderson
mixing, as the paper's "size of the least squares problem becomes very small".  No CPU fallback.
"""
from __future__ import annotations

import numpy as np

from . import binding


class PTCN:
    def __init__(self, cell, n, n_e: int, kernel: int = binding.KERNEL_HSE, omega: float = 0.106, alpha: float = 0.25,
                 v_ext=None, g: float = 0.0, device: int = 0):
        import torch
        self.n, self.n_e, self.alpha, self.g = tuple(int(x) for x in n), int(n_e), float(alpha), float(g)
        self.fock = binding.Plan(cell, n, n_e, n_e, kernel, omega, alpha if alpha != 0.0 else 1.0, device)
        self.kin = binding.Plan(cell, n, 1, n_e, binding.KERNEL_KINETIC, omega, 1.0, device)
        dev = torch.device("cuda", device)
        self.v_ext = (torch.zeros(self.n, dtype=torch.float64, device=dev) if v_ext is None
                      else v_ext.to(dev, torch.float64).contiguous())
        self.w = abs(float(np.linalg.det(np.asarray(cell, dtype=np.float64).reshape(3, 3)))) / self.fock.N

    def close(self):
        self.fock.destroy()
        self.kin.destroy()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def h_apply(self, psi):
        """H[Psi] Psi (Alg. 1 line 5: the potential and the exchange operator follow Psi_f)."""
        v = self.v_ext
        if self.g != 0.0:
            v = self.fock.vloc_update(self.v_ext, self.g, self.fock.density(psi))
        out = self.kin.hloc_apply(psi, v)
        if self.alpha != 0.0:
            vx = self.fock.apply(psi)                                   # Psi = Phi: pair-symmetric schedule
            self.fock.axpby(1.0, out, 1.0, vx, out=out)
        return out

    def step(self, psi_n, dt: float, tol: float = 1e-10, max_iter: int = 60, beta: float = 1.0, depth: int = 20):
        """Algorithm 1.  Returns (psi_{n+1}, info); psi_n is not modified."""
        f, n_e = self.fock, self.n_e
        h = self.h_apply(psi_n)
        r_n = f.residual(psi_n, h)                                      # line 1
        psi_half = f.axpby(1.0, psi_n, -0.5j * dt, r_n)                 # line 2
        psi_f = psi_half.clone()
        rho = f.density(psi_f)                                          # line 3
        # Anderson history: differences of consecutive iterates / residuals (newest first) and their Gram matrix per
        # wavefunction, grown by one row per iteration (the oldest difference drops out beyond `depth`)
        x_prev = r_prev = None
        dxs, drs = [], []
        gram = np.zeros((n_e, 0, 0), dtype=np.complex128)
        info = {"iterations": 0, "rho_change": None, "residual": None}
        for it in range(max_iter):                                      # lines 4-10
            h = self.h_apply(psi_f)                                     # line 5
            r_f = f.residual(psi_f, h, dt=dt, psi_half=psi_half)        # line 6
            info["residual"] = float(np.sqrt(f.banddot(r_f, r_f).real.sum() / n_e))
            if info["residual"] < tol:
                break
            if x_prev is not None:
                dxs.insert(0, f.axpby(1.0, psi_f, -1.0, x_prev))
                drs.insert(0, f.axpby(1.0, r_f, -1.0, r_prev))
                row = f.banddot_many(drs[0], drs).T                     # <dR_new, dR_b> for every stored b, one call
                m_old = gram.shape[1]
                g2 = np.empty((n_e, m_old + 1, m_old + 1), dtype=np.complex128)
                g2[:, 1:, 1:] = gram
                g2[:, 0, :] = row
                g2[:, :, 0] = row.conj()
                g2[:, 0, 0] = row[:, 0].real
                gram = g2
                if len(dxs) > depth:
                    dxs.pop()
                    drs.pop()
                    gram = gram[:, :depth, :depth]
            x_prev, r_prev = psi_f, r_f
            m = len(dxs)
            new = f.axpby(1.0, psi_f, -beta, r_f)                       # line 7: Anderson mixing, per wavefunction
            if m > 0:
                rhs = f.banddot_many(r_f, drs).conj().T                 # <dR_b, R_f> = conj <R_f, dR_b>, one call
                gamma = np.empty((n_e, m), dtype=np.complex128)
                for j in range(n_e):
                    gj = gram[j] + 1e-14 * np.trace(gram[j]).real / m * np.eye(m)
                    gamma[j] = np.linalg.solve(gj, rhs[j])
                for a in range(m):
                    f.axpby(1.0, new, -gamma[:, a], dxs[a], out=new)
                    f.axpby(1.0, new, beta * gamma[:, a], drs[a], out=new)
            psi_f = new
            rho_new = f.density(psi_f)                                  # line 8
            change = f.density_change(rho_new, rho) / n_e               # line 9
            rho = rho_new
            info.update(iterations=it + 1, rho_change=change)
        info["psi_f"] = psi_f                                           # the fixed point of Eq. (5) before line 11
        out = psi_f.clone()
        f.orthonormalize(out)                                           # line 11
        return out, info

