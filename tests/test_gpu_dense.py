"""GPU vs oracle parity for the dense-algebra neighbours (csrc/dense.cuh behind ptfock_overlap / ptfock_rotate /
ptfock_residual / ptfock_density / ptfock_orthonormalize; Alg. 3, Sec. 3.4).

Sizes: small ragged cases element by element (orbital counts that are not multiples of the 64-wide tiles, grids that
are not multiples of the 64-point tiles' split), and the BASELINE orbital counts (1024 on 64^3, 3072 on a short
128 x 48 slab stack) on sampled entries the oracle computes one by one.  Bar: floating point, the same fp64 sums in a
different order: 1e-12 relative to the largest entry (sum lengths up to 2.6e5; observed ~1e-15).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _rel(got, ref):
    return float(np.abs(got - ref).max() / max(np.abs(ref).max(), 1e-300))


def _noise(shape, seed, dev):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return torch.complex(torch.randn(shape, generator=g, dtype=torch.float64),
                         torch.randn(shape, generator=g, dtype=torch.float64)).to(dev)


CASES = [((16, 16, 16), 1, 1), ((16, 16, 16), 5, 3), ((16, 32, 16), 70, 65), ((32, 16, 32), 130, 7)]


@pytest.mark.parametrize("n,na,nb", CASES, ids=[f"{c[0][0]}x{c[0][1]}x{c[0][2]}-{c[1]}-{c[2]}" for c in CASES])
def test_overlap_rotate_density_small(cuda_device, n, na, nb):
    cfg = synth.Config("d", (9.0, 10.0, 11.0), n, na, synth.KERNEL_HSE)
    a = _noise((na,) + n, 1, cuda_device)
    b = _noise((nb,) + n, 2, cuda_device)
    w = cfg.volume / cfg.N
    with binding.plan_for(cfg) as plan:
        s = plan.overlap(a, b)
        coef = _noise((na, nb), 3, cuda_device)
        rot = plan.rotate(a, coef)
        rho = plan.density(a)
        torch.cuda.synchronize()
    an, bn = a.cpu().numpy(), b.cpu().numpy()
    assert _rel(s.cpu().numpy(), oracle.overlap(an, bn, w)) <= TOL
    assert _rel(rot.cpu().numpy(), oracle.rotate(an, coef.cpu().numpy())) <= TOL
    assert _rel(rho.cpu().numpy(), oracle.density(an)) <= TOL


@pytest.mark.parametrize("n_orb", [1, 64, 70, 200])
def test_hermitian_overlap_computes_the_lower_tiles_and_mirrors_the_rest(cuda_device, n_orb):
    """S = Psi^* Psi: with the same orbitals on both sides only the 64 x 64 tiles on and below the diagonal
    are contracted; the others are their conjugate mirror images.  Against the oracle, and against the general path."""
    n = (16, 16, 32)
    cfg = synth.Config("h", (9.0, 10.0, 11.0), n, n_orb, synth.KERNEL_HSE)
    a = _noise((n_orb,) + n, 31, cuda_device)
    w = cfg.volume / cfg.N
    with binding.plan_for(cfg) as plan:
        herm = plan.overlap(a, a).cpu().numpy()                         # same pointer: Hermitian path
        full = plan.overlap(a, a.clone()).cpu().numpy()                 # another pointer: every tile contracted
    assert _rel(herm, oracle.overlap(a.cpu().numpy(), a.cpu().numpy(), w)) <= TOL
    assert np.array_equal(herm, herm.conj().T) or _rel(herm, herm.conj().T) <= 1e-15
    t = np.arange(n_orb) // 64
    low = t[:, None] >= t[None, :]
    assert np.array_equal(herm[low], full[low])                         # computed tiles: the same sums
    assert _rel(herm, full) <= 1e-14


@pytest.mark.parametrize("n_orb", [1, 5, 64, 70, 130])
def test_residuals_and_orthonormalize_small(cuda_device, n_orb):
    n = (16, 16, 16)
    cfg = synth.Config("r", (9.0, 10.0, 11.0), n, n_orb, synth.KERNEL_HSE)
    w = cfg.volume / cfg.N
    psi = _noise((n_orb,) + n, 4, cuda_device)
    hpsi = _noise((n_orb,) + n, 5, cuda_device)
    half = _noise((n_orb,) + n, 6, cuda_device)
    with binding.plan_for(cfg) as plan:
        rn = plan.residual(psi, hpsi)
        rf = plan.residual(psi, hpsi, dt=0.37, psi_half=half)
        orth = plan.orthonormalize(psi.clone())
        s = plan.overlap(orth, orth)
        torch.cuda.synchronize()
    pn, hn = psi.cpu().numpy(), hpsi.cpu().numpy()
    assert _rel(rn.cpu().numpy(), oracle.residual(pn, hn, w)) <= TOL
    assert _rel(rf.cpu().numpy(), oracle.residual(pn, hn, w, dt=0.37, psi_half=half.cpu().numpy())) <= TOL
    # the triangular solve amplifies rounding by the condition of the overlap matrix of the noise set (a few units)
    assert _rel(orth.cpu().numpy(), oracle.orthonormalize(pn, w)) <= 1e-11
    assert np.abs(s.cpu().numpy() - np.eye(n_orb)).max() <= 1e-12


def test_orthonormalize_rejects_dependent_orbitals(cuda_device):
    n = (16, 16, 16)
    cfg = synth.Config("np", (9.0, 10.0, 11.0), n, 3, synth.KERNEL_HSE)
    psi = _noise((3,) + n, 7, cuda_device)
    psi[2] = psi[0] + psi[1]
    with binding.plan_for(cfg) as plan:
        with pytest.raises(binding.PtfockError) as ei:
            plan.orthonormalize(psi)
    assert ei.value.code == -8


def _sampled_overlap(a, b, w, idx):
    return np.array([w * np.vdot(a[m].ravel(), b[n].ravel()) for m, n in idx])


def test_Si512_sizes_sampled(cuda_device):
    """1024 orbitals on 64^3: overlap / residual / density / orthonormalisation at BASELINE size, checked on sampled
    entries the oracle evaluates one by one (full oracle runs would take hours)."""
    cfg = synth.CONFIGS["Si512"]
    psi = synth.orbitals(cfg, device=cuda_device)                       # orthonormal
    hpsi = _noise(tuple(psi.shape), 8, cuda_device)
    w = cfg.volume / cfg.N
    with binding.plan_for(cfg) as plan:
        s = plan.overlap(psi, hpsi)
        rn = plan.residual(psi, hpsi)
        rho = plan.density(psi)
        torch.cuda.synchronize()
        idx = [(0, 0), (5, 1000), (1023, 1023), (517, 64), (63, 960)]
        hn_cols = {n: hpsi[n].cpu().numpy() for _, n in idx}
        pn_rows = {m: psi[m].cpu().numpy() for m, _ in idx}
        ref = np.array([oracle.overlap(pn_rows[m][None], hn_cols[n][None], w)[0, 0] for m, n in idx])
        got = np.array([s[m, n].item() for m, n in idx])
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
        # R_n is orthogonal to the (orthonormal) Psi: Psi^* R_n = 0 at any size
        z = plan.overlap(psi, rn)
        assert float(z.abs().max()) <= 1e-11 * float(s.abs().max())
        # R_n and R_f element by element on sampled orbitals (both sides of a 64-wide tile edge, first and last), from the
        # oracle's overlap and rotation over ALL 1024 orbitals (Alg. 3 lines 2, 4, 5; a full
        # oracle.residual would take hours): R_n[c] = H psi_c - sum_m psi_m S[m][c], S[:, c] = (psi_m, H psi_c)
        cols, dt = [0, 63, 64, 1023], 0.37
        half = _noise(tuple(psi.shape), 10, cuda_device)
        rf = plan.residual(psi, hpsi, dt=dt, psi_half=half)
        torch.cuda.synchronize()
        psi_np = psi.cpu().numpy()
        h_c = np.ascontiguousarray(hpsi[cols].cpu().numpy())
        proj = oracle.rotate(psi_np, oracle.overlap(psi_np, h_c, w))
        ref_rn = h_c - proj
        ref_rf = psi_np[cols] + 0.5j * dt * ref_rn - half[cols].cpu().numpy()
        assert np.abs(rn[cols].cpu().numpy() - ref_rn).max() <= TOL * np.abs(ref_rn).max()
        assert np.abs(rf[cols].cpu().numpy() - ref_rf).max() <= TOL * np.abs(ref_rf).max()
        del psi_np, rf, half
        # density: sampled points against the oracle's definition, and the electron count
        pts = [0, 12345, 262143]
        flat = psi.reshape(1024, -1)
        ref_rho = np.array([oracle.density(np.ascontiguousarray(flat[:, p:p + 1].cpu().numpy()))[0] for p in pts])
        assert np.abs(rho.reshape(-1)[pts].cpu().numpy() - ref_rho).max() <= TOL * ref_rho.max()
        assert abs(float(rho.sum()) * w - 1024.0) <= 1e-9
        # orthonormalise a mildly non-orthogonal set; result: S = I, first column only normalised
        mix = psi + 0.05 * torch.roll(psi, 1, 0)
        first = mix[0].clone()
        plan.orthonormalize(mix)
        s2 = plan.overlap(mix, mix)
        torch.cuda.synchronize()
        assert float((s2 - torch.eye(1024, dtype=s2.dtype, device=s2.device)).abs().max()) <= 1e-11
        nrm = float(torch.sqrt(w * (first.abs() ** 2).sum()))
        assert float((mix[0] - first / nrm).abs().max()) <= 1e-13 * float(first.abs().max()) / nrm * 10


def test_Si1536_orbital_count_sampled(cuda_device):
    """3072 orbitals (the Si1536 count) on a short 16 x 128 x 48 stack: 48 panels of the blocked Cholesky, 48 block
    columns of the triangular solve."""
    n = (16, 128, 48)
    cfg = synth.Config("d3072", (10.26, 82.08, 30.78), n, 3072, synth.KERNEL_HSE)
    psi = _noise((3072,) + n, 9, cuda_device)
    w = cfg.volume / cfg.N
    with binding.plan_for(cfg) as plan:
        keep = psi[[0, 1, 70, 3071]].clone()
        head = psi[:70].cpu().numpy()                                   # columns 0..69 of Psi L^-H depend on these only
        s = plan.overlap(psi, psi)
        plan.orthonormalize(psi)
        s2 = plan.overlap(psi, psi)
        torch.cuda.synchronize()
    assert float((s2 - torch.eye(3072, dtype=s2.dtype, device=s2.device)).abs().max()) <= 1e-10
    # first two columns by hand (Gram-Schmidt): q0 = p0 / |p0|, q1 = (p1 - (q0, p1) q0) / |...|
    p0, p1 = keep[0].cpu().numpy().ravel(), keep[1].cpu().numpy().ravel()
    q0 = p0 / np.sqrt(w * np.vdot(p0, p0).real)
    v = p1 - w * np.vdot(q0, p1) * q0
    q1 = v / np.sqrt(w * np.vdot(v, v).real)
    assert np.abs(psi[0].cpu().numpy().ravel() - q0).max() <= 1e-12 * np.abs(q0).max()
    assert np.abs(psi[1].cpu().numpy().ravel() - q1).max() <= 1e-12 * np.abs(q1).max()
    ref = w * np.vdot(keep[2].cpu().numpy().ravel(), keep[3].cpu().numpy().ravel())
    assert abs(s[70, 3071].item() - ref) <= TOL * float(s.abs().max())
    # the first 70 columns (across the first 64-wide Cholesky panel) against the oracle: L is lower triangular, so column k of
    # Psi L^-H is fixed by orbitals 0..k and oracle.orthonormalize of the leading 70 orbitals gives exactly these columns
    ref_head = oracle.orthonormalize(np.ascontiguousarray(head), w)
    assert np.abs(psi[:70].cpu().numpy() - ref_head).max() <= 1e-11 * np.abs(ref_head).max()
