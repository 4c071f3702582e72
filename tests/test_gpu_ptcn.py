"""One PT-CN step on the GPU (paper_1905_01348_b200/ptcn.py driving the C ABI) against the CPU oracle
(oracle/ptcn_ref.py; Algorithm 1), the step helpers against their definitions, and the j-sharded apply.

Both sides iterate to the SAME fixed point of Eq. (5) (unique for these step sizes) by their own route; the bar is on
the result: |Psi_{n+1}^gpu - Psi_{n+1}^ref| <= 1e-8 max|Psi| with both residuals <= 1e-11 (the least-squares steps of the
Anderson mixing amplify rounding on the way, not at the fixed point).
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import ptcn_ref
from paper_1905_01348_b200 import binding, harness, ptcn, synth

pytestmark = pytest.mark.gpu


def _model(n, edges, n_e, alpha, g, dev):
    cell = [edges[0], 0, 0, 0, edges[1], 0, 0, 0, edges[2]]
    x = np.meshgrid(*[np.arange(k) / k for k in n], indexing="ij")
    v = 0.2 * np.cos(2 * np.pi * x[0]) + 0.1 * np.sin(2 * np.pi * (x[1] + x[2]))
    cfg = synth.Config("ptcn", edges, n, n_e, synth.KERNEL_HSE, ecut=3.0)
    psi0 = synth.orbitals(cfg, device=dev)                              # smooth orthonormal orbitals
    ref_model = ptcn_ref.Model(cell, n, kernel=1, omega=0.106, alpha=alpha, v_ext=v, g=g)
    return cell, v, psi0, ref_model


def test_step_helpers(cuda_device):
    n, edges = (16, 16, 16), (9.0, 10.0, 11.0)
    cell, v, psi, ref_model = _model(n, edges, 5, 0.25, 0.5, cuda_device)
    with ptcn.PTCN(cell, n, 5, alpha=0.25, v_ext=torch.from_numpy(v), g=0.5) as st:
        t = st.kin.hloc_apply(psi, st.v_ext).cpu().numpy()
        ref_t = ptcn_ref.kinetic_apply(cell, n, psi.cpu().numpy()) + v[None] * psi.cpu().numpy()
        assert np.abs(t - ref_t).max() <= 1e-12 * np.abs(ref_t).max()
        h = st.h_apply(psi).cpu().numpy()
        ref_h = ref_model.h_apply(psi.cpu().numpy())
        assert np.abs(h - ref_h).max() <= 1e-12 * np.abs(ref_h).max()
        a = np.array([1.0, 2.0j, -0.5, 0.25 + 1j, 3.0])
        b = np.array([0.5j, 1.0, 2.0, -1.0, 0.0])
        y = torch.roll(psi, 1, 0).contiguous()
        z = st.fock.axpby(a, psi, b, y).cpu().numpy()
        ref_z = a[:, None, None, None] * psi.cpu().numpy() + b[:, None, None, None] * y.cpu().numpy()
        assert np.abs(z - ref_z).max() <= 1e-15 * np.abs(ref_z).max() * 4
        d = st.fock.banddot(psi, y)
        ref_d = np.array([st.w * np.vdot(psi[j].cpu().numpy().ravel(), y[j].cpu().numpy().ravel()) for j in range(5)])
        assert np.abs(d - ref_d).max() <= 1e-13


@pytest.mark.parametrize("alpha,g", [(0.0, 0.0), (0.25, 0.5)], ids=["linear", "exchange+density"])
def test_one_step_matches_oracle(cuda_device, alpha, g):
    n, edges, n_e, dt = (16, 16, 16), (9.0, 10.0, 11.0), 4, 0.4
    cell, v, psi0, ref_model = _model(n, edges, n_e, alpha, g, cuda_device)
    with ptcn.PTCN(cell, n, n_e, alpha=alpha, v_ext=torch.from_numpy(v), g=g) as st:
        out, info = st.step(psi0, dt, tol=1e-11, max_iter=80)
        torch.cuda.synchronize()
        s = st.fock.overlap(out, out).cpu().numpy()
    ref, rinfo = ptcn_ref.ptcn_step(ref_model, psi0.cpu().numpy(), dt, tol=1e-11, max_iter=80)
    assert info["residual"] < 1e-11 and rinfo["residual"] < 1e-11 and info["iterations"] < 60
    assert np.abs(s - np.eye(n_e)).max() <= 1e-12
    got = out.cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-8 * np.abs(ref).max()
    rho, rho_ref = (np.abs(got) ** 2).sum(0), (np.abs(ref) ** 2).sum(0)
    assert np.abs(rho - rho_ref).max() <= 1e-9 * rho_ref.max()
    assert np.abs(got - psi0.cpu().numpy()).max() > 1e-3 * np.abs(ref).max()        # the step did move the orbitals


def test_sharded_apply_world1_equals_apply(cuda_device):
    cfg = synth.Config("sh", (9.0, 10.0, 11.0), (16, 16, 16), 7, synth.KERNEL_HSE)
    phi = synth.random_orbitals(cfg, 5, 7, cuda_device)
    with binding.plan_for(cfg) as plan:
        full = plan.apply(phi)
        part, (lo, hi) = harness.sharded_apply(plan, phi, 7)
        torch.cuda.synchronize()
    assert (lo, hi) == (0, 7) and torch.equal(part, full)
    # two "ranks" emulated one after the other on this GPU: the shards' outputs tile the full result
    with binding.plan_for(cfg) as plan:
        outs = []
        for r in range(2):
            lo, hi = harness.shard_range(7, 2, r)
            outs.append(plan.apply(phi, None, self_offset=lo, n_targets=hi - lo))
        torch.cuda.synchronize()
    assert torch.equal(torch.cat(outs), full)


@pytest.mark.parametrize("n", [(32, 32, 32), (48, 48, 48), (64, 64, 64), (16, 32, 16)])
def test_kinetic_plus_local_on_every_kernel_family(cuda_device, n):
    """ptfock_hloc_apply runs the exchange passes with the constant orbital and the table |G|^2 / 2 (one 'orbital', a wave
    of targets): on the two-stage kernels (32^3, 48^3, 64^3) and the generic three-stage ones, against the oracle's
    plane-wave definition of the Laplacian (H Psi of Algorithm 1)."""
    edges = (9.0 * n[0] / 16, 10.0 * n[1] / 16, 11.0 * n[2] / 16)
    cell = [edges[0], 0, 0, 0, edges[1], 0, 0, 0, edges[2]]
    cfg = synth.Config("kin", edges, n, 3, synth.KERNEL_HSE)
    psi = synth.random_orbitals(cfg, 41, 3, cuda_device)
    v = torch.rand(n, dtype=torch.float64, device=cuda_device)
    with binding.Plan(cell, n, 1, 3, binding.KERNEL_KINETIC, 0.106, 1.0) as kin:
        t = kin.hloc_apply(psi, v).cpu().numpy()
    ref = ptcn_ref.kinetic_apply(cell, n, psi.cpu().numpy()) + v.cpu().numpy()[None] * psi.cpu().numpy()
    assert np.abs(t - ref).max() <= 1e-12 * np.abs(ref).max()
