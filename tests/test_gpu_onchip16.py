"""GPU vs oracle parity for the single-pass on-chip kernel of 16^3 grids (csrc/onchip16.cuh):
the whole pair-solve -- product, 3-D DFT, x v', inverse, x phi_i, sum over i -- inside one CTA's shared memory, the i
loop split into chunks whose partial sums are added in order.  Covers Si8 at full size (BASELINE.json configs[0]),
one orbital, ragged chunking, many orbitals (several chunks and more CTAs than SMs), target batches, the host path,
one W_ij, a skew cell, and bit-exact repeatability.

Bar (BASELINE.json north_star): max |gpu - ref| / max |ref| <= 1e-10; every call goes through the C ABI.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10
EDGES = (10.26,) * 3
GRID = (16, 16, 16)


def _rel(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def _oracle(cfg, phi, psi=None, cols=None):
    return oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(),
                        None if psi is None else psi.cpu().numpy(), cols)


def test_Si8_full_and_energy(cuda_device):
    cfg = synth.CONFIGS["Si8"]
    phi = synth.orbitals(cfg, device=cuda_device)
    with binding.plan_for(cfg) as plan:
        out = plan.apply(phi)
        e = plan.exchange_energy(phi, vx_psi=out)
        e2 = plan.exchange_energy(phi)
        info = plan.info()
    assert info["pass8"] == 2 and info["last_pairs"] == 256 and info["last_launches"] == 2
    ref = _oracle(cfg, phi)
    assert _rel(out.cpu().numpy(), ref) <= TOL
    e_ref = oracle.exchange_energy(cfg.cell, cfg.n, phi.cpu().numpy(), ref).real
    assert abs(e - e_ref) <= TOL * abs(e_ref) and abs(e2 - e_ref) <= TOL * abs(e_ref) and e < 0.0


@pytest.mark.parametrize("n_occ,n_t", [(1, 1), (2, 3), (7, 5), (37, 2), (300, 1)])
@pytest.mark.parametrize("kernel", [synth.KERNEL_HSE, synth.KERNEL_COULOMB], ids=["hse", "coulomb"])
def test_general_ragged_chunks(cuda_device, n_occ, n_t, kernel):
    """Few targets x many orbitals: the i loop is cut into up to 2 x SMs / n_t chunks (ragged last chunk)."""
    cfg = synth.Config("oc", EDGES, GRID, n_occ, kernel, separate_psi=True)
    phi = synth.random_orbitals(cfg, 21, n_occ, cuda_device)
    psi = synth.random_orbitals(cfg, 22, n_t, cuda_device)
    with binding.plan_for(cfg, max_targets=n_t) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
        assert plan.info()["last_pairs"] == n_occ * n_t
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL


def test_many_targets_and_self_offsets(cuda_device):
    """More CTAs than SMs; Psi = Phi (whole set and streamed j-blocks); same bits either way."""
    cfg = synth.Config("ocs", EDGES, GRID, 200, synth.KERNEL_HSE)
    phi = synth.random_orbitals(cfg, 23, 200, cuda_device)
    with binding.plan_for(cfg) as plan:
        full = plan.apply(phi)
        blk = torch.cat([plan.apply(phi, None, self_offset=o, n_targets=min(64, 200 - o)) for o in range(0, 200, 64)])
        torch.cuda.synchronize()
    cols = [0, 63, 64, 199]
    ref = _oracle(cfg, phi, cols=cols)
    assert _rel(full[cols].cpu().numpy(), ref) <= TOL
    assert _rel(blk[cols].cpu().numpy(), ref) <= TOL


def test_small_workspace_batches_targets(cuda_device):
    """A workspace of 8 grids: targets go through in batches of <= 8 with one chunk each."""
    cfg = synth.Config("ocw", EDGES, GRID, 6, synth.KERNEL_COULOMB, separate_psi=True)
    phi = synth.random_orbitals(cfg, 25, 6, cuda_device)
    psi = synth.random_orbitals(cfg, 26, 19, cuda_device)
    with binding.plan_for(cfg, max_targets=19, workspace_bytes=8 * 4096 * 16) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL


def test_host_path_single_pair_and_skew_cell(cuda_device):
    cfg = synth.Config("och", EDGES, GRID, 6, synth.KERNEL_HSE, separate_psi=True, alpha=0.25)
    phi, psi = synth.make_case(cfg, cuda_device)
    with binding.plan_for(cfg) as plan:
        dev = plan.apply(phi, psi)
        host = plan.apply_host(phi.cpu().pin_memory(), psi.cpu().pin_memory())
        w = plan.debug_pair(phi[1], psi[2]).cpu().numpy()
        torch.cuda.synchronize()
    assert torch.equal(host, dev.cpu())
    assert _rel(dev.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL
    ref_w = -cfg.alpha * oracle.pair_w(cfg.cell, cfg.n, cfg.kernel, cfg.omega, phi[1].cpu().numpy(), psi[2].cpu().numpy())
    assert _rel(w, ref_w) <= TOL
    cell = [10.26, 0.0, 0.0, 1.0, 10.0, 0.0, -0.7, 0.4, 9.8]
    with binding.Plan(cell, GRID, 6, 6, synth.KERNEL_HSE, 0.106, 1.0) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
    ref = oracle.apply(cell, GRID, synth.KERNEL_HSE, 0.106, 1.0, phi.cpu().numpy(), psi.cpu().numpy(), None)
    assert _rel(out.cpu().numpy(), ref) <= TOL


def test_repeatable_and_equal_to_three_pass_path(cuda_device):
    cfg = synth.Config("ocr", EDGES, GRID, 40, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 31, 40, cuda_device)
    psi = synth.random_orbitals(cfg, 32, 9, cuda_device)
    with binding.plan_for(cfg, max_targets=9) as plan:
        first = plan.apply(phi, psi).clone()
        for _ in range(3):
            again = plan.apply(phi, psi)
            torch.cuda.synchronize()
            assert torch.equal(first, again)
    with binding.plan_for(cfg, max_targets=9, flags=binding.FLAG_THREE_STAGE_SLABS) as plan:
        other = plan.apply(phi, psi)
        torch.cuda.synchronize()
    ref = _oracle(cfg, phi, psi)
    assert _rel(first.cpu().numpy(), ref) <= TOL and _rel(other.cpu().numpy(), ref) <= TOL
