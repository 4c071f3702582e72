"""GPU vs oracle parity for the two-stage slab passes + 32 x 32 pencil pass (csrc/pass8.cuh), which serve 64^3 grids
(Si512): p8_fwd / p8_inv_acc with their TMA rings and in-place XOR-swizzled exchange, p8_mid with the swizzled
tensor-map tiles and the shared v' block.  64^3 pair-solves are cheap enough for the oracle when the orbital counts
are small; the cases walk through loops shorter than the rings (1, 2, 3 orbitals), ragged waves, the split i loop of
pass A, ragged pair triples in pass B, the conj(W) accumulate of the pair-symmetric schedule, j-blocks, one W_ij, and
the three-stage passes (PTFOCK_FLAG_THREE_STAGE_SLABS) as a second implementation of the same grid.

Bar (BASELINE.json north_star): max |gpu - ref| / max |ref| <= 1e-10; every call goes through the C ABI.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10
EDGES = (41.04, 41.04, 41.04)
GRID = (64, 64, 64)


def _rel(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def _oracle(cfg, phi, psi=None, cols=None):
    return oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(),
                        None if psi is None else psi.cpu().numpy(), cols)


@pytest.mark.parametrize("n_occ,n_t,bi,bj", [(1, 1, 1, 1), (2, 3, 2, 2), (3, 2, 3, 1), (7, 4, 4, 3), (9, 5, 0, 0)])
@pytest.mark.parametrize("flags", [0, binding.FLAG_THREE_STAGE_SLABS], ids=["pass8", "three_stage"])
def test_general_schedule_ragged(cuda_device, n_occ, n_t, bi, bj, flags):
    cfg = synth.Config("p8", EDGES, GRID, n_occ, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 21, n_occ, cuda_device)
    psi = synth.random_orbitals(cfg, 22, n_t, cuda_device)
    with binding.plan_for(cfg, max_targets=n_t, block_i=bi, block_j=bj, flags=flags) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
        info = plan.info()
    assert info["last_pairs"] == n_occ * n_t and info["pass8"] == (0 if flags else 1)
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL


def test_symmetric_schedule_uses_conj_accumulate(cuda_device):
    """Psi = Phi with blocks smaller than n_occ: off-diagonal block pairs feed out_i through conj(W_ij)."""
    cfg = synth.Config("p8s", EDGES, GRID, 6, synth.KERNEL_COULOMB)
    phi = synth.random_orbitals(cfg, 23, 6, cuda_device)
    with binding.plan_for(cfg, block_i=2, block_j=2) as plan:
        out = plan.apply(phi)
        torch.cuda.synchronize()
        info = plan.info()
    assert info["last_symmetric"] == 1 and info["last_pairs"] < 36 and info["pass8"] == 1
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi)) <= TOL


def test_j_blocks_and_energy(cuda_device):
    cfg = synth.Config("p8j", EDGES, GRID, 5, synth.KERNEL_HSE)
    phi = synth.orbitals(cfg, device=cuda_device)
    ref = _oracle(cfg, phi)
    with binding.plan_for(cfg, max_targets=2) as plan:
        blocks, e = [], 0.0
        for o in (0, 2, 4):
            nt = min(2, 5 - o)
            blk = plan.apply(phi, None, self_offset=o, n_targets=nt)
            e += plan.exchange_energy(phi, None, vx_psi=blk, self_offset=o, n_targets=nt)
            blocks.append(blk)
        torch.cuda.synchronize()
    assert _rel(torch.cat(blocks).cpu().numpy(), ref) <= TOL
    e_ref = oracle.exchange_energy(cfg.cell, cfg.n, phi.cpu().numpy(), ref).real
    assert abs(e - e_ref) <= TOL * abs(e_ref) and e < 0.0


def test_single_pair_W(cuda_device):
    cfg = synth.Config("p8w", EDGES, GRID, 2, synth.KERNEL_HSE, alpha=0.5)
    ab = synth.random_orbitals(cfg, 24, 2, cuda_device)
    with binding.plan_for(cfg) as plan:
        w = plan.debug_pair(ab[0], ab[1]).cpu().numpy()
    ref = -cfg.alpha * oracle.pair_w(cfg.cell, cfg.n, cfg.kernel, cfg.omega, ab[0].cpu().numpy(), ab[1].cpu().numpy())
    assert _rel(w, ref) <= TOL


def test_skew_cell_general_v_table(cuda_device):
    """A skew cell: v is not even on the grid's Nyquist planes, the v' table is built from the full reciprocal lattice."""
    cell = [41.04, 0.0, 0.0, 3.0, 40.0, 0.0, -2.0, 1.5, 39.0]
    phi = synth.random_orbitals(synth.Config("p8k", EDGES, GRID, 3, synth.KERNEL_HSE), 27, 3, cuda_device)
    psi = synth.random_orbitals(synth.Config("p8k", EDGES, GRID, 3, synth.KERNEL_HSE), 28, 2, cuda_device)
    with binding.Plan(cell, GRID, 3, 2, synth.KERNEL_HSE, 0.106, 1.0) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
    ref = oracle.apply(cell, GRID, synth.KERNEL_HSE, 0.106, 1.0, phi.cpu().numpy(), psi.cpu().numpy(), None)
    assert _rel(out.cpu().numpy(), ref) <= TOL


def test_repeated_applies_are_bit_identical(cuda_device):
    """No atomics on the path: every apply must reproduce the same bits; a hazard in the TMA rings or the in-place
    exchanges would show up as run-to-run noise.  20 orbitals per CTA loop = many trips around the rings."""
    cfg = synth.Config("p8r", EDGES, GRID, 20, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 31, 20, cuda_device)
    psi = synth.random_orbitals(cfg, 32, 7, cuda_device)
    with binding.plan_for(cfg, max_targets=7) as plan:
        first = plan.apply(phi, psi).clone()
        for _ in range(4):
            again = plan.apply(phi, psi)
            torch.cuda.synchronize()
            assert torch.equal(first, again)
    ref = _oracle(cfg, phi, psi[[0, 6]].contiguous())
    assert _rel(first[[0, 6]].cpu().numpy(), ref) <= TOL


def test_two_streams_back_to_back(cuda_device):
    """Two applies on the same plan queued on different streams without a host sync in between: the second waits for
    the first on the device (the plan's scratch is shared), so both results are right."""
    cfg = synth.Config("p8t", EDGES, GRID, 6, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 51, 6, cuda_device)
    psi_a = synth.random_orbitals(cfg, 52, 4, cuda_device)
    psi_b = synth.random_orbitals(cfg, 53, 4, cuda_device)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(cuda_device), torch.cuda.Stream(cuda_device)
    with binding.plan_for(cfg, max_targets=4, block_i=2, block_j=2) as plan:
        out_a = torch.empty_like(psi_a)
        out_b = torch.empty_like(psi_b)
        for _ in range(3):
            with torch.cuda.stream(s1):
                plan.apply(phi, psi_a, out=out_a)
            with torch.cuda.stream(s2):
                plan.apply(phi, psi_b, out=out_b)
        torch.cuda.synchronize()
    assert _rel(out_a.cpu().numpy(), _oracle(cfg, phi, psi_a)) <= TOL
    assert _rel(out_b.cpu().numpy(), _oracle(cfg, phi, psi_b)) <= TOL


def test_wrong_device_pointer_is_rejected(cuda_device):
    cfg = synth.Config("p8e", EDGES, (16, 16, 16), 2, synth.KERNEL_HSE)
    with binding.plan_for(cfg) as plan:
        host = torch.zeros((2, 16, 16, 16), dtype=torch.complex128).pin_memory()
        import ctypes
        rc = binding.lib().ptfock_apply(plan._h, ctypes.c_void_p(host.data_ptr()), None, 0, 2,
                                        ctypes.c_void_p(host.data_ptr()), None)
        assert rc == -1


# ---- the same two-stage kernels instantiated for 32^3 (Si64: 4 x 2 | 16 slab stages, 2 x 8 | 16 pencil stages): thread
# ---- counts differ between the stages (guards)
@pytest.mark.parametrize("n", [32, 48])
def test_small_cubic_grids_general_and_symmetric(cuda_device, n):
    edges = (10.26 * n / 16,) * 3
    cfg = synth.Config("p8n", edges, (n, n, n), 7, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 31, 7, cuda_device)
    psi = synth.random_orbitals(cfg, 32, 5, cuda_device)
    outs = []
    for flags in (0, binding.FLAG_THREE_STAGE_SLABS):
        with binding.plan_for(cfg, max_targets=5, block_i=4, block_j=3, flags=flags) as plan:
            outs.append(plan.apply(phi, psi))           # ragged i and j blocks, two waves in flight
            torch.cuda.synchronize()
            assert plan.info()["pass8"] == (0 if flags else 1)
    ref = _oracle(cfg, phi, psi)
    assert _rel(outs[0].cpu().numpy(), ref) <= TOL and _rel(outs[1].cpu().numpy(), ref) <= TOL
    # symmetric schedule with triangular diagonal blocks and the conj(W) accumulate, bare Coulomb
    cfg2 = synth.Config("p8ns", edges, (n, n, n), 6, synth.KERNEL_COULOMB)
    with binding.plan_for(cfg2, block_i=2, block_j=2) as plan:
        sym = plan.apply(phi[:6].contiguous())
        again = plan.apply(phi[:6].contiguous())
        torch.cuda.synchronize()
        info = plan.info()
    assert info["last_symmetric"] == 1 and info["last_pairs"] == 21 and info["pass8"] == 1
    assert torch.equal(sym, again)
    assert _rel(sym.cpu().numpy(), _oracle(cfg2, phi[:6])) <= TOL


@pytest.mark.parametrize("n", [32, 48])
def test_small_cubic_grids_skew_cell(cuda_device, n):
    """A skew cell: the v' table has no symmetry to lean on, every (k0, k1, k2) -> table slot must be right."""
    a = 10.26 * n / 16
    cell = [a, 0.0, 0.0, 0.21 * a, 0.93 * a, 0.0, 0.13 * a, -0.17 * a, 1.07 * a]
    cfg = synth.Config("p8k", (a, a, a), (n, n, n), 2, synth.KERNEL_HSE)
    phi = synth.random_orbitals(cfg, 33, 2, cuda_device)
    psi = synth.random_orbitals(cfg, 34, 1, cuda_device)
    with binding.Plan(cell, (n, n, n), 2, 1, synth.KERNEL_HSE, 0.106, 1.0) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
        assert plan.info()["pass8"] == 1
    ref = oracle.apply(cell, (n, n, n), synth.KERNEL_HSE, 0.106, 1.0, phi.cpu().numpy(), psi.cpu().numpy(), None)
    assert _rel(out.cpu().numpy(), ref) <= TOL
