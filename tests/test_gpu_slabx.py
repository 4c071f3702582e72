"""GPU vs oracle parity for the TMA-fed slab kernels (csrc/slabx.cuh), which serve the (x1, x2) slabs of the
Si512 (64 x 64), Si1536 (128 x 48), Si216 (48 x 48) and Si64 (32 x 32) configs.  A short x0 axis keeps the oracle fast; the cases walk through the
paths the full-size runs do not isolate: fewer loop iterations than rotating tiles (1, 2, 3 orbitals per CTA),
ragged waves, the split i loop of pass A, the conj(W) accumulate of the pair-symmetric schedule, j-blocks.

Bar (BASELINE.json north_star): max |gpu - ref| / max |ref| <= 1e-10; every call goes through the C ABI.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10

SHAPES = [
    ("s64x64", (11.0, 41.04, 41.04), (16, 64, 64)),        # kind P, bulk stores, three tiles
    ("s128x48", (11.0, 82.08, 30.78), (16, 128, 48)),      # kind Q, 24-point stage, two tiles
    ("s48x48", (11.0, 30.78, 30.78), (16, 48, 48)),        # kind Q, 9-point stage, 144-task DFT16 stages
    ("s32x32", (11.0, 20.52, 20.52), (16, 32, 32)),        # kind Q, 4-point stage, 64-task DFT16 stages (32^3 itself: pass8)
    ("s90x60", (11.0, 61.56, 41.04), (16, 90, 60)),        # paper grid's slab: 24-point stage (6 x 4), DFT15 stages, 225 of 256 threads in stage 1
]


def _rel(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def _oracle(cfg, phi, psi=None, cols=None):
    return oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(),
                        None if psi is None else psi.cpu().numpy(), cols)


@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
@pytest.mark.parametrize("n_occ,n_t,bi,bj", [(1, 1, 1, 1), (2, 3, 2, 2), (3, 2, 3, 1), (7, 3, 4, 2), (9, 5, 0, 0)])
def test_general_schedule_ragged(cuda_device, shape, n_occ, n_t, bi, bj):
    """Non-self targets; n_occ = 1, 2, 3 exercise loops shorter than the tile ring, (7, 4) a ragged last wave,
    and the tiny grids make pass A split its i loop over blockIdx.z."""
    name, edges, n = shape
    cfg = synth.Config(name, edges, n, n_occ, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 21, n_occ, cuda_device)
    psi = synth.random_orbitals(cfg, 22, n_t, cuda_device)
    with binding.plan_for(cfg, max_targets=n_t, block_i=bi, block_j=bj) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
        assert plan.info()["last_pairs"] == n_occ * n_t
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL


@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
def test_symmetric_schedule_uses_conj_accumulate(cuda_device, shape):
    """Psi = Phi with blocks smaller than n_occ: off-diagonal block pairs feed out_i through conj(W_ij)."""
    name, edges, n = shape
    cfg = synth.Config(name, edges, n, 6, synth.KERNEL_COULOMB)
    phi = synth.random_orbitals(cfg, 23, 6, cuda_device)
    with binding.plan_for(cfg, block_i=2, block_j=2) as plan:
        out = plan.apply(phi)
        torch.cuda.synchronize()
        info = plan.info()
    assert info["last_symmetric"] == 1 and info["last_pairs"] < 36
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi)) <= TOL


@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
def test_j_blocks_and_energy(cuda_device, shape):
    """Streamed j-blocks (psi = NULL, self_offset) equal the columns of the full result; E_x from the blocks."""
    name, edges, n = shape
    cfg = synth.Config(name, edges, n, 5, synth.KERNEL_HSE)
    phi = synth.orbitals(cfg, device=cuda_device)                      # smooth, orthonormal orbitals
    ref = _oracle(cfg, phi)
    with binding.plan_for(cfg, max_targets=2) as plan:
        blocks, e = [], 0.0
        for o in (0, 2, 4):
            nt = min(2, 5 - o)
            blk = plan.apply(phi, None, self_offset=o, n_targets=nt)
            e += plan.exchange_energy(phi, None, vx_psi=blk, self_offset=o, n_targets=nt)
            blocks.append(blk)
        torch.cuda.synchronize()
    got = torch.cat(blocks).cpu().numpy()
    assert _rel(got, ref) <= TOL
    e_ref = oracle.exchange_energy(cfg.cell, cfg.n, phi.cpu().numpy(), ref).real
    assert abs(e - e_ref) <= TOL * abs(e_ref) and e < 0.0


@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
def test_single_pair_W(cuda_device, shape):
    """One W_ij through the three passes (ptfock_debug_pair) against the oracle's pair solve."""
    name, edges, n = shape
    cfg = synth.Config(name, edges, n, 2, synth.KERNEL_HSE, alpha=0.5)
    ab = synth.random_orbitals(cfg, 24, 2, cuda_device)
    with binding.plan_for(cfg) as plan:
        w = plan.debug_pair(ab[0], ab[1]).cpu().numpy()
    ref = -cfg.alpha * oracle.pair_w(cfg.cell, cfg.n, cfg.kernel, cfg.omega, ab[0].cpu().numpy(), ab[1].cpu().numpy())
    assert _rel(w, ref) <= TOL


@pytest.mark.parametrize("shape", SHAPES[:2], ids=[s[0] for s in SHAPES[:2]])
def test_repeated_applies_are_bit_identical(cuda_device, shape):
    """No atomics anywhere on the path, so every apply must reproduce the same bits; a shared-memory / bulk-copy
    hazard in the rotating tiles (compute-sanitizer is closed on this pool) would show up as run-to-run noise.
    40 orbitals per CTA loop = many trips around the tile ring; sampled columns also checked against the oracle."""
    name, edges, n = shape
    cfg = synth.Config(name, edges, n, 40, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 31, 40, cuda_device)
    psi = synth.random_orbitals(cfg, 32, 9, cuda_device)
    with binding.plan_for(cfg, max_targets=9) as plan:
        first = plan.apply(phi, psi).clone()
        for _ in range(4):
            again = plan.apply(phi, psi)
            torch.cuda.synchronize()
            assert torch.equal(first, again)
    ref = _oracle(cfg, phi, psi[[0, 8]].contiguous())
    assert _rel(first[[0, 8]].cpu().numpy(), ref) <= TOL
