"""GPU vs oracle on the BASELINE.json configs at FULL size, in the launch configuration bench.py times,
checked on sampled output columns the oracle can compute one by one (each column sums over all i)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _oracle_columns(cfg, phi_np, tgt_np, parts=None):
    """oracle.apply for a few target columns with the sum over i split into `parts` slices of Phi run side by side
    (V_X[Phi] psi = sum_i ... is a plain sum of per-orbital terms; the oracle's own OpenMP runs over target columns
    only, which leaves the host cores idle when one or two columns are checked).  Partial sums are added in fp64."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    n_occ = phi_np.shape[0]
    if parts is None:
        parts = max(1, min(n_occ, (os.cpu_count() or 8) // max(1, tgt_np.shape[0])))
    bounds = np.linspace(0, n_occ, parts + 1).astype(int)

    def run(k):
        return oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha,
                            np.ascontiguousarray(phi_np[bounds[k]:bounds[k + 1]]), tgt_np, None)

    with ThreadPoolExecutor(parts) as ex:
        res = list(ex.map(run, range(parts)))
    total = res[0].copy()
    for r in res[1:]:
        total += r
    return total


def _check_cols(cfg, phi, tgt, out, cols, offset=0):
    ref = _oracle_columns(cfg, phi.cpu().numpy(), np.ascontiguousarray(tgt[[c + offset for c in cols]].cpu().numpy()))
    got = out[cols].cpu().numpy()
    err = float(np.abs(got - ref).max() / np.abs(ref).max())
    assert err <= TOL, err
    return err


def test_Si216_symmetric_full(cuda_device):
    cfg = synth.CONFIGS["Si216"]
    phi = synth.orbitals(cfg, device=cuda_device)
    with binding.plan_for(cfg) as plan:
        out = plan.apply(phi)
        torch.cuda.synchronize()
        info = plan.info()
    assert info["last_symmetric"] == 1 and info["last_pairs"] < cfg.n_occ ** 2
    _check_cols(cfg, phi, phi, out, [0, 100, 215, 431])


def test_Si512_nonself_full(cuda_device):
    cfg = synth.CONFIGS["Si512"]
    phi, psi = synth.make_case(cfg, cuda_device)
    with binding.plan_for(cfg) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
        info = plan.info()
        e = plan.exchange_energy(phi, psi, vx_psi=out)
    assert info["last_symmetric"] == 0 and info["last_pairs"] == 1024 * 1024
    # first / last columns of j-tiles and tile interiors (J_b = 16): 0, 5 | 517 | 1000, 1023
    cols = [0, 5, 517, 1000, 1023]
    ref = _oracle_columns(cfg, phi.cpu().numpy(), np.ascontiguousarray(psi[cols].cpu().numpy()))
    got = out[cols].cpu().numpy()
    assert float(np.abs(got - ref).max() / np.abs(ref).max()) <= TOL
    # E_x = sum over ALL columns of the library's result, so the check is: the library's dot-product reduction agrees with
    # the oracle's formula applied to the library's own V_X Psi (pins the reduction and the 1/2 Omega/N prefactor at full
    # size), and the sampled columns' contributions agree with the oracle's columns
    e_lib_cols = oracle.exchange_energy(cfg.cell, cfg.n, psi[cols].cpu().numpy(), got).real
    e_ref_cols = oracle.exchange_energy(cfg.cell, cfg.n, psi[cols].cpu().numpy(), ref).real
    assert abs(e_lib_cols - e_ref_cols) <= TOL * abs(e_ref_cols)
    with binding.plan_for(cfg, max_targets=len(cols)) as plan2:
        e_cols = plan2.exchange_energy(phi, psi[cols].contiguous())
    assert abs(e_cols - e_ref_cols) <= TOL * abs(e_ref_cols) and e_cols < 0.0
    assert np.isfinite(e) and e < e_cols


def test_Si1536_streamed_j_blocks(cuda_device):
    """Two j-blocks of 96 (first and an interior one) of the 3072-orbital, 128x128x48 case (38.65 GB of Phi)."""
    cfg = synth.CONFIGS["Si1536"]
    phi = synth.orbitals(cfg, device=cuda_device)
    host = phi.cpu().numpy()
    with binding.plan_for(cfg) as plan:
        out = torch.empty((cfg.j_block,) + cfg.n, dtype=torch.complex128, device=cuda_device)
        # one tile-edge and one tile-interior column (J_b = 8) per block
        refs = {}
        for offset, cols in ((0, [0, 43]), (1536, [50, 95])):
            plan.apply(phi, None, out=out, self_offset=offset, n_targets=cfg.j_block)
            torch.cuda.synchronize()
            assert plan.info()["last_pairs"] == 96 * 3072
            ref = _oracle_columns(cfg, host, np.ascontiguousarray(host[[offset + c for c in cols]]))
            got = out[cols].cpu().numpy()
            err = float(np.abs(got - ref).max() / np.abs(ref).max())
            assert err <= TOL, (offset, err)
            for k, c in enumerate(cols):
                refs[offset + c] = ref[k]
        # the whole application in ONE call (Phi and out both resident: 2 x 38.65 GB): the pair-symmetric schedule over
        # all block pairs executes n (n + 1) / 2 pair-solves and must give the same columns
        del out
        full = plan.apply(phi)
        torch.cuda.synchronize()
        info = plan.info()
        assert info["last_symmetric"] == 1 and info["last_pairs"] == 3072 * 3073 // 2
        for c, ref in refs.items():
            err = float(np.abs(full[c].cpu().numpy() - ref).max() / np.abs(ref).max())
            assert err <= TOL, (c, err)


def test_Si1536p_paper_grid_j_block(cuda_device):
    """the paper's own workload (60 x 90 x 120 grid as 120 x 90 x 60, 3072 orbitals),
    one interior j-block of 96, one sampled column against the oracle (radix-5 / 15 codelets, DFT15 slab stages)."""
    cfg = synth.CONFIGS["Si1536p"]
    phi = synth.orbitals(cfg, device=cuda_device)
    host = phi.cpu().numpy()
    with binding.plan_for(cfg) as plan:
        out = torch.empty((cfg.j_block,) + cfg.n, dtype=torch.complex128, device=cuda_device)
        offset, col = 960, 17
        plan.apply(phi, None, out=out, self_offset=offset, n_targets=cfg.j_block)
        torch.cuda.synchronize()
        assert plan.info()["last_pairs"] == 96 * 3072
    ref = _oracle_columns(cfg, host, host[offset + col:offset + col + 1])
    got = out[col].cpu().numpy()
    err = float(np.abs(got - ref[0]).max() / np.abs(ref[0]).max())
    assert err <= TOL, err
