"""GPU vs oracle on the BASELINE.json configs at FULL size, in the launch configuration bench.py times,
checked on sampled output columns the oracle can compute one by one (each column sums over all i)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _check_cols(cfg, phi, tgt, out, cols, offset=0):
    ref = oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(),
                       np.ascontiguousarray(tgt[[c + offset for c in cols]].cpu().numpy()), None)
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
    _check_cols(cfg, phi, psi, out, [0, 511, 1023])
    assert np.isfinite(e)


def test_Si1536_streamed_j_blocks(cuda_device):
    """Two j-blocks of 96 (first and an interior one) of the 3072-orbital, 128x128x48 case (38.65 GB of Phi)."""
    cfg = synth.CONFIGS["Si1536"]
    phi = synth.orbitals(cfg, device=cuda_device)
    host = phi.cpu().numpy()
    with binding.plan_for(cfg) as plan:
        out = torch.empty((cfg.j_block,) + cfg.n, dtype=torch.complex128, device=cuda_device)
        for offset, col in ((0, 0), (1536, 95)):
            plan.apply(phi, None, out=out, self_offset=offset, n_targets=cfg.j_block)
            torch.cuda.synchronize()
            assert plan.info()["last_pairs"] == 96 * 3072
            ref = oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, host, None, [offset + col])
            got = out[col].cpu().numpy()
            err = float(np.abs(got - ref[0]).max() / np.abs(ref[0]).max())
            assert err <= TOL, (offset, err)
