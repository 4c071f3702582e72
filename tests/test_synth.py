"""Input generator (paper_1905_01348_b200/synth.py): recipe of BASELINE.json configs / SURVEY.md 8(d)."""
import math

import numpy as np
import pytest
import torch

from paper_1905_01348_b200 import synth


def test_splitmix_matches_python_integers():
    z = torch.tensor([0, 1, 2, 12345678901234], dtype=torch.int64)
    got = synth._splitmix64(z).tolist()
    for a, g in zip(z.tolist(), got):
        assert (g & ((1 << 64) - 1)) == synth._splitmix64_int(a)


def test_normals_are_counter_based_and_standard():
    idx = torch.arange(200000, dtype=torch.int64)
    a, b = synth._normals(7, idx)
    a2, _ = synth._normals(7, idx[1000:1010])
    assert torch.equal(a[1000:1010], a2)                      # order independent
    for x in (a, b):
        assert abs(float(x.mean())) < 0.01 and abs(float(x.std()) - 1.0) < 0.01
    assert abs(float((a * b).mean())) < 0.01


@pytest.mark.parametrize("name,pw", [("Si8", 1647), ("Si64", 13133)])
def test_sphere_counts(name, pw):
    """Plane-wave counts of SURVEY.md Sec. 8 table (computed there independently)."""
    k_lin, g2 = synth.sphere(synth.CONFIGS[name])
    assert k_lin.numel() == pw
    assert float(g2.max()) / 2 <= synth.ECUT_HA
    assert torch.unique(k_lin).numel() == pw


def test_si8_orbitals_orthonormal_and_band_limited():
    cfg = synth.CONFIGS["Si8"]
    phi = synth.orbitals(cfg)
    assert phi.shape == (16, 16, 16, 16) and phi.dtype == torch.complex128
    flat = phi.reshape(16, -1)
    S = (flat.conj() @ flat.T) * (cfg.volume / cfg.N)
    assert torch.allclose(S, torch.eye(16, dtype=torch.complex128), atol=1e-12)
    spec = torch.fft.fftn(phi, dim=(1, 2, 3)).reshape(16, -1)
    k_lin, _ = synth.sphere(cfg)
    mask = torch.ones(cfg.N, dtype=torch.bool)
    mask[k_lin] = False
    assert float(spec[:, mask].abs().max()) < 1e-10 * float(spec.abs().max())
    # deterministic
    assert torch.equal(phi, synth.orbitals(cfg))
    assert not torch.equal(phi, synth.orbitals(cfg, seed=cfg.seed_psi))


def test_noncubic_config_and_make_case():
    cfg = synth.Config("t", (9.0, 12.0, 7.0), (16, 32, 16), 5, synth.KERNEL_HSE, separate_psi=True)
    phi, psi = synth.make_case(cfg)
    assert phi.shape == (5, 16, 32, 16) and psi.shape == phi.shape
    nrm = (phi.abs() ** 2).sum(dim=(1, 2, 3)) * cfg.volume / cfg.N
    assert torch.allclose(nrm, torch.ones(5, dtype=torch.float64), atol=1e-12)
    r = synth.random_orbitals(cfg, 3, 2)
    assert r.shape == (2, 16, 32, 16)
