"""GPU vs oracle parity (T9 of SURVEY.md 8(c)): every call goes through the C ABI (binding -> libptfock.so).

Bar (BASELINE.json north_star): max_{j,r} |gpu - ref| / max_{j,r} |ref| <= 1e-10.  The transforms are exact
circular convolutions in fp64, so the observed error is ~1e-15..1e-13.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _rel(got, ref):
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def _oracle(cfg, phi, psi=None, cols=None):
    return oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(),
                        None if psi is None else psi.cpu().numpy(), cols)


SMALL = [
    # name, edges, grid, n_occ, kernel, separate psi
    ("c16", (10.26,) * 3, (16, 16, 16), 5, synth.KERNEL_HSE, False),          # three-pass path (the flag below)
    ("c16ns", (10.26,) * 3, (16, 16, 16), 5, synth.KERNEL_COULOMB, True),
    ("g16x32x16", (9.0, 17.0, 12.0), (16, 32, 16), 4, synth.KERNEL_HSE, True),
    ("g32x16x32", (15.0, 9.0, 17.0), (32, 16, 32), 3, synth.KERNEL_COULOMB, False),
    ("g48x16x48", (22.0, 9.0, 23.0), (48, 16, 48), 3, synth.KERNEL_HSE, True),
    ("g64x48x32", (30.0, 22.0, 16.0), (64, 48, 32), 2, synth.KERNEL_HSE, True),
    ("g128x32x64", (50.0, 16.0, 30.0), (128, 32, 64), 2, synth.KERNEL_HSE, True),
    ("g32x128x48", (16.0, 50.0, 22.0), (32, 128, 48), 2, synth.KERNEL_COULOMB, False),
    ("g120x16x16", (82.08, 10.26, 10.26), (120, 16, 16), 3, synth.KERNEL_HSE, True),     # radix-15 pencil (paper grid)
    ("g120x90x60", (82.08, 61.56, 41.04), (120, 90, 60), 2, synth.KERNEL_HSE, False),    # the paper's 60x90x120 grid
]


@pytest.mark.parametrize("case", SMALL, ids=[c[0] for c in SMALL])
def test_small_grids_every_codelet(cuda_device, case):
    """Every supported edge length on every axis role (pencil x0, slab x1, slab x2), noise inputs."""
    name, edges, n, n_occ, kernel, sep = case
    cfg = synth.Config(name, edges, n, n_occ, kernel, separate_psi=sep)
    phi = synth.random_orbitals(cfg, 11, n_occ, cuda_device)
    psi = synth.random_orbitals(cfg, 12, 3, cuda_device) if sep else None
    with binding.plan_for(cfg, block_i=2, block_j=2, flags=binding.FLAG_THREE_STAGE_SLABS) as plan:
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL


# every slab shape (n1, n2) from {16, 32, 48, 64, 128}^2 that round 3 opened on the generic passes (north_star (1): "grid
# edges 16/32/48/64/128"; include/ptfock.h), on a 16-point pencil axis, plus three of them under long pencils
OPENED = [(16, n1, n2) for n1, n2 in [(16, 64), (16, 128), (32, 48), (32, 128), (48, 16), (48, 64), (48, 128), (64, 16), (64, 32),
                                      (64, 48), (64, 128), (128, 16), (128, 32), (128, 64)]] + \
         [(64, 64, 128), (128, 128, 64), (48, 64, 48)]


@pytest.mark.parametrize("n", OPENED, ids=["x".join(map(str, n)) for n in OPENED])
def test_opened_slab_shapes(cuda_device, n):
    edges = tuple(0.64 * k + 0.1 * d for d, k in enumerate(n))          # anisotropic spacing: a swapped axis shows
    cfg = synth.Config("open", edges, n, 2, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 71, 2, cuda_device)
    psi = synth.random_orbitals(cfg, 72, 2, cuda_device)
    with binding.plan_for(cfg, max_targets=2) as plan:
        out = plan.apply(phi, psi)
        sym = plan.apply(phi)                                           # Psi = Phi: the pair-symmetric schedule
        torch.cuda.synchronize()
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi, psi)) <= TOL
    assert _rel(sym.cpu().numpy(), _oracle(cfg, phi)) <= TOL


def test_debug_pair_matches_oracle_W(cuda_device):
    cfg = synth.Config("w", (9.0, 17.0, 12.0), (16, 32, 16), 2, synth.KERNEL_HSE, alpha=0.25)
    ab = synth.random_orbitals(cfg, 5, 2, cuda_device)
    with binding.plan_for(cfg) as plan:
        w = plan.debug_pair(ab[0], ab[1]).cpu().numpy()
    ref = -cfg.alpha * oracle.pair_w(cfg.cell, cfg.n, cfg.kernel, cfg.omega, ab[0].cpu().numpy(), ab[1].cpu().numpy())
    assert _rel(w, ref) <= TOL


def test_Si8_full(cuda_device):
    """Si8 through the three-pass path (symmetric schedule); the default on-chip kernel: tests/test_gpu_onchip16.py."""
    cfg = synth.CONFIGS["Si8"]
    phi = synth.orbitals(cfg, device=cuda_device)
    with binding.plan_for(cfg, flags=binding.FLAG_THREE_STAGE_SLABS) as plan:
        out = plan.apply(phi)
        e = plan.exchange_energy(phi, vx_psi=out)
        e2 = plan.exchange_energy(phi)
        info = plan.info()
    assert info["last_symmetric"] == 1 and info["pass8"] == 0
    ref = _oracle(cfg, phi)
    assert _rel(out.cpu().numpy(), ref) <= TOL
    e_ref = oracle.exchange_energy(cfg.cell, cfg.n, phi.cpu().numpy(), ref)
    assert abs(e - e_ref.real) <= TOL * abs(e_ref.real) and abs(e2 - e_ref.real) <= TOL * abs(e_ref.real)
    assert e < 0.0


def test_Si64_full(cuda_device):
    cfg = synth.CONFIGS["Si64"]
    phi = synth.orbitals(cfg, device=cuda_device)
    with binding.plan_for(cfg) as plan:
        out = plan.apply(phi)
        torch.cuda.synchronize()
        assert plan.info()["last_symmetric"] == 1
    assert _rel(out.cpu().numpy(), _oracle(cfg, phi)) <= TOL


@pytest.mark.parametrize("flags", [0, binding.FLAG_THREE_STAGE_SLABS], ids=["two_stage", "three_stage"])
def test_schedules_agree(cuda_device, flags):
    """Symmetric schedule == general schedule on a copy of Phi == j-blocked calls; ragged tiles.  32^3: the two-stage
    kernels (csrc/pass8.cuh) by default, the three-stage ones behind the flag."""
    cfg = synth.Config("s", (20.52,) * 3, (32, 32, 32), 13, synth.KERNEL_HSE)
    phi = synth.orbitals(cfg, device=cuda_device)
    with binding.plan_for(cfg, block_i=4, block_j=4, flags=flags) as plan:
        sym = plan.apply(phi)
        assert plan.info()["last_symmetric"] == 1 and plan.info()["pass8"] == (0 if flags else 1)
        gen = plan.apply(phi, phi.clone())
        assert plan.info()["last_symmetric"] == 0
        blk = torch.cat([plan.apply(phi, None, self_offset=o, n_targets=min(5, 13 - o)) for o in range(0, 13, 5)])
        torch.cuda.synchronize()
    ref = _oracle(cfg, phi)
    for got in (sym, gen, blk):
        assert _rel(got.cpu().numpy(), ref) <= TOL


def test_host_path_and_stream(cuda_device):
    cfg = synth.Config("h", (10.26,) * 3, (16, 16, 16), 6, synth.KERNEL_HSE, separate_psi=True)
    phi, psi = synth.make_case(cfg, cuda_device)
    with binding.plan_for(cfg) as plan:
        ref = plan.apply(phi, psi)
        host = plan.apply_host(phi.cpu().pin_memory(), psi.cpu().pin_memory())
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            on_s = plan.apply(phi, psi)
        s.synchronize()
        torch.cuda.synchronize()
    assert torch.equal(host, ref.cpu()) and torch.equal(on_s, ref)
    # host path, Psi = Phi: the chunked, overlapped copies (chunk = block_i orbitals) must not change a bit --
    # symmetric schedule (whole set), a streamed j-block whose targets sit in a later chunk, several j-blocks
    cfg2 = synth.Config("h2", (10.26,) * 3, (16, 16, 16), 7, synth.KERNEL_COULOMB)
    phi2 = synth.random_orbitals(cfg2, 3, 7, cuda_device)
    hphi = phi2.cpu().pin_memory()
    with binding.plan_for(cfg2, block_i=2, block_j=2, flags=binding.FLAG_THREE_STAGE_SLABS) as plan:
        for off, nt in ((0, 7), (5, 2), (1, 5)):
            dev = plan.apply(phi2, None, self_offset=off, n_targets=nt)
            sym = plan.info()["last_symmetric"]
            host = plan.apply_host(hphi, None, self_offset=off, n_targets=nt)
            torch.cuda.synchronize()
            assert sym == (1 if nt == 7 else 0)
            assert torch.equal(host, dev.cpu()), (off, nt)
        # separate Psi through the host path: Psi arrives in chunks of block_j targets, `out` leaves block by block
        # during the last i block (ragged last chunks on both sides); a second call reuses the events
        psi2 = synth.random_orbitals(cfg2, 4, 5, cuda_device)
        hpsi = psi2.cpu().pin_memory()
        dev = plan.apply(phi2, psi2)
        for _ in range(2):
            host = plan.apply_host(hphi, hpsi)
            assert torch.equal(host, dev.cpu())
        host1 = plan.apply_host(hphi, hpsi[:1].contiguous().pin_memory())
        assert torch.equal(host1, dev[:1].cpu())


def test_edge_cases_and_errors(cuda_device):
    cfg = synth.Config("e", (10.26,) * 3, (16, 16, 16), 3, synth.KERNEL_HSE)
    phi = synth.random_orbitals(cfg, 1, 3, cuda_device)
    with binding.plan_for(cfg) as plan:
        empty = plan.apply(phi, None, n_targets=0)
        assert empty.shape[0] == 0
        one = plan.apply(phi, None, self_offset=2, n_targets=1)
        assert _rel(one.cpu().numpy(), _oracle(cfg, phi, cols=[2])) <= TOL
        with pytest.raises(binding.PtfockError) as ei:
            plan.apply(phi, None, out=phi)                       # alias
        assert ei.value.code == -7
        with pytest.raises(binding.PtfockError) as ei:
            plan.apply(phi, None, self_offset=2, n_targets=2)    # out of range
        assert ei.value.code == -1
        mis_ptr = phi.data_ptr() + 8
        with pytest.raises(binding.PtfockError) as ei:
            binding._check(binding.lib().ptfock_apply(plan._h, mis_ptr, None, 0, 3, phi.data_ptr(), None), "x")
        assert ei.value.code == -4
    with pytest.raises(binding.PtfockError) as ei:
        binding.Plan(cfg.cell, (16, 20, 16), 3)
    assert ei.value.code == -2
    with pytest.raises(binding.PtfockError) as ei:
        binding.Plan(cfg.cell, (16, 16, 16), 3, kernel=5)
    assert ei.value.code == -1
    # single orbital, n_occ = 1
    cfg1 = synth.Config("one", (10.26,) * 3, (16, 16, 16), 1, synth.KERNEL_COULOMB)
    p1 = synth.random_orbitals(cfg1, 2, 1, cuda_device)
    with binding.plan_for(cfg1) as plan:
        o1 = plan.apply(p1)
    assert _rel(o1.cpu().numpy(), _oracle(cfg1, p1)) <= TOL


def test_oversized_tile_is_clamped(cuda_device):
    """block_i x block_j beyond what one launch can index (pass B: pairs on gridDim.y <= 65535) is reduced at plan
    creation instead of failing at launch."""
    cfg = synth.Config("big", (10.26,) * 3, (16, 16, 16), 300, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 7, 300, cuda_device)
    psi = synth.random_orbitals(cfg, 8, 300, cuda_device)
    with binding.plan_for(cfg, block_i=300, block_j=300, flags=binding.FLAG_THREE_STAGE_SLABS) as plan:
        info = plan.info()
        assert info["block_i"] * info["block_j"] <= 65535
        out = plan.apply(phi, psi)
        torch.cuda.synchronize()
    cols = [0, 149, 299]
    ref = _oracle(cfg, phi, psi[cols].contiguous())
    assert _rel(out[cols].cpu().numpy(), ref) <= TOL


def test_symmetric_blocks_stay_launchable(cuda_device):
    """Psi = Phi with 512 orbitals on 16^3: the square block of the symmetric schedule must stop doubling before
    block^2 pair-solves exceed what one launch can index."""
    cfg = synth.Config("sym512", (10.26,) * 3, (16, 16, 16), 512, synth.KERNEL_COULOMB)
    phi = synth.random_orbitals(cfg, 9, 512, cuda_device)
    with binding.plan_for(cfg, flags=binding.FLAG_THREE_STAGE_SLABS) as plan:
        out = plan.apply(phi)
        torch.cuda.synchronize()
        assert plan.info()["last_symmetric"] == 1
    cols = [0, 255, 511]
    ref = _oracle(cfg, phi, cols=cols)
    assert _rel(out[cols].cpu().numpy(), ref) <= TOL
