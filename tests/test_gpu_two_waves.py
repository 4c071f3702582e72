"""Two waves in flight (general schedule): j-blocks with an odd index run on the plan's aux stream in a second scratch
slot.  The result must be bit-identical to the single-stream schedule (PTFOCK_FLAG_SINGLE_STREAM) and match the oracle
(Eq. (3); Alg. 2: the j loop's iterations are independent)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1905_01348_b200 import binding, synth

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("n,flags", [((16, 32, 16), 0), ((64, 64, 64), 0), ((64, 64, 64), binding.FLAG_THREE_STAGE_SLABS),
                                     ((16, 128, 48), 0)])
def test_two_slots_equal_single_stream_and_oracle(cuda_device, n, flags):
    cell = (10.26 * n[0] / 16, 10.26 * n[1] / 16, 10.26 * n[2] / 16)
    cfg = synth.Config("tw", cell, n, 5, synth.KERNEL_HSE, separate_psi=True)
    phi = synth.random_orbitals(cfg, 11, 5, cuda_device)
    psi = synth.random_orbitals(cfg, 12, 7, cuda_device)
    outs = {}
    for single in (0, binding.FLAG_SINGLE_STREAM):
        with binding.plan_for(cfg, max_targets=7, block_i=2, block_j=2, flags=flags | single) as plan:
            assert plan.info()["slots"] == (1 if single else 2)
            a = plan.apply(phi, psi)                    # 4 j-blocks (ragged last), 3 i-blocks (ragged last)
            b = plan.apply(phi, psi)
            blk = plan.apply(phi, None, self_offset=1, n_targets=4)   # targets inside Phi, two j-blocks
            e = plan.exchange_energy(phi, psi)           # apply into the plan's buffer, then the reduction on `stream`
            host = plan.apply_host(phi.cpu().pin_memory(), psi.cpu().pin_memory())
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                on_s = plan.apply(phi, psi)
            s.synchronize()
            torch.cuda.synchronize()
            assert torch.equal(a, b) and torch.equal(on_s, a) and torch.equal(host, a.cpu())
            outs[single] = (a, blk, e)
    assert torch.equal(outs[0][0], outs[binding.FLAG_SINGLE_STREAM][0])
    assert torch.equal(outs[0][1], outs[binding.FLAG_SINGLE_STREAM][1])
    assert outs[0][2] == outs[binding.FLAG_SINGLE_STREAM][2]
    ref = oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(), psi.cpu().numpy())
    assert _rel(outs[0][0].cpu().numpy(), ref) <= TOL
    e_ref = oracle.exchange_energy(cfg.cell, cfg.n, psi.cpu().numpy(), ref).real
    assert abs(outs[0][2] - e_ref) <= 1e-10 * abs(e_ref)


def test_workspace_bound_keeps_one_slot(cuda_device):
    cfg = synth.Config("tw1", (10.26,) * 3, (16, 32, 16), 4, synth.KERNEL_COULOMB, separate_psi=True)
    phi, psi = synth.make_case(cfg, cuda_device)
    pair = 16 * 16 * 32 * 16
    with binding.plan_for(cfg, block_i=2, block_j=2, workspace_bytes=4 * pair) as one, \
            binding.plan_for(cfg, block_i=2, block_j=2, workspace_bytes=8 * pair) as two:
        assert one.info()["slots"] == 1 and two.info()["slots"] == 2
        # the bound is an upper bound on the whole scratch: the dense-algebra minimum does not inflate it (ptfock.h)
        assert one.info()["scratch_bytes"] <= 4 * pair and two.info()["scratch_bytes"] <= 8 * pair
        assert torch.equal(one.apply(phi, psi), two.apply(phi, psi))
