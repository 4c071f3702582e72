"""ptfock_banddot_static: the one entry point of libptfock.so that allocates nothing.

Why it exists: some host codes cannot let a library call cudaMalloc -- they gave every byte of HBM to their own pool at
start-up (a cudaMalloc from us would just fail), or they sit in a time-step loop where the device-wide synchronisation
inside cudaMalloc / cudaFree would stall their copy and communication streams.  Those callers cannot create a plan
either, so the entry point takes none and keeps its per-block partial sums in a fixed 4 MiB array inside the library
image (limit: PTFOCK_STATIC_MAX_BANDS = 4096 bands per call).

What is checked: its output against the existing path (Plan.banddot = ptfock_banddot with plan-owned, cudaMalloc'ed
scratch) on TWO calls in a row -- the second with other data and fewer bands, so that it finds the first call's partial
sums still lying in the shared array and must not be disturbed by them -- plus the size limit and that free device
memory does not shrink across a call.  The operation is the inner product of PAPER.md:194-198 (Sec. 3.4, the
least-squares problems of the Anderson mixing).

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It depends on no other test (runs alone in a fresh process as well).
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_1905_01348_b200 import binding, synth


def test_too_many_bands_is_refused_before_any_cuda_call():
    # argument check only: nothing is dereferenced or launched, so this runs without a GPU
    fake = ctypes.c_void_p(4096)
    rc = binding.lib().ptfock_banddot_static(0, 4096, 1.0, fake, fake, binding.STATIC_MAX_BANDS + 1, fake, None)
    assert rc == -9
    assert b"PTFOCK_STATIC_MAX_BANDS" in binding.lib().ptfock_strerror(rc)
    assert binding.lib().ptfock_banddot_static(0, 0, 1.0, fake, fake, 1, fake, None) == -1          # no grid points
    assert binding.lib().ptfock_banddot_static(0, 4096, 1.0, None, fake, 1, fake, None) == -1       # null input


@pytest.mark.gpu
@pytest.mark.parametrize("n", [(32, 32, 32), (16, 16, 16)], ids=["32^3:16 blocks per band", "16^3:2 blocks per band"])
def test_static_scratch_matches_plan_scratch_on_two_calls_in_a_row(cuda_device, n):
    cfg = synth.Config("noalloc", (9.0, 10.0, 11.0), n, 70, synth.KERNEL_HSE)
    a1 = synth.random_orbitals(cfg, 11, 70, cuda_device)
    b1 = synth.random_orbitals(cfg, 12, 70, cuda_device)
    a2 = synth.random_orbitals(cfg, 13, 5, cuda_device)
    b2 = synth.random_orbitals(cfg, 14, 5, cuda_device)
    with binding.plan_for(cfg) as plan:
        w = 9.0 * 10.0 * 11.0 / plan.N                                  # Omega / N of the orthorhombic cell above
        ref1, ref2 = plan.banddot(a1, b1), plan.banddot(a2, b2)        # existing path: partial sums in the plan's scratch
    out1 = torch.empty(70, dtype=torch.complex128, device=cuda_device)
    out2 = torch.empty(5, dtype=torch.complex128, device=cuda_device)
    binding.banddot_static(a1, b1, w, out=out1)                         # first call on the device: address look-up + launch
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(cuda_device)[0]
    binding.banddot_static(a2, b2, w, out=out2)                         # second call: the array still holds call 1's sums
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(cuda_device)[0] >= free_before       # nothing was allocated on the device
    got1, got2 = out1.cpu().numpy(), out2.cpu().numpy()
    assert np.abs(ref1).max() > 1e-3                                    # the comparison is not 0 == 0
    assert np.abs(got1 - ref1).max() <= 1e-13                           # the bar tests/test_gpu_ptcn.py sets for banddot
    assert np.abs(got2 - ref2).max() <= 1e-13
    assert np.array_equal(got1, ref1) and np.array_equal(got2, ref2)    # same kernels, same order of summation
    # and against the definition, so that "equal to the other path" is not the only anchor
    d = np.array([w * np.vdot(a2[j].cpu().numpy().ravel(), b2[j].cpu().numpy().ravel()) for j in range(5)])
    assert np.abs(got2 - d).max() <= 1e-13


@pytest.mark.gpu
def test_limit_and_pointer_checks_on_the_device(cuda_device):
    big = torch.zeros(binding.STATIC_MAX_BANDS + 1, 16, dtype=torch.complex128, device=cuda_device)
    with pytest.raises(binding.PtfockError) as e:
        binding.banddot_static(big, big, 1.0)
    assert e.value.code == -9
    ok = torch.ones(binding.STATIC_MAX_BANDS, 16, dtype=torch.complex128, device=cuda_device)     # exactly the limit
    got = binding.banddot_static(ok, ok, 0.5).cpu().numpy()
    assert np.array_equal(got, np.full(binding.STATIC_MAX_BANDS, 8.0 + 0j))
    host = torch.zeros(2, 16, dtype=torch.complex128)
    rc = binding.lib().ptfock_banddot_static(0, 16, 1.0, ctypes.c_void_p(host.data_ptr()), ctypes.c_void_p(host.data_ptr()), 2,
                                             ctypes.c_void_p(ok.data_ptr()), None)
    assert rc == -1                                                     # a host pointer is refused, not dereferenced
