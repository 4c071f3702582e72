"""Thin Python face of the C ABI in ``include/ptfock.h`` (argument marshalling only).

Every step of the path runs in the hand-written kernels of ``libptfock.so``; torch is used for device
memory and the stream handle.  There is no CPU fallback: if the library is missing or the device is
not a B200-class GPU the calls raise.  Operation: PAPER.md:57-61 (Eq. 3), PAPER.md:116-144 (Alg. 2).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
LIB_PATH = os.environ.get("PTFOCK_LIB", os.path.join(_HERE, "libptfock.so"))
SRC_DIR = os.path.join(_HERE, "csrc")

KERNEL_COULOMB = 0
KERNEL_HSE = 1
KERNEL_KINETIC = 2
FLAG_THREE_STAGE_SLABS = 1
FLAG_SINGLE_STREAM = 2

EXPORTS = ["ptfock_create", "ptfock_apply", "ptfock_exchange_energy", "ptfock_apply_host", "ptfock_destroy",
           "ptfock_strerror", "ptfock_last_cuda_error", "ptfock_plan_info", "ptfock_debug_pair",
           "ptfock_set_profiling", "ptfock_get_profile", "ptfock_measure_dfma_peak", "ptfock_measure_dmma_peak", "ptfock_measure_copy_bandwidth",
           "ptfock_overlap", "ptfock_rotate", "ptfock_residual", "ptfock_density", "ptfock_orthonormalize",
           "ptfock_hloc_apply", "ptfock_axpby", "ptfock_banddot", "ptfock_banddot_static",
           "ptfock_banddot_many", "ptfock_vloc_update", "ptfock_density_change"]
STATIC_MAX_BANDS = 4096

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "1886"]


class PtfockError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {code}")
        self.code = code


class Desc(ctypes.Structure):
    _fields_ = [("cell", ctypes.c_double * 9), ("n", ctypes.c_int32 * 3), ("n_occ", ctypes.c_int32),
                ("max_targets", ctypes.c_int32), ("kernel", ctypes.c_int32), ("omega", ctypes.c_double),
                ("alpha", ctypes.c_double), ("device", ctypes.c_int32), ("block_i", ctypes.c_int32),
                ("block_j", ctypes.c_int32), ("workspace_bytes", ctypes.c_uint64), ("flags", ctypes.c_uint32)]


def build_library(force: bool = False, verbose: bool = False) -> str:
    """nvcc -> paper_1905_01348_b200/libptfock.so (sm_100a only, built in-tree)."""
    srcs = [os.path.join(SRC_DIR, f) for f in sorted(os.listdir(SRC_DIR))]
    hdr = os.path.join(_ROOT, "include", "ptfock.h")
    newest = max(os.path.getmtime(f) for f in srcs + [hdr])
    if not force and os.path.exists(LIB_PATH) and os.path.getmtime(LIB_PATH) >= newest:
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB_PATH, os.path.join(SRC_DIR, "ptfock.cu")]
    subprocess.run(cmd, check=True)
    return LIB_PATH


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libptfock.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} is missing: run __graft_entry__.build() (nvcc, sm_100a); "
                                    "there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32 = ctypes.c_void_p, ctypes.c_int32
        L.ptfock_create.argtypes = [ctypes.POINTER(Desc), ctypes.POINTER(vp)]
        L.ptfock_apply.argtypes = [vp, vp, vp, i32, i32, vp, vp]
        L.ptfock_exchange_energy.argtypes = [vp, vp, vp, i32, i32, vp, ctypes.POINTER(ctypes.c_double), vp]
        L.ptfock_apply_host.argtypes = [vp, vp, vp, i32, i32, vp, vp]
        L.ptfock_destroy.argtypes = [vp]
        L.ptfock_strerror.argtypes = [ctypes.c_int]
        L.ptfock_strerror.restype = ctypes.c_char_p
        L.ptfock_last_cuda_error.argtypes = []
        L.ptfock_plan_info.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
        L.ptfock_debug_pair.argtypes = [vp, vp, vp, vp, vp]
        L.ptfock_set_profiling.argtypes = [vp, i32]
        L.ptfock_get_profile.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64), i32]
        L.ptfock_measure_dfma_peak.argtypes = [i32, ctypes.POINTER(ctypes.c_double)]
        L.ptfock_measure_dmma_peak.argtypes = [i32, ctypes.POINTER(ctypes.c_double)]
        L.ptfock_measure_copy_bandwidth.argtypes = [i32, ctypes.c_uint64, i32, ctypes.POINTER(ctypes.c_double)]
        L.ptfock_overlap.argtypes = [vp, vp, i32, vp, i32, vp, vp]
        L.ptfock_rotate.argtypes = [vp, vp, i32, vp, i32, vp, vp]
        L.ptfock_residual.argtypes = [vp, vp, vp, vp, i32, ctypes.c_double, vp, vp]
        L.ptfock_density.argtypes = [vp, vp, i32, vp, vp]
        L.ptfock_orthonormalize.argtypes = [vp, vp, i32, vp]
        L.ptfock_hloc_apply.argtypes = [vp, vp, vp, i32, vp, vp]
        L.ptfock_axpby.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
        L.ptfock_banddot.argtypes = [vp, vp, vp, i32, vp, vp]
        L.ptfock_banddot_many.argtypes = [vp, vp, ctypes.POINTER(vp), i32, i32, vp, vp]
        L.ptfock_vloc_update.argtypes = [vp, vp, ctypes.c_double, vp, vp, vp]
        L.ptfock_density_change.argtypes = [vp, vp, vp, ctypes.POINTER(ctypes.c_double), vp]
        L.ptfock_banddot_static.argtypes = [i32, ctypes.c_int64, ctypes.c_double, vp, vp, i32, vp, vp]
        for name in EXPORTS:
            if name != "ptfock_strerror":
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        L = lib()
        msg = L.ptfock_strerror(rc).decode()
        if rc == -6:
            msg += f" [cudaError {L.ptfock_last_cuda_error()}]"
        raise PtfockError(rc, f"{what}: {msg}")


def _dev_ptr(t, what: str, device_index: int):
    import torch
    if t is None:
        return ctypes.c_void_p(0)
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise TypeError(f"{what} must be a contiguous complex128 CUDA tensor")
    if t.device.index != device_index:
        raise ValueError(f"{what} is on {t.device}, the plan is on cuda:{device_index}")
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(t, what: str):
    import torch
    if t is None:
        return ctypes.c_void_p(0)
    if not (isinstance(t, torch.Tensor) and (not t.is_cuda) and t.dtype == torch.complex128 and t.is_contiguous()):
        raise TypeError(f"{what} must be a contiguous complex128 CPU tensor")
    return ctypes.c_void_p(t.data_ptr())


def _stream(device_index: int):
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream(device_index).cuda_stream)


class Plan:
    """ptfock_create / ptfock_destroy.  ``cell``: 9 doubles (rows = lattice vectors, bohr)."""

    def __init__(self, cell, n, n_occ: int, max_targets: int | None = None, kernel: int = KERNEL_HSE,
                 omega: float = 0.106, alpha: float = 1.0, device: int = 0, block_i: int = 0, block_j: int = 0,
                 workspace_bytes: int = 0, flags: int = 0):
        d = Desc()
        cell = [float(x) for x in cell]
        if len(cell) != 9 or len(n) != 3:
            raise ValueError("cell needs 9 numbers and n needs 3")
        d.cell = (ctypes.c_double * 9)(*cell)
        d.n = (ctypes.c_int32 * 3)(*[int(x) for x in n])
        d.n_occ = int(n_occ)
        d.max_targets = int(n_occ if max_targets is None else max_targets)
        d.kernel, d.omega, d.alpha, d.device = int(kernel), float(omega), float(alpha), int(device)
        d.block_i, d.block_j, d.workspace_bytes = int(block_i), int(block_j), int(workspace_bytes)
        d.flags = int(flags)
        self._h = ctypes.c_void_p(0)
        self.n = tuple(int(x) for x in n)
        self.N = self.n[0] * self.n[1] * self.n[2]
        self.n_occ = d.n_occ
        self.device = d.device
        _check(lib().ptfock_create(ctypes.byref(d), ctypes.byref(self._h)), "ptfock_create")

    def _grids(self, t, what):
        if t.numel() % self.N:
            raise ValueError(f"{what} does not hold whole grids")
        return t.numel() // self.N

    def apply(self, phi, psi=None, out=None, self_offset: int = 0, n_targets: int | None = None):
        """out[j] = V_X[phi] psi_j.  psi None: targets are phi[self_offset : self_offset + n_targets]."""
        import torch
        if self._grids(phi, "phi") != self.n_occ:
            raise ValueError("phi must hold n_occ grids")
        if psi is not None:
            nt = self._grids(psi, "psi")
            if n_targets is not None and n_targets != nt:
                raise ValueError("n_targets disagrees with psi")
        else:
            nt = self.n_occ - self_offset if n_targets is None else n_targets
        if out is None:
            out = torch.empty((nt,) + self.n, dtype=torch.complex128, device=phi.device)
        elif self._grids(out, "out") < nt:
            raise ValueError("out is too small")
        _check(lib().ptfock_apply(self._h, _dev_ptr(phi, "phi", self.device), _dev_ptr(psi, "psi", self.device),
                                  int(self_offset), int(nt), _dev_ptr(out, "out", self.device), _stream(self.device)),
               "ptfock_apply")
        return out

    def exchange_energy(self, phi, psi=None, vx_psi=None, self_offset: int = 0, n_targets: int | None = None) -> float:
        if psi is not None:
            nt = self._grids(psi, "psi")
        else:
            nt = self.n_occ - self_offset if n_targets is None else n_targets
        e = ctypes.c_double(0.0)
        _check(lib().ptfock_exchange_energy(self._h, _dev_ptr(phi, "phi", self.device),
                                            _dev_ptr(psi, "psi", self.device), int(self_offset), int(nt),
                                            _dev_ptr(vx_psi, "vx_psi", self.device), ctypes.byref(e),
                                            _stream(self.device)), "ptfock_exchange_energy")
        return e.value

    def apply_host(self, phi, psi=None, out=None, self_offset: int = 0, n_targets: int | None = None):
        """Host-buffer variant (ptfock_apply_host): CPU tensors in, CPU tensor out, copies inside the call."""
        import torch
        if psi is not None:
            nt = self._grids(psi, "psi")
        else:
            nt = self.n_occ - self_offset if n_targets is None else n_targets
        if out is None:
            out = torch.empty((nt,) + self.n, dtype=torch.complex128)
        _check(lib().ptfock_apply_host(self._h, _host_ptr(phi, "phi"), _host_ptr(psi, "psi"), int(self_offset),
                                       int(nt), _host_ptr(out, "out"), _stream(self.device)), "ptfock_apply_host")
        return out

    def debug_pair(self, phi_i, psi_j):
        import torch
        w = torch.empty(self.n, dtype=torch.complex128, device=phi_i.device)
        _check(lib().ptfock_debug_pair(self._h, _dev_ptr(phi_i, "phi_i", self.device),
                                       _dev_ptr(psi_j, "psi_j", self.device), _dev_ptr(w, "w", self.device),
                                       _stream(self.device)), "ptfock_debug_pair")
        return w

    # ---- dense-algebra neighbours (Alg. 3, Sec. 3.4) ----------------------------------------------------
    def _mat_ptr(self, t, what):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
            raise TypeError(f"{what} must be a contiguous complex128 CUDA tensor")
        if t.device.index != self.device:
            raise ValueError(f"{what} is on {t.device}, the plan is on cuda:{self.device}")
        return ctypes.c_void_p(t.data_ptr())

    def overlap(self, a, b, out=None):
        """S[m, n] = (Omega/N) sum_r conj(a_m(r)) b_n(r)."""
        import torch
        n_a, n_b = self._grids(a, "a"), self._grids(b, "b")
        if out is None:
            out = torch.empty((n_a, n_b), dtype=torch.complex128, device=a.device)
        _check(lib().ptfock_overlap(self._h, _dev_ptr(a, "a", self.device), n_a, _dev_ptr(b, "b", self.device), n_b,
                                    self._mat_ptr(out, "out"), _stream(self.device)), "ptfock_overlap")
        return out

    def rotate(self, a, s, out=None):
        """out_n = sum_m a_m S[m, n]."""
        import torch
        n_a = self._grids(a, "a")
        if s.shape[0] != n_a:
            raise ValueError("S must be [n_a, n_out]")
        if out is None:
            out = torch.empty((s.shape[1],) + self.n, dtype=torch.complex128, device=a.device)
        _check(lib().ptfock_rotate(self._h, _dev_ptr(a, "a", self.device), n_a, self._mat_ptr(s, "s"), int(s.shape[1]),
                                   _dev_ptr(out, "out", self.device), _stream(self.device)), "ptfock_rotate")
        return out

    def residual(self, psi, hpsi, dt: float = 0.0, psi_half=None, out=None):
        """psi_half None: H psi - psi (psi^* H psi); else psi + (i dt/2)(H psi - psi (psi^* H psi)) - psi_half."""
        import torch
        n = self._grids(psi, "psi")
        if out is None:
            out = torch.empty_like(psi)
        _check(lib().ptfock_residual(self._h, _dev_ptr(psi, "psi", self.device), _dev_ptr(hpsi, "hpsi", self.device),
                                     _dev_ptr(psi_half, "psi_half", self.device), n, float(dt),
                                     _dev_ptr(out, "out", self.device), _stream(self.device)), "ptfock_residual")
        return out

    def density(self, psi, out=None):
        import torch
        n = self._grids(psi, "psi")
        if out is None:
            out = torch.empty(self.n, dtype=torch.float64, device=psi.device)
        _check(lib().ptfock_density(self._h, _dev_ptr(psi, "psi", self.device), n, ctypes.c_void_p(out.data_ptr()),
                                    _stream(self.device)), "ptfock_density")
        return out

    def orthonormalize(self, psi):
        """In place: psi <- psi L^{-H}, L L^H = psi^* psi."""
        n = self._grids(psi, "psi")
        _check(lib().ptfock_orthonormalize(self._h, _dev_ptr(psi, "psi", self.device), n, _stream(self.device)),
               "ptfock_orthonormalize")
        return psi

    # ---- PT-CN step helpers (Alg. 1) -------------------------------------------------------------------
    def hloc_apply(self, psi, vloc=None, out=None):
        """out_j = -1/2 Laplacian psi_j + vloc psi_j (plan created with KERNEL_KINETIC, n_occ = 1)."""
        import torch
        n = self._grids(psi, "psi")
        if out is None:
            out = torch.empty_like(psi)
        vp_ = ctypes.c_void_p(0)
        if vloc is not None:
            if not (vloc.is_cuda and vloc.dtype == torch.float64 and vloc.is_contiguous() and vloc.numel() == self.N):
                raise TypeError("vloc must be a contiguous float64 CUDA tensor of one grid")
            vp_ = ctypes.c_void_p(vloc.data_ptr())
        _check(lib().ptfock_hloc_apply(self._h, vp_, _dev_ptr(psi, "psi", self.device), n,
                                       _dev_ptr(out, "out", self.device), _stream(self.device)), "ptfock_hloc_apply")
        return out

    def axpby(self, a, x, b=None, y=None, out=None):
        """out_j = a_j x_j + b_j y_j; a, b: scalars or per-orbital sequences of complex numbers."""
        import numpy as np
        import torch
        n = self._grids(x, "x")
        av = np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.complex128), (n,)))
        bv = None if y is None else np.ascontiguousarray(np.broadcast_to(np.asarray(b, dtype=np.complex128), (n,)))
        if out is None:
            out = torch.empty_like(x)
        _check(lib().ptfock_axpby(self._h, n, ctypes.c_void_p(av.ctypes.data), _dev_ptr(x, "x", self.device),
                                  ctypes.c_void_p(0 if bv is None else bv.ctypes.data), _dev_ptr(y, "y", self.device),
                                  _dev_ptr(out, "out", self.device), _stream(self.device)), "ptfock_axpby")
        return out

    def banddot(self, a, b):
        """numpy array of (a_j, b_j), j < n."""
        import numpy as np
        n = self._grids(a, "a")
        res = np.empty(n, dtype=np.complex128)
        _check(lib().ptfock_banddot(self._h, _dev_ptr(a, "a", self.device), _dev_ptr(b, "b", self.device), n,
                                    ctypes.c_void_p(res.ctypes.data), _stream(self.device)), "ptfock_banddot")
        return res

    def banddot_many(self, a, b_sets):
        """numpy array [len(b_sets), n] of (a_j, b^k_j) in one call (one synchronisation)."""
        import numpy as np
        n = self._grids(a, "a")
        ptrs = (ctypes.c_void_p * len(b_sets))(*[_dev_ptr(b, "b_sets[k]", self.device).value for b in b_sets])
        for b in b_sets:
            if self._grids(b, "b_sets[k]") != n:
                raise ValueError("every set must hold as many orbitals as a")
        res = np.empty((len(b_sets), n), dtype=np.complex128)
        _check(lib().ptfock_banddot_many(self._h, _dev_ptr(a, "a", self.device), ptrs, len(b_sets), n,
                                         ctypes.c_void_p(res.ctypes.data), _stream(self.device)), "ptfock_banddot_many")
        return res

    def _real_grid(self, t, what):
        import torch
        if t is None:
            return ctypes.c_void_p(0)
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.numel() == self.N and t.device.index == self.device):
            raise TypeError(f"{what} must be a contiguous float64 CUDA tensor of one grid on cuda:{self.device}")
        return ctypes.c_void_p(t.data_ptr())

    def vloc_update(self, v_ext, g: float, rho, out=None):
        """v_ext + g rho on the device (Alg. 1 line 5)."""
        import torch
        if out is None:
            out = torch.empty_like(rho)
        _check(lib().ptfock_vloc_update(self._h, self._real_grid(v_ext, "v_ext"), float(g), self._real_grid(rho, "rho"),
                                        self._real_grid(out, "out"), _stream(self.device)), "ptfock_vloc_update")
        return out

    def density_change(self, rho_a, rho_b) -> float:
        """(Omega/N) sum_r |rho_a - rho_b| (Alg. 1 line 9)."""
        v = ctypes.c_double(0.0)
        _check(lib().ptfock_density_change(self._h, self._real_grid(rho_a, "rho_a"), self._real_grid(rho_b, "rho_b"),
                                           ctypes.byref(v), _stream(self.device)), "ptfock_density_change")
        return v.value

    def info(self) -> dict:
        a = (ctypes.c_int64 * 8)()
        _check(lib().ptfock_plan_info(self._h, a), "ptfock_plan_info")
        return {"block_i": a[0], "block_j": a[1], "scratch_bytes": a[2], "last_launches": a[3], "last_pairs": a[4],
                "last_symmetric": a[5], "total_launches": a[6], "pass8": a[7] & 15, "slots": 1 + ((a[7] >> 4) & 1)}

    def set_profiling(self, on: bool):
        _check(lib().ptfock_set_profiling(self._h, 1 if on else 0), "ptfock_set_profiling")

    def get_profile(self, reset: bool = True) -> dict:
        ms = (ctypes.c_double * 3)()
        cnt = (ctypes.c_int64 * 3)()
        _check(lib().ptfock_get_profile(self._h, ms, cnt, 1 if reset else 0), "ptfock_get_profile")
        return {"ms": [ms[0], ms[1], ms[2]], "launches": [cnt[0], cnt[1], cnt[2]]}

    def destroy(self):
        if self._h:
            lib().ptfock_destroy(self._h)
            self._h = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()


def banddot_static(a, b, weight: float, out=None):
    """out[j] = weight * sum_r conj(a_j(r)) b_j(r) through ptfock_banddot_static: no plan, and no allocation inside the
    library (its partial sums live in a fixed 4 MiB array built into libptfock.so), for host codes that own all device
    memory themselves or cannot afford cudaMalloc's device-wide stall.  ``a``, ``b``: [n, ...] complex128 CUDA tensors,
    n <= STATIC_MAX_BANDS; ``out``: optional complex128 CUDA tensor of n numbers (pass it to keep torch from allocating
    too).  Asynchronous on torch's current stream; calls that may overlap on the GPU race on the shared array."""
    import torch
    if not (isinstance(a, torch.Tensor) and isinstance(b, torch.Tensor) and a.is_cuda and a.dim() >= 2 and a.shape == b.shape):
        raise TypeError("a and b must be CUDA tensors of the same shape [n, ...]")
    dev = a.device.index
    n = a.shape[0]
    if out is None:
        out = torch.empty(n, dtype=torch.complex128, device=a.device)
    elif out.numel() != n:
        raise ValueError("out must hold n complex numbers")
    _check(lib().ptfock_banddot_static(dev, a[0].numel(), float(weight), _dev_ptr(a, "a", dev), _dev_ptr(b, "b", dev), n,
                                       _dev_ptr(out, "out", dev), _stream(dev)), "ptfock_banddot_static")
    return out


def measure_fp64_peak(device: int = 0) -> float:
    """Sustained DFMA rate of the device in TFLOP/s (ptfock_measure_dfma_peak)."""
    v = ctypes.c_double(0.0)
    _check(lib().ptfock_measure_dfma_peak(int(device), ctypes.byref(v)), "ptfock_measure_dfma_peak")
    return v.value


def measure_fp64_tensor_peak(device: int = 0) -> float:
    """Sustained FP64 tensor-core (DMMA) rate of the device in TFLOP/s (ptfock_measure_dmma_peak)."""
    v = ctypes.c_double(0.0)
    _check(lib().ptfock_measure_dmma_peak(int(device), ctypes.byref(v)), "ptfock_measure_dmma_peak")
    return v.value


def measure_copy_bandwidth(nbytes: int, reps: int = 20, device: int = 0) -> float:
    """Device-to-device copy rate in GB/s (read + write) for a source of ``nbytes`` (ptfock_measure_copy_bandwidth)."""
    v = ctypes.c_double(0.0)
    _check(lib().ptfock_measure_copy_bandwidth(int(device), int(nbytes), int(reps), ctypes.byref(v)),
           "ptfock_measure_copy_bandwidth")
    return v.value


def plan_for(cfg, device: int = 0, max_targets: int | None = None, **kw) -> Plan:
    """Plan for a ``synth.Config``."""
    mt = max_targets if max_targets is not None else (cfg.j_block if cfg.j_block else cfg.n_occ)
    return Plan(cfg.cell, cfg.n, cfg.n_occ, mt, cfg.kernel, cfg.omega, cfg.alpha, device, **kw)
