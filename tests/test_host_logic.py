"""CPU-only checks: the C-ABI library loads and exports what include/ptfock.h declares, it refuses to
run without a B200 (no CPU fallback), and the N > 1 replica bookkeeping works (gloo, world_size 2)."""
import ctypes
import os
import re
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_1905_01348_b200 import binding
    binding.build_library()
    return binding


def test_every_declared_symbol_is_exported(built_lib):
    hdr = open(os.path.join(ROOT, "include", "ptfock.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ptfock_[a-z_]+)\s*\(", hdr))
    assert {"ptfock_create", "ptfock_apply", "ptfock_exchange_energy", "ptfock_destroy"} <= declared
    L = built_lib.lib()
    for name in declared:
        assert hasattr(L, name), f"{name} declared in ptfock.h but not exported"
    assert declared == set(built_lib.EXPORTS)


def test_library_is_sm100a_only(built_lib):
    out = subprocess.run(["cuobjdump", "--list-elf", built_lib.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_strerror_and_desc_layout(built_lib):
    L = built_lib.lib()
    assert L.ptfock_strerror(0) == b"ok"
    assert b"no CPU fallback" in L.ptfock_strerror(-3)
    assert L.ptfock_destroy(None) == 0
    # ptfock_desc: 9 doubles, 3+1+1+1 int32, 2 doubles, 3 int32 (+pad), uint64, uint32 (+pad)
    assert ctypes.sizeof(built_lib.Desc) == 72 + 24 + 16 + 16 + 8 + 8
    assert b"slab shapes" in L.ptfock_strerror(-2)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback(built_lib):
    """Without a CUDA device the product path must fail loudly, not compute on the host."""
    with pytest.raises(built_lib.PtfockError) as ei:
        built_lib.Plan([10.0, 0, 0, 0, 10.0, 0, 0, 0, 10.0], (16, 16, 16), 2)
    assert ei.value.code in (-3, -6)
    with pytest.raises(TypeError):
        built_lib._dev_ptr(torch.zeros(4, dtype=torch.complex128), "phi", 0)


def test_invalid_descriptors_rejected_before_touching_the_device(built_lib):
    for kw, code in [(dict(n=(16, 20, 16)), -2), (dict(n=(16, 16, 16), kernel=7), -1),
                     (dict(n=(16, 16, 16), omega=0.0), -1), (dict(n=(16, 16, 16), n_occ=0), -1),
                     (dict(n=(64, 128, 128)), -2)]:
        args = dict(cell=[10.0, 0, 0, 0, 10.0, 0, 0, 0, 10.0], n=(16, 16, 16), n_occ=2)
        args.update(kw)
        with pytest.raises(built_lib.PtfockError) as ei:
            built_lib.Plan(**args)
        assert ei.value.code == code, kw


def test_missing_library_raises(tmp_path):
    code = ("import os, sys; sys.path.insert(0, %r); os.environ['PTFOCK_LIB'] = %r\n"
            "from paper_1905_01348_b200 import binding\n"
            "try:\n    binding.lib()\nexcept FileNotFoundError as e:\n    print('RAISED'); sys.exit(0)\nsys.exit(1)\n"
            % (ROOT, str(tmp_path / "nope.so")))
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True)
    assert r.returncode == 0 and "RAISED" in r.stdout


def _replica_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1905_01348_b200 import harness
    harness.barrier()
    secs = 2.0 if rank == 0 else 4.0                     # rank 1 is the slow replica
    q.put((rank, harness.max_over_ranks(secs), harness.replica_throughput(1000.0, secs)))
    dist.destroy_process_group()


def test_replicas_only_bookkeeping_gloo_world2():
    """N > 1 = independent replicas: value = N * units / max over ranks of the device time."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_replica_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, thr in res:
        assert mx == 4.0 and thr == pytest.approx(2 * 1000.0 / 4.0)


def _gather_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1905_01348_b200 import harness
    n_total, shape = 5, (2, 3, 2)
    g = torch.Generator().manual_seed(7)
    full = torch.complex(torch.randn((n_total,) + shape, generator=g, dtype=torch.float64),
                         torch.randn((n_total,) + shape, generator=g, dtype=torch.float64))
    lo, hi = harness.shard_range(n_total, world, rank)
    got64 = harness.allgather_orbitals(full[lo:hi].clone(), n_total)
    got32 = harness.allgather_orbitals(full[lo:hi].clone(), n_total, wire="fp32")
    q.put((rank, (lo, hi), bool(torch.equal(got64, full)), float((got32 - full).abs().max() / full.abs().max())))
    dist.destroy_process_group()


def test_j_sharding_allgather_gloo_world2():
    """N > 1 with Phi distributed: uneven blocks (3 + 2 of 5 orbitals) all-gathered bit-exactly in fp64; the fp32 wire
    format of PAPER.md:154 costs at most single-precision rounding."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gather_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [(0, 3), (3, 5)]
    for _, _, exact, err32 in res:
        assert exact and 0.0 < err32 < 2.0 ** -23


def test_shard_range_partitions():
    from paper_1905_01348_b200 import harness
    for n, world in ((3072, 8), (5, 2), (7, 3), (2, 4)):
        parts = [harness.shard_range(n, world, r) for r in range(world)]
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(parts[k][1] == parts[k + 1][0] for k in range(world - 1))
        sizes = [hi - lo for lo, hi in parts]
        assert max(sizes) - min(sizes) <= 1


def test_harness_single_process_identity():
    from paper_1905_01348_b200 import harness
    assert harness.max_over_ranks(3.5) == 3.5
    assert harness.replica_throughput(10.0, 2.0) == 5.0


def test_bench_reference_arm_runs_on_cpu():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "Si8",
                        "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "pair-FFTs/s"
