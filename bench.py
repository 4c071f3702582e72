#!/usr/bin/env python
"""Benchmark harness: Fock exchange pair-FFTs/s in fp64 on B200 (BASELINE.json ``metric``).

One "step" = one whole pass of the hot path over one batch of synthetic input:
  Si512  : ptfock_apply of 1024 targets against 1024 orbitals (1 048 576 pair-solves), 64^3 grid (default);
  Si1536 : one streamed j-block of 96 targets against 3072 orbitals (294 912 pair-solves), 128x128x48;
  Si8 / Si64 / Si216 : the full Psi = Phi application (pair-symmetric schedule).
``value`` counts EFFECTIVE pair-solves N_i * N_j per second (equal to the executed count for Si512/Si1536).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config Si512] [--impl ours|reference]

N > 1 (torchrun): the path is single-GPU by construction (BASELINE.json north_star), so ranks are independent
replicas ("replicas only"); value = pairs of all ranks / max-over-ranks time.
``--impl reference`` times the CPU oracle (oracle/ptfock_ref.c) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Fock exchange pair-FFTs/s (fp64, 1 B200) and % of HBM roofline"
UNIT = "pair-FFTs/s"
HBM_FALLBACK_GBS = 6650.0       # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# BASELINE.md holds a paper number only for the paper's own workload (3072 orbitals on the 60 x 90 x 120 grid):
# 2881 pair-solves/s per V100, computation only (derived from PAPER.md:299, Table 1, 36 GPUs).  Another machine's: context.
PAPER_PAIRS_PER_S = {"Si1536p": 2881.0}


def load_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [s for s, p in zip(sm, pw) if p >= 0.5 * max(pw)] or sm
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(cfg):
    """(n_i, n_j, description) of one step."""
    if cfg.j_block:
        return cfg.n_occ, cfg.j_block, f"{cfg.name}: one j-block of {cfg.j_block} targets x {cfg.n_occ} orbitals"
    return cfg.n_occ, cfg.n_occ, f"{cfg.name}: {cfg.n_occ} targets x {cfg.n_occ} orbitals"


def cpu_sample(cfg, n_threads: int):
    """Bounded oracle sample: (n_cols, n_i) sized for ~10-30 s of CPU work at this grid."""
    rate_per_core = {4096: 1500.0, 32768: 170.0, 110592: 45.0, 262144: 17.0, 786432: 5.0}.get(cfg.N, 3e6 / cfg.N)
    n_cols = min(n_threads, workload(cfg)[1])
    n_i = int(max(1, min(cfg.n_occ, 15.0 * rate_per_core)))
    return n_cols, n_i


def run_oracle_sample(cfg, phi_np, psi_np, n_cols, n_i):
    import numpy as np
    import oracle
    cols = list(range(n_cols))
    phi_s = np.ascontiguousarray(phi_np[:n_i])
    tgt = phi_np if psi_np is None else psi_np
    tgt_s = np.ascontiguousarray(tgt[:n_cols])
    t0 = time.perf_counter()
    oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi_s, tgt_s, cols)
    dt = time.perf_counter() - t0
    return n_cols * n_i, dt


def reference_arm(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; each step = one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    import torch
    from paper_1905_01348_b200 import synth
    oracle.build()
    cores = oracle.num_threads()
    n_cols, n_i = cpu_sample(cfg, cores)
    n_orb = max(n_i, n_cols)
    phi = synth.orbitals(cfg, cfg.seed_phi, n_orb, "cpu").numpy()
    psi = synth.orbitals(cfg, cfg.seed_psi, n_cols, "cpu").numpy() if cfg.separate_psi else None
    for _ in range(args.warmup):
        run_oracle_sample(cfg, phi, psi, n_cols, min(n_i, 8))
    pairs, secs = 0, 0.0
    for _ in range(args.steps):
        p, dt = run_oracle_sample(cfg, phi, psi, n_cols, n_i)
        pairs += p
        secs += dt
    value = pairs / secs
    sample = f"{n_cols} target columns x first {n_i} orbitals of {cfg.name} ({n_cols * n_i} pair-solves) per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload(cfg)[2], "grid": list(cfg.n), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def measure(cfg, args, dev, local, rank, world, steps, warmup, do_e2e, do_cpu, check=False):
    """Times `steps` steps of cfg's workload on this rank; returns the pieces of the JSON line."""
    import torch
    from paper_1905_01348_b200 import binding, harness, synth

    def barrier():
        harness.barrier(dev)

    n_i, n_j, wl = workload(cfg)
    if args.full_application and cfg.j_block:
        # the whole application V_X[Phi] Phi in one call: Phi AND out resident (2 x 38.65 GB at Si1536), pair-symmetric
        # schedule over all block pairs (half the pair-solves of 32 streamed j-blocks)
        n_j, wl = cfg.n_occ, f"{cfg.name}: whole application, {cfg.n_occ} targets x {cfg.n_occ} orbitals (Psi = Phi, symmetric schedule)"
    if args.targets:
        n_j = min(n_j, args.targets)
        wl += f" (slice: first {n_j} targets)"
    phi = synth.orbitals(cfg, cfg.seed_phi, cfg.n_occ, dev)
    psi = synth.orbitals(cfg, cfg.seed_psi, n_j, dev) if cfg.separate_psi else None
    out = torch.empty((n_j,) + tuple(cfg.n), dtype=torch.complex128, device=dev)
    plan = binding.plan_for(cfg, device=local, max_targets=n_j, block_i=args.block_i, block_j=args.block_j,
                            workspace_bytes=int(args.workspace_gb * (1 << 30)), flags=args.flags)

    def step():
        if args.full_application and cfg.j_block:
            plan.apply(phi, out=out)
        elif cfg.j_block or (args.targets and psi is None):
            plan.apply(phi, None, out=out, self_offset=0, n_targets=n_j)
        else:
            plan.apply(phi, psi, out=out)

    for _ in range(warmup):
        step()
    barrier()
    info0 = plan.info()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):                      # the headline region: no per-launch events inside
        step()
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = e0.elapsed_time(e1)
    info1 = plan.info()
    ms_total = harness.max_over_ranks(ms_total, dev)
    ms_step = ms_total / steps
    pairs_eff = n_i * n_j
    pairs_exec = info1["last_pairs"]
    value = world * pairs_eff / (ms_step * 1e-3)
    launches = info1["total_launches"] - info0["total_launches"]

    # ---- per-pass timing: a separate step with every launch bracketed by CUDA events on the launching stream ----
    plan.set_profiling(True)
    plan.get_profile(reset=True)
    n_prof = max(1, min(2, steps))
    for _ in range(n_prof):
        step()
    prof = plan.get_profile(reset=True)
    plan.set_profiling(False)

    peak, peak_src = load_peak()
    N = cfg.N
    Ib, Jb = info1["block_i"], info1["block_j"]
    if info1.get("pass8") == 2:
        names = ["onchip16_apply (whole pair-solve on chip)", "(no pass B)", "onchip_reduce (sum of the i-chunks)"]
    elif info1.get("pass8"):
        names = ["p8_fwd (pass A)", "p8_mid (pass B)", "p8_inv_acc (pass C)"]
    else:
        names = ["slabx_fwd / slab_fwd (pass A)", "pencil_tma / pencil_mid (pass B)", "slabx_inv_acc / slab_inv_acc (pass C)"]
    # algorithmic bytes per executed pair-solve: A reads its share of phi / psi and writes the pair density; B reads
    # and writes it (v' amortised over the wave); C reads it, reads phi_i, and read-modify-writes out once per
    # (target, wave).  DESIGN.md 5.
    per_pair = [16.0 * N * (1.0 + 1.0 / Jb + 1.0 / Ib), 32.0 * N, 16.0 * N * (1.0 + 1.0 / Jb + 2.0 / Ib)]
    if info1.get("last_symmetric"):
        # pair-symmetric schedule: every executed pair density is read by two C launches (out_j, and out_i through conj)
        per_pair[2] *= 2.0
    if info1.get("pass8") == 2:
        # on chip: phi_i twice (product, final multiply; the second read hits L1/L2), psi_j and the partial sums once per
        # CTA; no pair-density traffic at all.  Per pair-solve at most 32 N + (16 N + 32 N) / (orbitals per CTA).
        per_pair = [32.0 * N + 48.0 * N * max(1, launches // max(1, steps) // 2) / max(1, n_i), 0.0, 0.0]
    tot_ms = max(1e-9, sum(prof["ms"]))
    pairs_prof = pairs_exec * n_prof
    per_kernel = {}
    for q in range(3):
        gbs = per_pair[q] * pairs_prof / max(1e-9, prof["ms"][q] * 1e-3) / 1e9
        per_kernel[names[q]] = {"ms_per_step": prof["ms"][q] / n_prof, "share": prof["ms"][q] / tot_ms, "GB/s": gbs,
                                "frac": gbs / peak, "launches_per_step": prof["launches"][q] // n_prof,
                                "avg_launch_ms": prof["ms"][q] / max(1, prof["launches"][q]),
                                "bytes_per_pair_solve": per_pair[q]}
    k = max(range(3), key=lambda q: prof["ms"][q])
    rate = pairs_exec / (ms_step * 1e-3)
    frac72 = rate / (peak * 1e9 / (72.0 * N))
    roofline = {"bound": "hbm", "unit": "GB/s", "peak": peak, "peak_source": peak_src,
                # the path: SURVEY.md 8(d)'s contract roofline, 72 N bytes per executed pair-solve
                "achieved": 72.0 * N * rate / 1e9, "frac": frac72, "survey_72N_frac": frac72,
                "executed_pair_solves_per_s": rate,      # `value` is the EFFECTIVE rate n_i * n_j / time
                "bytes_model": "72 N per executed pair-solve (SURVEY.md 8(d) B_3pass); own model below",
                "own_bytes_per_pair_solve": sum(per_pair), "own_bytes_frac": rate / (peak * 1e9 / sum(per_pair)),
                "frac_note": "frac uses the 72 N contract model on the timed region's rate; this build moves own_bytes_per_pair_solve "
                             "(< 72 N), so own_bytes_frac is the fraction of the peak its own traffic reaches",
                "worst_pass_frac": min(v["frac"] for v in per_kernel.values()),
                "dominant_kernel": names[k], "per_kernel": per_kernel,
                "per_kernel_schedule": "separate profiling step after the timed region: single stream, every launch bracketed by "
                                       "CUDA events on the launching stream (the timed region itself runs two waves on two "
                                       "streams with no per-launch events)",
                "traffic": None, "traffic_source": None}
    try:
        import math
        p64 = binding.measure_fp64_peak(local)
        flops = 10.0 * N * math.log2(N) + 16.0 * N
        roofline["fp64"] = {"peak_tflops": p64, "peak_source": "measured live (ptfock_measure_dfma_peak, DFMA loop)",
                            "nominal_flops_per_pair_solve": flops, "achieved_tflops": rate * flops / 1e12,
                            "frac": rate * flops / 1e12 / p64, "pairs_per_s_at_peak": p64 * 1e12 / flops}
    except Exception as e:                      # a measurement aid only: never fail the bench on it
        roofline["fp64"] = {"error": str(e)}
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            roofline["traffic"] = json.load(f).get(cfg.name, {}).get(names[k].split(" ")[0])
        if roofline["traffic"] is not None:
            roofline["traffic_source"] = ("profiles/traffic.json: dram bytes per launch from an ncu --set full capture of an "
                                          "earlier run of the same kernel, not measured in this run")
    except Exception:
        pass

    # ---- end to end through the host-buffer entry point (pinned host memory, copies timed) -----------
    e2e = None
    if do_e2e:
        h_phi = torch.empty(phi.shape, dtype=phi.dtype, pin_memory=True).copy_(phi)
        h_psi = torch.empty(psi.shape, dtype=psi.dtype, pin_memory=True).copy_(psi) if psi is not None else None
        h_out = torch.empty(out.shape, dtype=out.dtype, pin_memory=True)
        plan.apply_host(h_phi, h_psi, out=h_out, n_targets=n_j)                    # warm-up (allocates staging)
        n_e2e = max(1, min(steps, 2))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            plan.apply_host(h_phi, h_psi, out=h_out, n_targets=n_j)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = harness.max_over_ranks(dt, dev)
        gb = 16 * N
        e2e = {"value": world * pairs_eff * n_e2e / dt, "unit": UNIT,
               "h2d_bytes_per_step": gb * (cfg.n_occ + (n_j if psi is not None else 0)), "d2h_bytes_per_step": gb * n_j,
               "steps": n_e2e, "api": "ptfock_apply_host (pinned host buffers)"}
        del h_phi, h_psi, h_out

    # ---- parity on sampled columns + CPU baseline (rank 0, N = 1 only) ------------------------------
    cpu_baseline, parity = None, None
    if rank == 0 and world == 1 and do_cpu:
        import numpy as np
        import oracle
        oracle.build()
        cores = oracle.num_threads()
        n_cols, n_is = cpu_sample(cfg, cores)
        phi_np = phi[:max(n_is, n_cols)].cpu().numpy()
        psi_np = psi[:n_cols].cpu().numpy() if psi is not None else None
        p, dt = run_oracle_sample(cfg, phi_np, psi_np, n_cols, n_is)
        cpu_baseline = {"value": p / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{n_cols} target columns x first {n_is} orbitals of {cfg.name} ({p} pair-solves, {dt:.1f} s)"}
        if check:
            cols = sorted({0, n_j // 2, n_j - 1})
            tgt = phi if psi is None else psi
            ref = oracle.apply(cfg.cell, cfg.n, cfg.kernel, cfg.omega, cfg.alpha, phi.cpu().numpy(),
                               tgt[:n_j].cpu().numpy(), cols)
            got = out[cols].cpu().numpy()
            parity = {"columns": cols, "max_rel_err": float(np.abs(got - ref).max() / np.abs(ref).max())}

    config = {"workload": wl, "grid": list(cfg.n), "n_i": n_i, "n_j": n_j,
              "kernel": "HSE" if cfg.kernel == 1 else "Coulomb",
              "pair_solves_executed_per_step": pairs_exec, "symmetric_schedule": bool(info1["last_symmetric"]),
              "block_i": Ib, "block_j": Jb, "scratch_bytes": info1["scratch_bytes"],
              "kernels": {0: "three-stage slab passes + pencil pass", 1: "pass8 (two-stage slab passes + two-stage pencil pass)",
                          2: "onchip16 (whole pair-solve in one CTA, no scratch)"}[int(info1.get("pass8", 0))],
              "l2": f"inputs + scratch per step = {(16 * N * (n_i + 2 * n_j) + info1['scratch_bytes']) / 1e9:.2f} GB"
                    " (larger than the 126 MB L2; no explicit flush)",
              "parallelism": "replicas only" if world > 1 else "single GPU"}
    plan.destroy()
    del phi, psi, out
    torch.cuda.empty_cache()
    return {"value": value, "ms_per_step": ms_step, "steps": steps, "warmup": warmup, "config": config, "clocks": clocks,
            "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline, "parity": parity,
            "vs_baseline": (value / world / PAPER_PAIRS_PER_S[cfg.name]) if cfg.name in PAPER_PAIRS_PER_S else None}


def dense_leg(cfg, args, dev, local, emit=True):
    """--leg dense: the dense-algebra neighbours (Alg. 3, Sec. 3.4) at cfg's sizes, each
    timed alone with CUDA events on the launching stream; roofline = the plain FP64 pipe (measured live) for the
    contractions, HBM for the density."""
    import torch
    from paper_1905_01348_b200 import binding, synth
    n = cfg.j_block * 8 if cfg.j_block else cfg.n_occ          # Si1536: 768 orbitals keep the run inside a minute
    psi = synth.orbitals(cfg, cfg.seed_phi, n, dev)
    g = torch.Generator(device="cpu").manual_seed(5)
    hpsi = psi * 0.5 + 0.1 * torch.roll(psi, 1, 0)
    half = torch.roll(psi, 2, 0).contiguous()
    N = cfg.N
    peak_hbm, _ = load_peak()
    p64 = binding.measure_fp64_tensor_peak(local)      # the contractions run on the FP64 tensor pipe (DMMA.8x8x4)
    p64_fma = binding.measure_fp64_peak(local)
    out = {}
    with binding.Plan(cfg.cell, cfg.n, n, n, cfg.kernel, cfg.omega, cfg.alpha, local) as plan:
        s = torch.empty((n, n), dtype=torch.complex128, device=dev)
        r = torch.empty_like(psi)
        rho = torch.empty(cfg.n, dtype=torch.float64, device=dev)
        mix = (psi + 0.05 * torch.roll(psi, 1, 0)).contiguous()
        work = mix.clone()

        def timed(fn, reps, setup=None):
            ts = []
            for k in range(reps + 1):
                if setup:
                    setup()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                fn()
                e1.record()
                torch.cuda.synchronize()
                if k:
                    ts.append(e0.elapsed_time(e1))
            return statistics.median(ts)

        legs = {
            "overlap (Alg. 3 line 2)": (lambda: plan.overlap(psi, hpsi, out=s), None, 8.0 * N * n * n, 32.0 * N * n),
            "residual R_f (Alg. 3 lines 2-5)": (lambda: plan.residual(psi, hpsi, dt=0.5, psi_half=half, out=r), None,
                                                16.0 * N * n * n, 80.0 * N * n),
            "density (Sec. 3.4)": (lambda: plan.density(psi, out=rho), None, 4.0 * N * n, 16.0 * N * n),
            "orthonormalize (Sec. 3.4: overlap + Cholesky + Trsm)": (lambda: plan.orthonormalize(work), lambda: work.copy_(mix),
                                                                    # Hermitian overlap on the lower tiles (4 N n^2 of the full
                                                                    # 8 N n^2) + triangular solve (4 N n^2) + Cholesky
                                                                    8.0 * N * n * n + 4.0 / 3.0 * n ** 3, 48.0 * N * n),
        }
        for name, (fn, setup, flops, byts) in legs.items():
            ms = timed(fn, args.steps, setup)
            tf, gbs = flops / (ms * 1e-3) / 1e12, byts / (ms * 1e-3) / 1e9
            bound = "hbm" if name.startswith("density") else "tensor"
            out[name] = {"ms": ms, "TFLOP/s": tf, "GB/s": gbs, "bound": bound,
                         "frac": gbs / peak_hbm if bound == "hbm" else tf / p64}
    line = {"metric": "dense-algebra neighbours of the Fock exchange path (fp64, 1 B200)", "unit": "ms per call",
            "config": {"workload": f"{cfg.name}: {n} orbitals on {'x'.join(map(str, cfg.n))}", "leg": "dense"},
            "dtype": "f64", "data": "synthetic", "steps": args.steps,
            "roofline": {"tensor_peak_tflops": p64, "tensor_peak_source": "measured live (ptfock_measure_dmma_peak: fp64 mma.sync m8n8k4)",
                         "fma_peak_tflops": p64_fma,
                         "hbm_peak_gbs": peak_hbm, "per_call": out}}
    if emit:
        print(json.dumps(line), flush=True)
    return line


def ptcn_leg(cfg, args, dev, local, emit=True):
    """--leg ptcn: whole PT-CN time steps (Algorithm 1: residual, Anderson-mixed fixed point, density,
    re-orthogonalisation) with the model Hamiltonian of DESIGN.md Q17 at cfg's grid and orbital count, sequenced over
    the C ABI by paper_1905_01348_b200/ptcn.py; wall time per step (host least-squares included) and the share of it
    spent applying the exchange operator."""
    import torch
    from paper_1905_01348_b200 import binding, ptcn, synth
    n_e = cfg.n_occ
    psi = synth.orbitals(cfg, cfg.seed_phi, n_e, dev)
    x = torch.meshgrid(*[torch.arange(k, dtype=torch.float64) / k for k in cfg.n], indexing="ij")
    v_ext = 0.2 * torch.cos(2 * math.pi * x[0]) + 0.1 * torch.sin(2 * math.pi * (x[1] + x[2]))
    # a.u. (9.7 as).  The paper steps 50 as with its production solver; the plain Anderson-mixed fixed
    # point of DESIGN.md Q18 has no preconditioner and converges for dt * (spectral width) / 2 up to ~10
    dt = 0.4
    steps_out = []
    with ptcn.PTCN(cfg.cell, cfg.n, n_e, kernel=cfg.kernel, omega=cfg.omega, alpha=0.25, v_ext=v_ext, g=0.5, device=local) as st:
        fock_ms = [0.0]
        apply0 = st.fock.apply

        def timed_apply(*a, **k):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            out = apply0(*a, **k)
            e1.record()
            fock_ms.append((e0, e1))
            return out
        st.fock.apply = timed_apply
        for k in range(args.steps + 1):             # first step: warm-up
            del fock_ms[:]
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            psi, info = st.step(psi, dt, tol=1e-8)
            torch.cuda.synchronize()
            wall = (time.perf_counter() - t0) * 1e3
            fock = sum(a.elapsed_time(b) for a, b in fock_ms)
            if k:
                steps_out.append({"ms": wall, "fock_exchange_ms": fock, "fock_applications": len(fock_ms),
                                  "scf_iterations": info["iterations"], "residual": info["residual"]})
    ms = statistics.median(s["ms"] for s in steps_out)
    line = {"metric": "PT-CN time step with a model Hamiltonian (fp64, 1 B200)", "unit": "ms per step", "value": ms,
            "config": {"workload": f"{cfg.name}: {n_e} orbitals on {'x'.join(map(str, cfg.n))}, dt = {dt} a.u., "
                                   "alpha = 0.25, residual < 1e-8", "leg": "ptcn"},
            "dtype": "f64", "data": "synthetic", "steps": args.steps, "higher_is_better": False,
            "fock_exchange_share": statistics.median(s["fock_exchange_ms"] / s["ms"] for s in steps_out),
            "per_step": steps_out}
    if emit:
        print(json.dumps(line), flush=True)
    return line


def cufft_leg(cfg, args, dev, local, emit=True, n_targets=None):
    """--leg cufft: SIDE COMPARISON only (north_star: "cuFFT-based runs may be timed only as a side comparison").  The paper's
    own method on this GPU (Sec. 3.2 items 1-2: batched cuFFT with custom kernels in the gaps), written
    with torch: batched torch.fft.fftn / ifftn (cuFFT) and element-wise torch ops for the pair product, the v(G) multiply,
    the phi_i multiply and the sum over i.  Nothing of this is linked into libptfock.so or used by the product path.
    Times a slice (all orbitals x n_targets targets) with CUDA events and compares the result with ptfock_apply."""
    import numpy as np
    import torch
    from paper_1905_01348_b200 import binding, synth
    n_i = cfg.n_occ
    n_j = n_targets or (cfg.j_block if cfg.j_block else min(cfg.n_occ, 64))
    phi = synth.orbitals(cfg, cfg.seed_phi, n_i, dev)
    psi = synth.orbitals(cfg, cfg.seed_psi, n_j, dev) if cfg.separate_psi else phi[:n_j].clone()
    # v(G) on torch's FFT frequency order; m_d in [-n_d/2, n_d/2), G = m B, B = 2 pi inv(A)^T (include/ptfock.h)
    a = np.asarray(cfg.cell, dtype=np.float64).reshape(3, 3)
    b = 2.0 * np.pi * np.linalg.inv(a).T
    ms = [np.where(np.arange(k) < (k + 1) // 2, np.arange(k), np.arange(k) - k) for k in cfg.n]
    m0, m1, m2 = np.meshgrid(*ms, indexing="ij")
    g = m0[..., None] * b[0] + m1[..., None] * b[1] + m2[..., None] * b[2]
    g2 = (g * g).sum(-1)
    with np.errstate(divide="ignore", invalid="ignore"):
        if cfg.kernel == 1:
            v = np.where(g2 > 0, 4 * np.pi / g2 * -np.expm1(-g2 / (4 * cfg.omega ** 2)), np.pi / cfg.omega ** 2)
        else:
            v = np.where(g2 > 0, 4 * np.pi / g2, 0.0)
    v_t = torch.from_numpy(-cfg.alpha * v).to(dev)
    N = cfg.N
    # batch: as many pair densities per cuFFT call as ~4 GB allow (input, output and cuFFT's workspace live together)
    ib = max(1, min(n_i, int((4 << 30) // (16 * N))))
    out = torch.zeros((n_j,) + tuple(cfg.n), dtype=torch.complex128, device=dev)

    def run():
        out.zero_()
        for j in range(n_j):
            for i0 in range(0, n_i, ib):
                p = phi[i0:i0 + ib]
                w = torch.fft.fftn(p.conj() * psi[j], dim=(-3, -2, -1))
                w *= v_t
                w = torch.fft.ifftn(w, dim=(-3, -2, -1))
                out[j] += (p * w).sum(0)
    run()                                                                # warm-up (plans, allocator)
    torch.cuda.synchronize()
    reps = max(1, min(3, args.steps))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        run()
    e1.record()
    torch.cuda.synchronize()
    ms_run = e0.elapsed_time(e1) / reps
    with binding.plan_for(cfg, device=local, max_targets=n_j) as plan:
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ours = plan.apply(phi, psi)
        t0.record()
        for _ in range(reps):
            plan.apply(phi, psi, out=ours)
        t1.record()
        torch.cuda.synchronize()
        ms_ours = t0.elapsed_time(t1) / reps
    diff = float((ours - out).abs().max() / ours.abs().max())
    pairs = n_i * n_j
    line = {"metric": "cuFFT side comparison: batched torch.fft + element-wise torch ops (the paper's method, PAPER.md:148-149)",
            "side_comparison": True, "unit": UNIT, "value": pairs / (ms_run * 1e-3), "ptfock_value_same_slice": pairs / (ms_ours * 1e-3),
            "ptfock_over_cufft": ms_run / ms_ours, "max_rel_diff_vs_ptfock": diff, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {n_j} targets x {n_i} orbitals (general schedule on both sides)", "leg": "cufft",
                       "grid": list(cfg.n), "pairs_per_cufft_batch": ib, "reps": reps}}
    del phi, psi, out
    torch.cuda.empty_cache()
    if emit:
        print(json.dumps(line), flush=True)
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="Si512")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--block-i", type=int, default=0)
    ap.add_argument("--block-j", type=int, default=0)
    ap.add_argument("--workspace-gb", type=float, default=0.0)
    ap.add_argument("--flags", type=int, default=0, help="ptfock_desc.flags (1 = three-stage slab passes, 2 = single stream: one wave in flight)")
    ap.add_argument("--targets", type=int, default=0, help="restrict the step to the first T targets (profiling slices)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--full-application", action="store_true",
                    help="Si1536 / Si1536p: time the whole application (all 3072 targets, symmetric schedule, ~1 min per step) "
                         "instead of one streamed j-block; use with --steps 1 --warmup 0 --no-e2e --no-cpu")
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the second headline config (one Si1536 j-block) that the default Si512 run also times")
    ap.add_argument("--check", action="store_true", help="also compare sampled output columns with the oracle")
    ap.add_argument("--leg", default="fock", choices=["fock", "dense", "copybw", "ptcn", "cufft"],
                    help="fock: the headline exchange path (default); dense: the dense-algebra neighbours; copybw: device "
                         "copy bandwidth vs working-set size (L2-resident vs HBM; profiles/r02_l2_resident.md); ptcn: whole PT-CN time "
                         "steps with the model Hamiltonian (use --config Si64 / Si216); own JSON lines")
    args = ap.parse_args()

    from paper_1905_01348_b200 import synth
    cfg = synth.CONFIGS[args.config]
    if args.impl == "reference":
        reference_arm(args, cfg)
        return

    import torch
    from paper_1905_01348_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    binding.lib()                                   # fails loudly if the CUDA library is missing
    if args.leg == "copybw":
        if rank == 0:
            res = {f"{mb} MiB": binding.measure_copy_bandwidth(mb << 20, reps=max(4, 2048 // mb), device=local)
                   for mb in (16, 24, 32, 48, 64, 128, 512, 2048)}
            print(json.dumps({"metric": "device-to-device copy, read + write GB/s vs source size (working set = 2x)",
                              "unit": "GB/s", "l2_bytes": torch.cuda.get_device_properties(local).L2_cache_size,
                              "copy_GBs": res}), flush=True)
        if dist is not None:
            dist.destroy_process_group()
        return
    if args.leg in ("dense", "ptcn", "cufft"):
        if rank == 0:
            {"dense": dense_leg, "ptcn": ptcn_leg, "cufft": cufft_leg}[args.leg](cfg, args, dev, local)
        if dist is not None:
            dist.destroy_process_group()
        return
    m = measure(cfg, args, dev, local, rank, world, args.steps, args.warmup, not args.no_e2e, not args.no_cpu, args.check)
    # the north-star target names Si512 AND Si1536: the default run also times one streamed j-block of Si1536
    # (bounded: 2 warm-up + 3 timed steps, no e2e / CPU legs) and reports it under config.secondary / roofline.by_config
    second = None
    if cfg.name == "Si512" and not args.no_secondary and not args.targets and world == 1:
        try:
            second = measure(synth.CONFIGS["Si1536"], args, dev, local, rank, world, 3, 2, False, False)
        except Exception as e:                      # e.g. not enough free memory: the headline line still prints
            second = {"error": f"{type(e).__name__}: {e}"}

    # bounded extras of the default run (a few seconds each, after the timed region): the dense-algebra neighbours at the
    # headline size, one PT-CN step at Si64, and the cuFFT side comparison on a 32-target slice
    extras = {}
    if rank == 0 and cfg.name == "Si512" and not args.no_secondary and not args.targets and world == 1:
        small = argparse.Namespace(**dict(vars(args), steps=2))
        for name, fn in (("dense", lambda: dense_leg(cfg, small, dev, local, emit=False)),
                         ("ptcn", lambda: ptcn_leg(synth.CONFIGS["Si64"], small, dev, local, emit=False)),
                         ("cufft", lambda: cufft_leg(cfg, small, dev, local, emit=False, n_targets=32))):
            try:
                extras[name] = fn()
            except Exception as e:                  # never lose the headline line to an extra
                extras[name] = {"error": f"{type(e).__name__}: {e}"}
            torch.cuda.empty_cache()

    if rank == 0:
        line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": m["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": m["vs_baseline"], "dtype": "f64", "data": "synthetic", "config": m["config"],
                "clocks": m["clocks"], "e2e": m["e2e"], "gpu_launches": m["gpu_launches"], "roofline": m["roofline"],
                "survey_72N_frac": m["roofline"]["survey_72N_frac"], "cpu_baseline": m["cpu_baseline"]}
        if second is not None:
            if "error" in second:
                line["config"]["secondary"] = second
            else:
                line["config"]["secondary"] = dict(second["config"], value=second["value"], unit=UNIT,
                                                   ms_per_step=second["ms_per_step"], steps=second["steps"],
                                                   warmup=second["warmup"], clocks=second["clocks"])
                line["roofline"]["by_config"] = {
                    cfg.name: {"frac": m["roofline"]["frac"], "worst_pass_frac": m["roofline"]["worst_pass_frac"]},
                    "Si1536": {"frac": second["roofline"]["frac"], "worst_pass_frac": second["roofline"]["worst_pass_frac"],
                               "per_kernel": second["roofline"]["per_kernel"]}}
                line["survey_72N_frac_Si1536"] = second["roofline"]["survey_72N_frac"]
        if m["parity"]:
            line["parity"] = m["parity"]
        if extras:
            line["config"]["secondary_legs"] = {k: v for k, v in extras.items() if k != "cufft"}
            if "cufft" in extras:
                line["side_comparison_cufft"] = extras["cufft"]
                line["vs_cufft"] = extras["cufft"].get("ptfock_over_cufft")
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
