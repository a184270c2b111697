#!/usr/bin/env python
"""bench.py -- throughput of the stage-2 eigenvector back-transformation (Eq. 6d)
on synthetic inputs of BASELINE.json's shapes.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

One "step" = one call of ``elpa2_trans_ev_tridi_to_band_{d,z}`` over the whole N x nev block (all
SURVEY.md 8(a) rows a1-a6 happen inside that call: T-factor prepass + compact-WY DMMA
kernel).  Default workload: config 4
(real FP64, N = 32768, nbw = 64, nev = 32768), the configuration BASELINE.json's target is quoted
on.  Reflectors for the timed run are the seeded synthetic unitary stream of
``synth_inputs.synthetic_reflectors`` (same layout, lengths, tau != 0 pattern and value range as
chase output; the kernel's work does not depend on the values), X is i.i.d. N(0,1), both generated
on the device.

Prints ONE JSON line (rank 0).  ``value`` = model GFLOP/s (2 N^2 nev real / 8 N^2 nev complex) of
the whole job with all buffers resident in HBM; ``e2e`` = the same metric through the C-ABI
host-buffer entry point with pinned host memory (H2D of reflectors and q, kernel, D2H of q inside
the timed region); ``roofline`` = the kernel against the FP64 ALU peak; ``cpu_baseline`` = the
oracle timed on this box's host cores on a bounded column sample.

N > 1 (torchrun): columns are independent, so every rank back-transforms its own
nev columns with a replicated reflector stream -- no data-path collective; weak scaling.

``--impl reference`` times the CPU oracle (oracle/) on the same config; that leg and the
cpu_baseline leg are the only places this file touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# SURVEY.md 8(d) / BASELINE.json configs: (complex, N, nbw, nev, seed_reflectors, seed_X)
CONFIGS = {
    1: (False, 512, 32, 512, 1001, 2001),
    2: (False, 4096, 64, 4096, 1002, 2002),
    3: (True, 8192, 64, 4096, 1003, 2003),
    4: (False, 32768, 64, 32768, 1004, 2004),
    5: (True, 16384, 128, 8192, 1005, 2005),
}
METRIC = "back-transform FP64 GFLOP/s (2N^2*nev real / 8N^2*nev cplx)"
# FP64 ALU roofline: 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def source_sha() -> str:
    """Fingerprint of the CUDA sources the loaded library was built from (the .git directory does not
    travel to the GPU box, so a commit hash is not available there): sha256 over csrc/*, 16 hex digits."""
    import hashlib

    d = os.path.join(ROOT, "paper_2002_10991_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def lookup_traffic(step: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from
    profiles/traffic.json (written from an ``ncu --set full`` capture; each entry names its profile and
    the source fingerprint it was taken at).  None unless an entry matches this step, this workload AND
    the sources the library in use was built from: a number measured on other code is not reported."""
    try:
        entries = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))["entries"]
    except (OSError, ValueError, KeyError):
        return None, None
    sha = source_sha()
    for e in entries:
        if e.get("step") == step and e.get("workload") == workload and e.get("source_sha") == sha:
            return float(e["dram_bytes_per_launch"]), e.get("profile")
    return None, None


def model_flops(cplx: bool, N: int, nev: int) -> float:
    return (8.0 if cplx else 2.0) * float(N) * float(N) * float(nev)


def workload_name(cfg: int) -> str:
    cplx, N, nbw, nev, _, _ = CONFIGS[cfg]
    if cfg == 0:
        return f"custom (--shape): {'complex' if cplx else 'real'} FP64 N={N} nbw={nbw} nev={nev}"
    return f"config{cfg}: {'complex' if cplx else 'real'} FP64 N={N} nbw={nbw} nev={nev}"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _pump(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def __exit__(self, *exc):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.thread.join(timeout=5)

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_sample_run(cplx, N, nbw, hh_v_np, hh_tau_np, ncols, seed, single=False):
    """Times the oracle, as it stands, on ``ncols`` seeded N(0,1) columns.  Returns (seconds, threads)."""
    import numpy as np

    import oracle

    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, ncols))
    if cplx:
        x = x + 1j * rng.standard_normal((N, ncols))
    x = np.asfortranarray(x.astype(hh_v_np.dtype) if single else x)
    t0 = time.perf_counter()
    oracle.back_transform(N, nbw, hh_v_np, hh_tau_np, x)
    return time.perf_counter() - t0, oracle.num_threads()


def oracle_sample_cols(cplx: bool, N: int, cores: int) -> int:
    """Column count giving roughly 10-30 s of CPU work: the oracle runs about 1.9 (real) / 2.9
    (complex) model GFLOP/s per thread, so one config-4 column is about 1.1 s of one core."""
    per_col = model_flops(cplx, N, 1) / (2.9e9 if cplx else 1.9e9)
    per_core = max(1, min(64, int(16.0 / max(per_col, 1e-9))))
    return cores * per_core


def run_reference(args, rank: int) -> None:
    """--impl reference: the CPU oracle on the same config and metric (rank 0 only)."""
    if rank != 0:
        return
    import numpy as np
    import torch

    import oracle
    from paper_2002_10991_b200 import synth_inputs as si

    cplx, N, nbw, nev, seed_r, seed_x = CONFIGS[args.config]
    cores = oracle.num_threads()
    # per-slot lengths from the oracle's own layout (this arm never loads the CUDA library)
    K = np.array([oracle.hh_blocks(N, nbw, s) for s in range(N - 1)], dtype=np.int64)
    s_of_g = np.repeat(np.arange(N - 1, dtype=np.int64), K)
    k_of_g = np.arange(int(K.sum()), dtype=np.int64) - np.repeat(np.cumsum(K) - K, K)
    lengths = np.minimum(nbw, N - 1 - s_of_g - k_of_g * nbw)
    hv, ht = si.synthetic_reflectors(lengths, nbw, seed_r, cplx, "cpu")
    hv, ht = hv.numpy(), ht.numpy()
    single = args.dtype == "f32"
    if single:                                         # the FP32 oracle on the same stream rounded to float
        f32 = np.complex64 if cplx else np.float32
        hv, ht = hv.astype(f32), ht.astype(f32)
    ncols = oracle_sample_cols(cplx, N, cores)
    times = []
    for i in range(args.warmup + args.steps):
        t, _ = oracle_sample_run(cplx, N, nbw, hv, ht, ncols, seed_x + i, single)
        if i >= args.warmup:
            times.append(t)
    total = sum(times)
    gflops = model_flops(cplx, N, ncols) * len(times) / total / 1e9
    sample = f"{ncols} seeded N(0,1) columns of {nev} per step (columns are independent, PAPER.md:134)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC.replace("FP64", "FP32") if single else METRIC, "value": gflops,
        "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic", "config": {"workload": workload_name(args.config) + (" [FP32 arithmetic]" if single else ""),
                                        "reflectors":
                                        "synthetic unitary stream (host-generated)"},
        "cpu_baseline": {"value": gflops, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gflops, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def chase_kernel_name(cplx: bool, nbw: int) -> str:
    """The kernel elpa2_bulge_chase_{d,z} launches (csrc/bc_chase.cuh), for the JSON line."""
    if os.environ.get("ELPA2_BC_WAVEFRONT", "")[:1] == "1":
        return ("bc_wavefront_kernel_z" if cplx else
                ("bc_wavefront_smem_kernel" if nbw <= 64 else "bc_wavefront_kernel")) + " (one launch per wavefront)"
    if cplx:
        return "bc_persistent_smem_kernel_z" if nbw <= 64 else "bc_persistent_kernel_z"
    return "bc_persistent_kernel" if nbw <= 64 else "bc_persistent_global_kernel"


def run_chase(args, N, nbw, cplx, seed, rank, world, local_rank) -> None:
    """--chase: SURVEY.md 8(f) NEXT-1.  One step = one band -> tridiagonal reduction of the config's seeded
    band matrix on the device (one persistent cooperative kernel + the d/e extraction; one launch per
    wavefront only with ELPA2_BC_WAVEFRONT=1); model work 6 N^2 nbw flops.  Replicas only: the
    chase does not shard."""
    import numpy as np
    import torch

    from paper_2002_10991_b200 import binding, shard, synth_inputs as si

    ab_h = torch.from_numpy(np.ascontiguousarray(si.band_matrix(N, nbw, seed, cplx).T)).pin_memory()
    ab = torch.empty_like(ab_h, device="cuda")
    flops = (24.0 if cplx else 6.0) * float(N) * float(N) * nbw
    stream = torch.cuda.current_stream()
    times, launches = [], 0
    dfma_tf = binding.probe_fp64(0, 8192, 20)
    with ClockSampler(local_rank) as clocks:
        for i in range(args.warmup + args.steps):
            ab.copy_(ab_h, non_blocking=True)          # the chase overwrites its input: restore, untimed
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            hv, ht, d, e = binding.bulge_chase(N, nbw, ab, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            if i >= args.warmup:
                times.append(e0.elapsed_time(e1))
                launches += binding.last_launch_count()
    ms = shard.max_over_ranks(sum(times) / len(times), None)
    # sanity of the result that was timed: T has the eigenvalue sum (trace) of B
    diag = ab_h[:, 0].real if cplx else ab_h[:, 0]
    tr_err = abs(float(d.sum().item()) - float(diag.sum().item())) / max(1.0, float(diag.abs().sum().item()))
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle

        Ns = min(N, 2048 if cplx else 4096)             # bounded sample: work grows like N^2
        ab_s = si.band_matrix(Ns, nbw, seed, cplx)
        t0 = time.perf_counter()
        oracle.bulge_chase(ab_s, nbw)
        ts = time.perf_counter() - t0
        cpu = {"value": (24.0 if cplx else 6.0) * Ns * Ns * nbw / ts / 1e9, "unit": "GFLOP/s", "cores": 1, "kind": "oracle", "seconds": ts,
               "sample": f"the same seeded band matrix truncated to N = {Ns} (single thread: the chase is sequential)"}
    if rank == 0:
        achieved = flops / (ms * 1e-3) / 1e12
        print(json.dumps({
            "metric": "bulge chase FP64 GFLOP/s (6 N^2 nbw real / 24 N^2 nbw cplx)", "value": world * flops / (ms * 1e-3) / 1e9, "unit": "GFLOP/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"bulge chase of config {args.config}'s band matrix: "
                                   f"{'complex' if cplx else 'real'} FP64 N={N} nbw={nbw}",
                       "parallelism": "replicas only", "l2": "band matrix restored from host before every step"},
            "roofline": {"bound": "alu", "achieved": achieved, "peak": dfma_tf, "unit": "TFLOP/s", "frac": achieved / dfma_tf,
                         "peak_source": "DFMA probe of this run; first version: launch- and latency-bound",
                         "kernel": chase_kernel_name(cplx, nbw), "kernel_ms": ms,
                         "traffic": None},
            "clocks": clocks.summary(), "e2e": None, "gpu_launches": launches, "cpu_baseline": cpu,
            "checks": {"relative_trace_error": tr_err},
        }), flush=True)


METRIC_6E = "band->full back-transform FP64 GFLOP/s (4*nev*sum(L) real / 16*nev*sum(L) cplx)"


def b2f_flops(cplx: bool, N: int, nbw: int, nev: int) -> float:
    """Algorithmic flops of Eq. 6e: one reflector of length L on one column = 4 L flops (16 L complex);
    sum over j < Nv of L_j = N - nbw - j is Nv (Nv + 3) / 2."""
    Nv = max(N - nbw - 1, 0)
    return (16.0 if cplx else 4.0) * nev * (Nv * (Nv + 3) / 2.0)


def b2f_workload_name(cfg: int) -> str:
    cplx, N, nbw, nev, _, _ = CONFIGS[cfg]
    tag = "custom (--shape)" if cfg == 0 else f"6e-config{cfg}"
    return f"{tag}: {'complex' if cplx else 'real'} FP64 N={N} nbw={nbw} nev={nev}"


def b2f_oracle_cols(cplx: bool, N: int, nbw: int, cores: int) -> int:
    per_col = b2f_flops(cplx, N, nbw, 1) / (2.9e9 if cplx else 1.9e9)
    return cores * max(1, min(64, int(16.0 / max(per_col, 1e-9))))


def b2f_oracle_run(cplx, N, nbw, hv_np, tau_np, ncols, seed):
    import numpy as np

    import oracle

    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, ncols))
    if cplx:
        x = x + 1j * rng.standard_normal((N, ncols))
    x = np.asfortranarray(x)
    t0 = time.perf_counter()
    oracle.band_to_full_back(N, nbw, hv_np, tau_np, x)
    return time.perf_counter() - t0, oracle.num_threads()


def run_b2f_reference(args, rank: int) -> None:
    """--impl reference --step 6e: the oracle's plain sequential application on a column sample."""
    if rank != 0:
        return
    import oracle
    from paper_2002_10991_b200 import synth_inputs as si

    cplx, N, nbw, nev, seed_r, seed_x = CONFIGS[args.config]
    cores = oracle.num_threads()
    hv, tau = si.synthetic_full_reflectors(N, nbw, seed_r, cplx, "cpu")
    hv_np, tau_np = hv.numpy(), tau.numpy()
    ncols = b2f_oracle_cols(cplx, N, nbw, cores)
    times = []
    for i in range(args.warmup + args.steps):
        t, _ = b2f_oracle_run(cplx, N, nbw, hv_np, tau_np, ncols, seed_x + i)
        if i >= args.warmup:
            times.append(t)
    total = sum(times)
    gflops = b2f_flops(cplx, N, nbw, ncols) * len(times) / total / 1e9
    sample = f"{ncols} seeded N(0,1) columns of {nev} per step (columns are independent, PAPER.md:134)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC_6E, "value": gflops, "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": b2f_workload_name(args.config), "reflectors": "synthetic unitary set (host-generated)"},
        "cpu_baseline": {"value": gflops, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gflops, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def run_b2f(args, rank, world, local_rank, dist) -> None:
    """--step 6e: SURVEY.md 8(f) NEXT-2.  One step = one call of ``elpa2_trans_ev_band_to_full_{d,z}`` over the
    whole N x nev block (T-factor prepass + the fused DMMA kernel).  Reflectors: the seeded synthetic
    unitary set in the Eq. 6e layout (the oracle's O(N^3) full -> band reduction is out of reach at these
    sizes); q i.i.d. N(0,1); both generated on the device.  N > 1: column shards, no collective."""
    import torch

    from paper_2002_10991_b200 import binding, shard, synth_inputs as si

    cplx, N, nbw, nev, seed_r, seed_x = CONFIGS[args.config]
    esz = 16 if cplx else 8
    Nv = max(N - nbw - 1, 0)
    flops = b2f_flops(cplx, N, nbw, nev)
    hv, tau = si.synthetic_full_reflectors(N, nbw, seed_r, cplx, "cuda")
    q = si.gaussian_block(N, nev, seed_x + 7919 * rank, cplx, "cuda")
    stream = torch.cuda.current_stream()

    def step():
        binding.trans_ev_band_to_full(N, nbw, hv, tau, q, stream=stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    dfma_tf = binding.probe_fp64(0, 8192, 20)
    dmma_tf = binding.probe_fp64(1, 8192, 20)
    ncheck = min(nev, 64)
    nrm0 = torch.linalg.vector_norm(q[:, :ncheck], dim=0)
    for _ in range(args.warmup):
        step()
    barrier()
    launches = 0
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local_rank) as clocks:
        barrier()
        ev[0].record(stream)
        for i in range(args.steps):
            step()
            launches += binding.last_launch_count()
            ev[i + 1].record(stream)
        barrier()
    clk = clocks.summary()
    step_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = shard.max_over_ranks(ev[0].elapsed_time(ev[args.steps]), dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = shard.aggregate_throughput(flops, world, ms_per_step * 1e-3) / 1e9
    nrm = torch.linalg.vector_norm(q[:, :ncheck], dim=0)
    norm_dev = float((nrm / nrm0 - 1.0).abs().max().item())

    e2e = None
    if args.e2e_steps > 0:
        ldv = hv.stride(1) if Nv > 1 else N + (N & 1)
        hv_h = torch.empty((Nv, ldv), dtype=hv.dtype, pin_memory=True)
        hv_h[:, :N].copy_(hv.t())
        if ldv > N:
            hv_h[:, N:].zero_()
        tau_h = torch.empty(tau.shape, dtype=tau.dtype, pin_memory=True).copy_(tau)
        q_h = torch.empty((nev, N), dtype=q.dtype, pin_memory=True).copy_(q.t())
        torch.cuda.synchronize()
        hv_np, tau_np, q_np = hv_h.numpy().T, tau_h.numpy(), q_h.numpy().T
        binding.trans_ev_band_to_full_host(N, nbw, hv_np, tau_np, q_np)         # warm-up: scratch alloc
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            binding.trans_ev_band_to_full_host(N, nbw, hv_np, tau_np, q_np)
            launches += binding.last_launch_count()
        torch.cuda.synchronize()
        dt = shard.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        e2e = {"value": world * flops * args.e2e_steps / dt / 1e9, "unit": "GFLOP/s",
               "h2d_bytes_per_step": (ldv * Nv + Nv + N * nev) * esz, "d2h_bytes_per_step": N * nev * esz,
               "steps": args.e2e_steps, "timer": "host wall clock around synchronous calls"}
        del hv_h, tau_h, q_h

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle

        cores = oracle.num_threads()
        ncols = b2f_oracle_cols(cplx, N, nbw, cores)
        hv_np = hv.t().cpu().numpy().T                       # (N, Nv), column-major, whatever ldv the copy keeps
        tsec, cores = b2f_oracle_run(cplx, N, nbw, hv_np, tau.cpu().numpy(), ncols, seed_x)
        cpu = {"value": b2f_flops(cplx, N, nbw, ncols) / tsec / 1e9, "unit": "GFLOP/s", "cores": cores,
               "kind": "oracle", "seconds": tsec,
               "sample": f"{ncols} seeded N(0,1) columns of {nev}, all {Nv} reflectors (columns are independent, PAPER.md:134)"}
        del hv_np

    if rank == 0:
        kern_ms = sum(step_ms) / len(step_ms)
        achieved = flops / (kern_ms * 1e-3) / 1e12
        traffic, traffic_profile = lookup_traffic("6e", b2f_workload_name(args.config))
        print(json.dumps({
            "metric": METRIC_6E, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": b2f_workload_name(args.config), "N": N, "nbw": nbw, "nev_per_gpu": nev, "reflectors_Nv": Nv,
                       "reflectors": "synthetic unitary set in the Eq. 6e layout, device-generated (DESIGN.md input recipe)",
                       "l2": "inputs larger than L2 (%.2f GiB of q + reflectors per step)" % ((N * Nv + 2 * N * nev) * esz / 2**30),
                       "parallelism": "column shards, no collective" if world > 1 else "single GPU",
                       "source_sha": source_sha()},
            "roofline": {"bound": "tensor", "achieved": achieved, "peak": dmma_tf, "unit": "TFLOP/s", "frac": achieved / dmma_tf,
                         "peak_source": "FP64 DMMA m8n8k4 probe measured in this run (elpa2_bt_probe_fp64 kind 1); "
                                        "MEASURED_PEAKS.json has no FP64 figure",
                         "peak_dfma_probe": dfma_tf, "peak_dmma_probe": dmma_tf, "peak_nominal": NOMINAL_FP64_TFLOPS,
                         "frac_nominal": achieved / NOMINAL_FP64_TFLOPS,
                         "kernel": ("bt_b2fz_kernel" if cplx else "bt_b2f_kernel") + " (the interval also holds its T-factor prepass kernel)",
                         "kernel_ms": kern_ms, "algorithmic_flops_per_launch": flops,
                         "traffic": traffic, "traffic_profile": traffic_profile},
            "clocks": clk, "e2e": e2e, "gpu_launches": launches, "cpu_baseline": cpu,
            "checks": {"max_rel_column_norm_drift_after_all_steps": norm_dev},
        }), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_rowpipe(args, rank, world, local_rank, dist) -> None:
    """--row-pipeline R: SURVEY.md 8(f) NEXT-3.  One step = the whole back-transformation of
    the config's N x nev block with the rows spread over R ranks (paper_2002_10991_b200/rowpipe.py).
    world > 1: R = world real ranks, "scaling": "strong", value = model flops / max-over-ranks time.
    world == 1: R emulated ranks on this device, one after another."""
    import torch

    from paper_2002_10991_b200 import binding, rowpipe, shard, synth_inputs as si

    cplx, N, nbw, nev, seed_r, seed_x = CONFIGS[args.config]
    R = world if world > 1 else args.row_pipeline
    flops = model_flops(cplx, N, nev)
    lengths = binding.hh_lengths(N, nbw)
    hh_v, hh_tau = si.synthetic_reflectors(lengths, nbw, seed_r, cplx, "cuda")
    bounds = rowpipe.partition_rows(N, R, nbw)
    mine = range(R) if world == 1 else [rank]
    dt = torch.complex128 if cplx else torch.float64
    gen = torch.Generator(device="cuda")
    bufs = {}
    for r in mine:
        n = rowpipe.local_rows(N, nbw, bounds, r)
        gen.manual_seed(seed_x + r)
        back = torch.randn((nev, n, 2) if cplx else (nev, n), generator=gen, device="cuda", dtype=torch.float64)
        bufs[r] = (torch.view_as_complex(back) if cplx else back).t()          # (n, nev) column-major, ldq = n
    apply_fn = rowpipe.device_apply(N, nbw, hh_v, hh_tau)
    stream = torch.cuda.current_stream()

    def step():
        if world == 1:
            rowpipe.run_emulated(N, nbw, bounds, [bufs[r] for r in range(R)], apply_fn)
        else:
            rowpipe.run(N, nbw, bounds, bufs[rank], dist, apply_fn)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    dmma_tf = binding.probe_fp64(1, 8192, 20)
    for _ in range(args.warmup):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        barrier()
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        barrier()
    ms = shard.max_over_ranks(e0.elapsed_time(e1), dist, "cuda") / args.steps
    if rank == 0:
        nops = sum(1 for r in range(R) for o in rowpipe.schedule(N, nbw, bounds, r) if o.kind == "apply")
        nmsg = sum(1 for r in range(R) for o in rowpipe.schedule(N, nbw, bounds, r) if o.kind == "send")
        achieved = flops / (ms * 1e-3) / 1e12
        print(json.dumps({
            "metric": METRIC, "value": flops / (ms * 1e-3) / 1e9, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config) + f" [row pipeline, R = {R}"
                                   + (" emulated on one device" if world == 1 else " ranks") + "]",
                       "N": N, "nbw": nbw, "nev": nev, "row_bounds": bounds, "row_block_calls_per_step": nops,
                       "halo_messages_per_step": nmsg, "halo_message_bytes": nbw * nev * (16 if cplx else 8),
                       "parallelism": f"rows over {R} ranks, nbw-row halos" + (" over NCCL" if world > 1 else " (device copies)"),
                       "source_sha": source_sha()},
            "roofline": {"bound": "tensor", "achieved": achieved, "peak": dmma_tf * max(world, 1), "unit": "TFLOP/s",
                         "frac": achieved / (dmma_tf * max(world, 1)),
                         "peak_source": "FP64 DMMA probe of rank 0 x ranks", "kernel": "bt_wy(z)_kernel, sub-range launches",
                         "kernel_ms": ms, "algorithmic_flops_per_launch": flops, "traffic": None},
            "clocks": clocks.summary(), "e2e": None, "gpu_launches": 2 * nops * args.steps, "cpu_baseline": None,
        }), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2, help="timed host-buffer calls (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variant", type=int, default=0, choices=[0, 1, 2, 3],
                    help="library variant for A/B runs (include/elpa2_bt.h): 0 default, 2 register window, 3 two chains per pass")
    ap.add_argument("--chain-parallel", type=int, default=0, choices=[0, 1, 2, 4],
                    help="testing aid: force P warps per slab in the default variant (0 = the library's plan)")
    ap.add_argument("--chase", action="store_true",
                    help="time SURVEY 8(f) NEXT-1 instead: the GPU bulge chase (real configs) that produces the reflectors")
    ap.add_argument("--step", default="6d", choices=["6d", "6e"],
                    help="6d (default): tridiagonal -> band back-transformation, the north star; 6e: SURVEY 8(f) NEXT-2, "
                         "band -> full back-transformation on the same config's N, nbw, nev")
    ap.add_argument("--nev-frac", type=float, default=None,
                    help="partial spectrum (PAPER.md:218): replace nev by round(frac * N)")
    ap.add_argument("--reflectors", default="chase", choices=["chase", "synthetic"],
                    help="step 6d: 'chase' (default) = the reflectors BASELINE.json specifies, produced on the device by "
                         "elpa2_bulge_chase_{d,z} from the config's seeded band matrix (bit-identical to the oracle's chase: "
                         "tests/test_gpu_configs.py), outside the timed region; 'synthetic' = the seeded unitary stream")
    ap.add_argument("--row-pipeline", type=int, default=0, metavar="R",
                    help="SURVEY 8(f) NEXT-3: time the row-pipelined form instead (strong scaling over rows).  Under "
                         "torchrun every rank owns a block of rows of ALL nev columns and hands nbw-row halos over NCCL; "
                         "on one GPU, R ranks are emulated one after another on the same device (the sum of all ranks' "
                         "work: measures the cost of the row-block form, not a speed-up)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"],
                    help="f32: SURVEY 8(f) NEXT-4, the FP32 calls elpa2_trans_ev_tridi_to_band_{s,c} on the config's shape "
                         "(step 6d only; real nbw <= 128, complex nbw <= 64)")
    ap.add_argument("--shape", default=None, metavar="d|z,N,nbw,nev",
                    help="profiling aid: replace the chosen config's shape (named 'custom' in the output)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        print(f"note: --warmup {args.warmup} < 3 breaks the timing rules", file=sys.stderr)

    if args.shape:
        t, n_, b_, e_ = args.shape.split(",")
        CONFIGS[0] = (t == "z", int(n_), int(b_), int(e_), 1000, 2000)
        args.config = 0

    if args.nev_frac is not None:
        c = CONFIGS[args.config]
        CONFIGS[0] = (c[0], c[1], c[2], max(1, int(round(args.nev_frac * c[1]))), c[4], c[5])
        args.config = 0

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if args.step == "6e":
            run_b2f_reference(args, rank)
        else:
            run_reference(args, rank)
        return

    import numpy as np
    import torch

    from paper_2002_10991_b200 import binding, shard, synth_inputs as si

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cplx, N, nbw, nev, seed_r, seed_x = CONFIGS[args.config]
    esz = 16 if cplx else 8
    flops = model_flops(cplx, N, nev)
    if args.chase:
        run_chase(args, N, nbw, cplx, seed_r, rank, world, local_rank)
        return
    if args.step == "6e":
        run_b2f(args, rank, world, local_rank, dist)
        return
    if args.row_pipeline > 0:
        run_rowpipe(args, rank, world, local_rank, dist)
        return

    # ---- inputs, generated on the device (each rank: its own nev columns, same reflectors) ----
    lengths = binding.hh_lengths(N, nbw)
    G = int(lengths.shape[0])
    assert G == binding.hh_count(N, nbw)
    chase_ms = None
    if args.reflectors == "chase" and nbw in (32, 64, 128):
        ab = torch.from_numpy(np.ascontiguousarray(si.band_matrix(N, nbw, seed_r, cplx).T)).cuda()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        hh_v, hh_tau, _d, _e = binding.bulge_chase(N, nbw, ab)
        c1.record()
        torch.cuda.synchronize()
        chase_ms = c0.elapsed_time(c1)
        del ab, _d, _e
        reflector_text = ("GPU bulge chase (elpa2_bulge_chase) of the config's seeded band matrix, seed %d: "
                          "BASELINE.json's reflectors, untimed (%.0f ms)" % (seed_r, chase_ms))
    else:
        hh_v, hh_tau = si.synthetic_reflectors(lengths, nbw, seed_r, cplx, "cuda")
        reflector_text = "synthetic unitary stream, device-generated (DESIGN.md input recipe)"
    q = si.gaussian_block(N, nev, seed_x + 7919 * rank, cplx, "cuda")
    single = args.dtype == "f32"
    if single:
        # the FP64 stream rounded to float: unitary to FP32 rounding, same layout
        f32 = torch.complex64 if cplx else torch.float32
        hh_v, hh_tau = hh_v.to(f32), hh_tau.to(f32)
        q = q.t().to(f32).t()                      # keeps the column-major storage
        esz //= 2
    stream = torch.cuda.current_stream()
    binding.set_variant(args.variant)
    binding.set_chain_parallel(args.chain_parallel)

    def step():
        binding.trans_ev_tridi_to_band(N, nbw, hh_v, hh_tau, q, stream=stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- FP64 peaks of this device, measured live (outside the timed region): the real path is a
    #      path is a DMMA (FP64 tensor core) contraction, judged against the DMMA probe; the DFMA
    #      probe (the same pipe) is reported beside it
    dfma_tf = binding.probe_fp64(0, 8192, 20)
    dmma_tf = binding.probe_fp64(1, 8192, 20)
    tensor_path = True
    peak_tf = dmma_tf if tensor_path else dfma_tf

    ncheck = min(nev, 64)
    nrm0 = torch.linalg.vector_norm(q[:, :ncheck], dim=0)
    for _ in range(args.warmup):
        step()
    barrier()
    launches = 0
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local_rank) as clocks:
        barrier()
        ev[0].record(stream)
        for i in range(args.steps):
            step()
            launches += binding.last_launch_count()
            ev[i + 1].record(stream)
        barrier()
    clk = clocks.summary()
    step_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = shard.max_over_ranks(ev[0].elapsed_time(ev[args.steps]), dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = shard.aggregate_throughput(flops, world, ms_per_step * 1e-3) / 1e9

    # unitarity check on the timed buffer (every H is unitary, so column norms must not move)
    nrm = torch.linalg.vector_norm(q[:, :ncheck], dim=0)
    norm_dev = float((nrm / nrm0 - 1.0).abs().max().item())

    # ---- e2e: host buffers through the C-ABI host entry point (rank-local, pinned memory) ----
    e2e = None
    if args.e2e_steps > 0:
        hv_h = torch.empty(hh_v.shape, dtype=hh_v.dtype, pin_memory=True).copy_(hh_v)
        ht_h = torch.empty(hh_tau.shape, dtype=hh_tau.dtype, pin_memory=True).copy_(hh_tau)
        q_h = torch.empty((nev, N), dtype=q.dtype, pin_memory=True).copy_(q.t())
        torch.cuda.synchronize()
        hv_np, ht_np, q_np = hv_h.numpy(), ht_h.numpy(), q_h.numpy().T      # q_np: (N, nev) Fortran
        binding.trans_ev_tridi_to_band_host(N, nbw, hv_np, ht_np, q_np)     # warm-up: scratch alloc
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            binding.trans_ev_tridi_to_band_host(N, nbw, hv_np, ht_np, q_np)
            launches += binding.last_launch_count()
        torch.cuda.synchronize()
        dt = shard.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        h2d = (G * nbw + G + N * nev) * esz
        d2h = N * nev * esz
        e2e = {"value": world * flops * args.e2e_steps / dt / 1e9, "unit": "GFLOP/s",
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": args.e2e_steps,
               "timer": "host wall clock around synchronous calls"}
        del hv_h, ht_h, q_h

    # ---- cpu_baseline: the oracle on a bounded column sample (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle

        cores = oracle.num_threads()
        ncols = oracle_sample_cols(cplx, N, cores)
        tsec, cores = oracle_sample_run(cplx, N, nbw, hh_v.cpu().numpy(), hh_tau.cpu().numpy(), ncols, seed_x, single)
        cpu = {"value": model_flops(cplx, N, ncols) / tsec / 1e9, "unit": "GFLOP/s", "cores": cores,
               "kind": "oracle", "seconds": tsec,
               "sample": f"{ncols} seeded N(0,1) columns of {nev}, all {G} reflectors "
                         "(columns are independent, PAPER.md:134)"}

    if rank == 0:
        kern_ms = sum(step_ms) / len(step_ms)
        achieved = flops / (kern_ms * 1e-3) / 1e12
        traffic, traffic_profile = lookup_traffic("6d", workload_name(args.config)) if args.variant == 0 else (None, None)
        if single:
            traffic, traffic_profile = lookup_traffic("6d-f32", workload_name(args.config))
        out = {
            "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": workload_name(args.config) + (" [FP32 arithmetic]" if single else ""), "N": N, "nbw": nbw, "nev_per_gpu": nev,
                       "reflector_slots": G,
                       "reflectors": reflector_text,
                       "l2": ("inputs larger than L2 (%.2f GiB of q + reflectors per step)"
                              % ((G * nbw + G + 2 * N * nev) * esz / 2**30)) if (G * nbw + N * nev) * esz > 2**28
                             else "inputs smaller than L2; config is latency-bound (DESIGN.md)",
                       "parallelism": "column shards, no collective" if world > 1 else "single GPU",
                       "variant": args.variant, "chain_parallel": args.chain_parallel or "planned",
                       "plan": binding.plan(cplx, N, nbw, nev, torch.cuda.get_device_properties(local_rank).multi_processor_count),
                       "source_sha": source_sha()},
            "roofline": {"bound": "tensor" if tensor_path else "alu", "achieved": achieved, "peak": peak_tf,
                         "unit": "TFLOP/s", "frac": achieved / peak_tf,
                         "peak_source": ("FP64 %s probe measured in this run (elpa2_bt_probe_fp64 kind %d); "
                                         "MEASURED_PEAKS.json has no FP64 figure"
                                         % (("DMMA m8n8k4", 1) if tensor_path else ("DFMA", 0))),
                         "peak_dfma_probe": dfma_tf, "peak_dmma_probe": dmma_tf,
                         "peak_nominal": NOMINAL_FP64_TFLOPS, "frac_nominal": achieved / NOMINAL_FP64_TFLOPS,
                         "kernel": ("bt_wyz_kernel" if cplx else "bt_wy_kernel")
                                   + " (the interval also holds its T-factor prepass kernel)",
                         "kernel_ms": kern_ms, "algorithmic_flops_per_launch": flops,
                         "traffic": traffic, "traffic_profile": traffic_profile},
            "clocks": clk, "e2e": e2e, "gpu_launches": launches, "cpu_baseline": cpu,
            "checks": {"max_rel_column_norm_drift_after_all_steps": norm_dev},
        }
        if single:
            # plain FP32 FMA pipe: 148 SMs x 128 FFMA/clk x 2 flop x 1.965 GHz, nominal -- no FP32
            # figure in MEASURED_PEAKS.json; the metric's model flops are counted in FP32 here
            out["metric"] = METRIC.replace("FP64", "FP32")
            out["roofline"] = {"bound": "alu", "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
                               "frac": achieved / NOMINAL_FP32_TFLOPS,
                               "peak_source": "nominal FP32 FMA rate: 148 SMs x 128 FFMA/clk x 2 x 1.965 GHz (DESIGN.md 10)",
                               "kernel": "bt_f32_kernel", "kernel_ms": kern_ms, "algorithmic_flops_per_launch": flops,
                               "traffic": traffic, "traffic_profile": traffic_profile}
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
