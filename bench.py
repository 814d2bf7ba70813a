#!/usr/bin/env python
"""bench.py -- the driver's benchmark contract for the QMC hot path.

A "step" is one pass of the whole hot path over one batch of synthetic walkers of
BASELINE.json configs[3] (CO, 14 electrons, 30 STOs, 100 determinants, 131072 walkers
per GPU): 20 all-electron Metropolis sweeps (qmc_metropolis) + the local energy of the
resulting walkers (qmc_local_energy) + the batch mean / standard error (qmc_batch_stats).

value   = walker*E_L evaluations per second (M / device time of qmc_local_energy), inputs
          resident in HBM; the Metropolis walker-steps/s of the same steps is reported
          beside it ("metropolis").
e2e     = the same metric through the C ABI call that takes HOST buffers (qmc_local_energy_host): pinned
          host walkers -> H2D -> kernels -> D2H of log|Psi|, sign, E_L, all inside the timed region (the
          call pipelines walker ranges over two streams so the copies overlap the kernels).
roofline= model FP64 flop-equivalents per launch / mean launch time of the kernel that dominates the timed step (the
          sampler: one launch = 20 sweeps), against the FP64 peak measured in this same process: the largest of the
          DFMA and DMMA microbenchmarks of qmc_fp64_peak (they run on one pipe); the fused E_L kernel and the whole
          E_L call are reported beside it (roofline.local_energy_kernel) against the same denominator.
cpu_baseline = the CPU oracle, as it stands, on the host cores, on a bounded sample.

N > 1 (torchrun): walkers are sharded, M per GPU fixed (weak scaling), no data-path
collective; Philox counters use the global walker index.  --impl reference times the oracle.
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
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

WORKLOAD = "BASELINE configs[3]: CO 14e, 30 STOs, 14 MOs, 100 determinants, 131072 walkers/GPU, " \
           "20 Metropolis sweeps (step 0.2) + E_L + batch stats"
METRIC = "walker*E_L evals/sec (CO 14e, FP64); Metropolis walker-steps/sec reported beside it"
UNIT = "walker*E_L evals/s"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for row in self.rows:
            p = [x.strip() for x in row.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for nm, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(d, r, n_sample, threads):
    """Time the CPU oracle's E_L on the first n_sample walkers; returns walkers/s."""
    from oracle import binding as ob
    o = ob.OracleSystem(d)
    rs = np.ascontiguousarray(r[:, :, :n_sample])
    ob.local_energy(o, rs[:, :, :64], threads=1)  # load + warm
    t0 = time.perf_counter()
    ob.local_energy(o, rs, threads=threads)
    dt = time.perf_counter() - t0
    return n_sample / dt, dt


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config / metric."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2506_09743_b200 import workloads as wl
    cores = os.cpu_count() or 1
    n_sample = 4096
    d, r = wl.co(M=n_sample)
    times = []
    for i in range(args.warmup + args.steps):
        v, dt = oracle_sample(d, r, n_sample, cores)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = n_sample / (ms * 1e-3)
    sample = f"E_L of {n_sample} CO walkers per step (the oracle's explicit per-determinant path), {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


K_DERIV = 5  # timed repetitions of the NEXT-1 block


def profile_traffic(name):
    """DRAM bytes (read + written) per launch of a kernel, from its committed ncu summary under profiles/."""
    import re
    path = os.path.join(ROOT, "profiles", name)
    try:
        m = re.search(r"dram_bytes_per_launch:\s*(\d+)", open(path).read())
        return int(m.group(1)) if m else None
    except OSError:
        return None
E2E_CHUNKS = 4  # walker ranges pipelined by qmc_local_energy_host (measured: 1, 2, 4, 8, 16 ranges -> 91, 116, 126, 119, 105 M walker*E_L/s)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--walkers", type=int, default=131072, help="walkers per GPU")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2506_09743_b200 import binding as qb
    from paper_2506_09743_b200 import workloads as wl
    from paper_2506_09743_b200.sharding import max_over_ranks

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    M = args.walkers
    n_sweeps, step_size, seed = 20, 0.2, 20250609
    d, r_host = wl.co(M=M)
    if world > 1:  # every rank gets its own walkers; constants are replicated
        r_host = wl.make_walkers(np.random.default_rng([3, 100 + rank]), d.atom_xyz, d.n_e, M)
    sysh = qb.QmcSystem(d, device=local_rank)
    st = torch.cuda.current_stream()

    peak_dfma = qb.fp64_peak(0, reps=5, device=local_rank)
    peak_dmma = qb.fp64_peak(1, reps=5, device=local_rank)
    peak_dfma2 = qb.fp64_peak(3, reps=5, device=local_rank)   # two-register operand form
    peak_dfma3 = qb.fp64_peak(4, reps=5, device=local_rank)   # three distinct registers
    rate_chain = qb.fp64_peak(5, reps=5, device=local_rank)   # one dependent chain per SM sub-partition (latency)
    peak = max(peak_dfma, peak_dmma, peak_dfma2)              # DFMA and DMMA share the FP64 pipe: its demonstrated rate

    r0 = torch.from_numpy(r_host).to(dev)
    r = r0.clone()
    lp = torch.empty(M, dtype=torch.float64, device=dev)
    sg = torch.empty_like(lp)
    el = torch.empty_like(lp)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)  # > 126 MB L2
    r_pin = torch.from_numpy(r_host).pin_memory()
    out_pin = torch.empty((3, M), dtype=torch.float64).pin_memory()

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def one_step(k, timed):
        """Metropolis (20 sweeps) -> E_L -> batch stats; returns event triple."""
        flush.fill_(k & 0xFF)
        a, b, c, e = ev(), ev(), ev(), ev()
        a.record(st)
        sysh.metropolis(r, step_size, n_sweeps, seed, sweep_offset=k * n_sweeps, walker_offset=rank * M,
                        logpsi=lp, sign=sg)
        b.record(st)
        sysh.local_energy(r, lp, sg, el)
        c.record(st)
        mean, err = qb.batch_stats(el)
        e.record(st)
        return (a, b, c, e, mean, err)

    for k in range(args.warmup):
        one_step(k, False)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    qb.launch_count(reset=True)
    torch.cuda.synchronize()
    recs = [one_step(args.warmup + k, True) for k in range(args.steps)]
    torch.cuda.synchronize()
    launches = qb.launch_count()
    if world > 1:
        dist.barrier()
    t_met = sum(x[0].elapsed_time(x[1]) for x in recs) * 1e-3
    t_el = sum(x[1].elapsed_time(x[2]) for x in recs) * 1e-3
    t_all = sum(x[0].elapsed_time(x[3]) for x in recs) * 1e-3
    # ---- the dominant kernel's own launch duration (roofline): the same K steps once more (flush, sampler, E_L,
    # statistics) with CUDA events recorded INSIDE the library on the launching stream before and after the
    # table-path kernel.  Not done in the timed steps above: the extra event records between the two kernels
    # lengthen the call by ~10 us (measured), which would tax the headline value.
    sysh.set_kernel_timing(True)
    t_kmain = t_kfb = 0.0
    for k in range(args.steps):
        one_step(args.warmup + args.steps + k, False)   # batch_stats synchronises the stream
        k_main, k_fb = sysh.kernel_times()
        t_kmain += k_main * 1e-3
        t_kfb += k_fb * 1e-3
    sysh.set_kernel_timing(False)

    # ---- end to end through the C ABI with host buffers
    # qmc_local_energy_host: pinned host walkers -> (chunked, pipelined) H2D -> kernels -> D2H of log|Psi|, sign,
    # E_L into pinned host memory; the call is synchronous, so wall-clock time around it is the end-to-end time
    def e2e_step():
        sysh.local_energy_host(r_pin, out_pin, n_chunks=E2E_CHUNKS)
    for _ in range(3):
        e2e_step()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    t_e2e = time.perf_counter() - t0
    # the same through one upload: sample AND evaluate from host buffers (qmc_vmc_step_host: H2D of the walkers,
    # 20 sweeps, E_L, statistics, D2H of walkers and energies) -- what a VMC iteration moves over PCIe
    el_pin = torch.empty(M, dtype=torch.float64).pin_memory()
    r_step = r_pin.clone().pin_memory()
    for k in range(2):
        sysh.vmc_step_host(r_step, step_size, n_sweeps, seed, sweep_offset=k * n_sweeps, walker_offset=rank * M, eloc_host=el_pin, n_chunks=2)
    t0 = time.perf_counter()
    for k in range(args.steps):
        sysh.vmc_step_host(r_step, step_size, n_sweeps, seed, sweep_offset=(2 + k) * n_sweeps, walker_offset=rank * M, eloc_host=el_pin, n_chunks=2)
    t_vmc = time.perf_counter() - t0
    clocks = sampler.stop()

    # ---- E_L + parameter derivatives O (eq. 6 factors) and the gradient estimator,
    # reported beside the headline (same walkers; O is [M][n_param = 6 + n_det] doubles written to and read from HBM)
    n_par = sysh.n_param()
    O = torch.empty((M, n_par), dtype=torch.float64, device=dev)
    t_d = t_g = 0.0
    for k in range(3 + K_DERIV):
        flush.fill_(k & 0xFF)
        a, b, c = ev(), ev(), ev()
        a.record(st)
        sysh.log_derivatives(r, lp, sg, el, O)
        b.record(st)
        e_v, grad = qb.energy_gradient(el, O)
        c.record(st)
        torch.cuda.synchronize()
        if k >= 3:
            t_d += a.elapsed_time(b) * 1e-3
            t_g += b.elapsed_time(c) * 1e-3
    del O
    t_fu = 0.0
    for k in range(3 + K_DERIV):
        flush.fill_(k & 0xFF)
        a, b = ev(), ev()
        a.record(st)
        _, _, _, e_vf, grad_f = sysh.local_energy_gradient(r, lp, sg, el)
        b.record(st)
        torch.cuda.synchronize()
        if k >= 3:
            t_fu += a.elapsed_time(b) * 1e-3
    # orbital-parameter derivatives (MO coefficients, AO exponents) on the first 32768 walkers of the batch
    M_orb = min(M, 32768)
    r_orb = r[:, :, :M_orb].contiguous()
    t_o = 0.0
    for k in range(3 + K_DERIV):
        a, b = ev(), ev()
        a.record(st)
        dC, dz = sysh.orbital_derivatives(r_orb, d.n_ao, d.n_mo)
        b.record(st)
        torch.cuda.synchronize()
        if k >= 3:
            t_o += a.elapsed_time(b) * 1e-3
    # nuclear log-gradient (eq. 7's grad_alpha ln rho / 2) on the same walkers
    t_n = 0.0
    for k in range(3 + K_DERIV):
        a, b = ev(), ev()
        a.record(st)
        dR = sysh.nuclear_log_gradient(r_orb, d.n_atoms)
        b.record(st)
        torch.cuda.synchronize()
        if k >= 3:
            t_n += a.elapsed_time(b) * 1e-3
    # nuclear energy gradient (first term of eq. 7, explicit route) and the force estimator on the same walkers
    t_f = t_fr = 0.0
    lp_o, sg_o, el_o = sysh.local_energy(r_orb)
    for k in range(3 + K_DERIV):
        a, b, c = ev(), ev(), ev()
        a.record(st)
        dE = sysh.nuclear_energy_gradient(r_orb, d.n_atoms)
        b.record(st)
        F, Fterms = qb.force(el_o, dE, dR)
        c.record(st)
        torch.cuda.synchronize()
        if k >= 3:
            t_f += a.elapsed_time(b) * 1e-3
            t_fr += b.elapsed_time(c) * 1e-3
    # NEXT-3: the same wavefunction with the inverse backflow transformation (w = 0.05): E_L by the table-route
    # backflow kernel, log|Psi| and the sampler with the orbitals at the backflow coordinates
    import copy
    d_bf = copy.copy(d)
    d_bf.backflow_w = 0.05
    sys_bf = qb.QmcSystem(d_bf, device=local_rank)
    r_bf = r0.clone()
    t_b = [0.0, 0.0, 0.0, 0.0]
    O_bf = torch.empty((r_orb.shape[2], sys_bf.n_param()), dtype=torch.float64, device=dev)
    for k in range(3 + K_DERIV):
        e0_, e1_, e2_, e3_, e4_ = ev(), ev(), ev(), ev(), ev()
        e4_.record(st)
        sys_bf.log_derivatives(r_orb, lp_o, sg_o, el_o, O_bf)
        e0_.record(st)
        sys_bf.local_energy(r_orb, lp_o, sg_o, el_o)
        e1_.record(st)
        sys_bf.log_psi(r_bf, lp, sg)
        e2_.record(st)
        sys_bf.metropolis(r_bf, step_size, n_sweeps, seed, sweep_offset=k * n_sweeps, walker_offset=rank * M, logpsi=lp, sign=sg)
        e3_.record(st)
        torch.cuda.synchronize()
        if k >= 3:
            t_b[0] += e0_.elapsed_time(e1_) * 1e-3
            t_b[1] += e1_.elapsed_time(e2_) * 1e-3
            t_b[2] += e2_.elapsed_time(e3_) * 1e-3
            t_b[3] += e4_.elapsed_time(e0_) * 1e-3
    sys_bf.close()
    del O_bf
    del dC, dz, dR, dE, r_orb, r_bf

    t_met, t_el, t_all, t_e2e, t_kmain, t_kfb = max_over_ranks([t_met, t_el, t_all, t_e2e, t_kmain, t_kfb], device=dev)

    K = args.steps
    el_rate = world * M * K / t_el
    met_rate = world * M * n_sweeps * K / t_met
    e2e_rate = world * M * K / t_e2e
    flops_el, flops_st = sysh.model_flops(0), sysh.model_flops(1)
    achieved = flops_el * M * K / t_kmain / 1e12    # per GPU, the dominant kernel's own launch duration
    achieved_call = flops_el * M * K / t_el / 1e12  # the whole qmc_local_energy call (kernel + explicit fallback kernel)
    achieved_met = flops_st * M * n_sweeps * K / t_met / 1e12

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_sample = min(M, 8192 * cores)  # ~20-30 core-seconds of CPU work
        v, dt = oracle_sample(d, r_host, n_sample, cores)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"E_L of the first {n_sample} walkers of the same batch, {cores} threads, {dt:.1f} s"}

    if rank == 0:
        mean, err = recs[-1][4], recs[-1][5]
        line = {
            "metric": METRIC, "value": el_rate, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_all / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "walkers_per_gpu": M, "n_sweeps": n_sweeps, "step_bohr": step_size,
                       "l2": "flushed between steps (256 MB write, outside the event-timed regions)",
                       "timing": "CUDA events on torch's current stream around each call; sums over the K steps; max over ranks"},
            "metropolis": {"value": met_rate, "unit": "walker-steps/s", "ms_per_call": 1e3 * t_met / K,
                           "model_tflops": achieved_met, "frac": achieved_met / peak,
                           "frac_of_dfma_peak": achieved_met / peak_dfma,
                           "model_flop_eq_per_walker_step": flops_st},
            "local_energy_ms": 1e3 * t_el / K,
            # the dominant kernel of the timed step BY TIME is the sampler (one launch = 20 sweeps of M walkers, ~90 % of
            # the step: profiles/r02_launches.md); the fused E_L kernel that north_star's 50 % target names is reported
            # beside it, against the same peak
            "roofline": {"bound": "alu", "kernel": "metropolis_kernel<7,14> (one launch = 20 sweeps of 131072 walkers)",
                         "achieved": achieved_met, "peak": peak, "unit": "TFLOP/s", "frac": achieved_met / peak,
                         "kernel_ms": 1e3 * t_met / K,
                         "model_flop_eq_per_launch": flops_st * M * n_sweeps, "model_flop_eq_per_walker_step": flops_st,
                         "traffic": profile_traffic("r02_metro_kernel.md"),
                         "algorithmic_bytes_per_launch": int(M) * (2 * 3 * d.n_e * 8 + 16),
                         "timing": "CUDA events on the launching stream around the single-launch qmc_metropolis call, sum over the "
                                   "K timed steps",
                         "local_energy_kernel": {
                             "kernel": "local_energy_kernel<7,14,true>", "achieved": achieved, "frac": achieved / peak,
                             "kernel_ms": 1e3 * t_kmain / K, "fallback_kernel_ms": 1e3 * t_kfb / K,
                             "achieved_call": achieved_call, "frac_call": achieved_call / peak,
                             "frac_of_dfma_microbenchmark": achieved / peak_dfma,
                             "model_flop_eq_per_walker": flops_el, "traffic": profile_traffic("r02_el_kernel.md"),
                             "algorithmic_bytes_per_launch": int(M) * (3 * d.n_e * 8 + 24),
                             "timing": "kernel_ms: CUDA events recorded inside qmc_local_energy on the launching stream before and "
                                       "after the table-path kernel (qmc_set_kernel_timing), mean over a replay of the K steps "
                                       "(flush, sampler, E_L, statistics) right after the timed ones; *_call: events around the "
                                       "whole call in the K timed steps, which also runs the explicit fallback kernel"},
                         "peak_source": "max of the qmc_fp64_peak DFMA (8 chains), DFMA (two-register form) and DMMA m8n8k4 "
                                        "microbenchmarks measured in this process: one shared FP64 pipe (no FP64 entry in "
                                        "MEASURED_PEAKS.json)",
                         "dfma_peak": peak_dfma, "dfma_two_register_peak": peak_dfma2, "dfma_three_register_rate": peak_dfma3,
                         "dmma_peak": peak_dmma,
                         "dfma_dependent_latency_cycles": 64.0 * 4 * 148 * (clocks.get("sm_mhz") or 1965.0) * 1e6 / (rate_chain * 1e12),
                         # 148 SMs x 64 FP64 FMA/clk x 2 x the SM clock seen during the run
                         "peak_nominal": 148 * 64 * 2 * (clocks.get("sm_mhz") or 1965.0) * 1e-6},
            "cpu_baseline": cpu,
            "e2e": {"value": e2e_rate, "unit": UNIT, "h2d_bytes_per_step": int(r_pin.numel() * 8),
                    "d2h_bytes_per_step": int(out_pin.numel() * 8)},
            "e2e_vmc_step": {"ms": 1e3 * t_vmc / K, "walker_steps_per_s": world * M * n_sweeps / (t_vmc / K),
                             "walker_E_L_per_s": world * M / (t_vmc / K),
                             "h2d_bytes_per_step": int(r_pin.numel() * 8), "d2h_bytes_per_step": int(r_pin.numel() * 8 + M * 8),
                             "note": "qmc_vmc_step_host: one upload, 20 sweeps + E_L + statistics, walkers and E_L back; wall clock"},
            "log_derivatives": {"n_param": n_par, "ms_local_energy_plus_O": 1e3 * t_d / K_DERIV,
                                "ms_energy_gradient": 1e3 * t_g / K_DERIV, "O_bytes": int(M) * n_par * 8,
                                "gradient_hbm_gbs": int(M) * (n_par + 1) * 8 / (t_g / K_DERIV) / 1e9,
                                "E_v": e_v, "grad_norm": float(np.linalg.norm(grad)),
                                "ms_fused_local_energy_and_gradient": 1e3 * t_fu / K_DERIV,
                                "fused_over_plain_local_energy": (t_fu / K_DERIV) / (t_el / K),
                                "fused_grad_max_abs_diff": float(np.max(np.abs(grad_f - grad))),
                                "note": "SURVEY 8(f) NEXT-1, eq. 6; gradient time includes batch stats, the D2H of the result and a stream synchronise"},
            "orbital_derivatives": {"walkers": int(M_orb), "outputs_per_walker": int(d.n_ao * d.n_mo + d.n_ao),
                                    "ms": 1e3 * t_o / K_DERIV,
                                    "note": "SURVEY 8(f) NEXT-1: d ln Psi / d C and d ln Psi / d zeta per walker"},
            "nuclear_log_gradient": {"walkers": int(M_orb), "outputs_per_walker": int(3 * d.n_atoms),
                                     "ms": 1e3 * t_n / K_DERIV,
                                     "note": "SURVEY 8(f) NEXT-4, first half: grad_alpha ln|Psi| of eq. 7 per walker"},
            "nuclear_energy_gradient": {"walkers": int(M_orb), "outputs_per_walker": int(3 * d.n_atoms),
                                        "ms": 1e3 * t_f / K_DERIV, "ms_force_reduction": 1e3 * t_fr / K_DERIV,
                                        "F_z": [float(F[a_, 2]) for a_ in range(d.n_atoms)],
                                        "note": "SURVEY 8(f) NEXT-4: grad_alpha E_L per walker (weight matrices from the reference's "
                                                "tables, explicit route for groups with a near-singular reference) and the "
                                                "estimator of eq. 7; the walkers are not equilibrated here, so F is a throughput "
                                                "figure, not a physical force"},
            "backflow": {"w": 0.05, "ms_local_energy": 1e3 * t_b[0] / K_DERIV, "ms_log_derivatives": 1e3 * t_b[3] / K_DERIV, "walkers_local_energy": int(M_orb),
                         "ms_log_psi": 1e3 * t_b[1] / K_DERIV, "ms_metropolis": 1e3 * t_b[2] / K_DERIV, "walkers": int(M),
                         "walker_steps_per_s": world * M * n_sweeps / (t_b[2] / K_DERIV),
                         "note": "SURVEY 8(f) NEXT-3: inverse backflow K_BF = w/r; E_L from the reference's tables (F.6-F.9, "
                                 "explicit route for walkers with a nearly singular reference), values-only kernels on "
                                 "the excitation tables; ms_log_derivatives = E_L + the eq. 6 factors with the backflow "
                                 "weight as a parameter"},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "last_step": {"mean_E_L": mean, "stderr": err},
        }
        print(json.dumps(line))
    sysh.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
