"""All five BASELINE.json configurations on one GPU: absolute rates and the fraction of the FP64 roofline.

    python -m paper_2506_09743_b200.configs_report [--scan-geometries 16]

Per configuration: device time of qmc_local_energy (walker*E_L/s) and of qmc_metropolis with the
configuration's own sweep count and step (walker-steps/s), both as model FP64 TFLOP/s (qmc_model_flops) and as
a fraction of the FP64 peak measured in the same process (the largest of the DFMA and DMMA microbenchmarks of
qmc_fp64_peak: one pipe); the sampler + E_L pair is also timed as one captured CUDA graph (the way to run the
launch-bound small systems).  Configuration 5 (CO dissociation scan) runs its 50
sweeps with E_L after every sweep and reports mean E_L and its standard error per geometry (DESIGN.md reading
Q16: per-walker sweep average first, then the standard error over walkers; no burn-in is discarded -- this is a
throughput and parity benchmark, not a physics result).  CUDA events on the current stream around 10 back-to-back calls, 3 warm-ups,
best of 3 batches.  There is no CPU fallback: without a GPU this raises.
"""
from __future__ import annotations

import argparse
import copy

import torch

from . import binding as qb
from . import workloads as wl


def _time(fn, reps=10, warm=3):
    """mean device time of fn: `reps` calls enqueued back to back between two events (the host runs ahead,
    so launch latency is not part of the figure), best of 3 such batches"""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        best = min(best, a.elapsed_time(b) * 1e-3 / reps)
    return best


def measure(name, d, r_host, peak):
    s = qb.QmcSystem(d, 0)
    M = r_host.shape[2]
    r0 = torch.from_numpy(r_host).cuda()
    r = r0.clone()
    lp = torch.empty(M, dtype=torch.float64, device="cuda")
    sg, el = torch.empty_like(lp), torch.empty_like(lp)
    sweeps, step = int(d.extra.get("sweeps", 10)), float(d.extra.get("step", 0.3))
    s.metropolis(r, step, sweeps, seed=1, logpsi=lp, sign=sg)  # equilibrate a little: time E_L on sampled walkers
    t_el = _time(lambda: s.local_energy(r, lp, sg, el))

    def met():
        r.copy_(r0)
        s.metropolis(r, step, sweeps, seed=1, logpsi=lp, sign=sg)

    t_cp = _time(lambda: r.copy_(r0))
    t_met = _time(met) - t_cp
    # E_L + O_p (eq. 6 factors) and the orbital-parameter derivatives, on at most 32768 walkers
    Md = min(M, 32768)
    rd = r[:, :, :Md].contiguous()
    O = torch.empty((Md, s.n_param()), dtype=torch.float64, device="cuda")
    t_el_d = _time(lambda: s.local_energy(rd))
    t_O = _time(lambda: s.log_derivatives(rd, O=O))
    t_orb = _time(lambda: s.orbital_derivatives(rd, d.n_ao, d.n_mo))
    t_nuc = _time(lambda: s.nuclear_log_gradient(rd, d.n_atoms))
    t_frc = _time(lambda: s.nuclear_energy_gradient(rd, d.n_atoms))
    t_fuse = _time(lambda: s.local_energy_gradient(rd))
    # sampler + E_L as one CUDA graph (no allocation after the warm-up calls above), replayed back to back
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        s.metropolis(r, step, sweeps, seed=1, logpsi=lp, sign=sg, stream=st)
        s.local_energy(r, lp, sg, el, stream=st)
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        g.capture_begin()
        s.metropolis(r, step, sweeps, seed=1, logpsi=lp, sign=sg, stream=st)
        s.local_energy(r, lp, sg, el, stream=st)
        g.capture_end()
    torch.cuda.current_stream().wait_stream(st)
    t_graph = _time(lambda: g.replay())

    def eager_pair():
        s.metropolis(r, step, sweeps, seed=1, logpsi=lp, sign=sg)
        s.local_energy(r, lp, sg, el)

    t_pair = _time(eager_pair)
    f_el, f_st = s.model_flops(0), s.model_flops(1)
    row = dict(config=name, n_e=d.n_e, n_ao=d.n_ao, n_mo=d.n_mo, n_det=d.n_det, walkers=M, el_ms=1e3 * t_el, el_rate=M / t_el,
               el_tflops=f_el * M / t_el / 1e12, el_frac=f_el * M / t_el / 1e12 / peak, sweeps=sweeps,
               met_ms=1e3 * t_met, met_rate=M * sweeps / t_met, met_tflops=f_st * M * sweeps / t_met / 1e12,
               met_frac=f_st * M * sweeps / t_met / 1e12 / peak, deriv_walkers=Md, n_param=s.n_param(),
               el_d_ms=1e3 * t_el_d, O_ms=1e3 * t_O, orb_ms=1e3 * t_orb, nuc_ms=1e3 * t_nuc, frc_ms=1e3 * t_frc,
               fuse_ms=1e3 * t_fuse, graph_ms=1e3 * t_graph, pair_ms=1e3 * t_pair)
    s.close()
    return row


def fig11(walkers=32768, n_dets=(1, 4, 20, 100, 500)):
    """The comparison of PAPER.md:345-349 (Fig. 11): E_L through the excitation tables of the reference
    (F.6/F.7, qmc_local_energy) against every determinant eliminated on its own (qmc_local_energy_explicit),
    CO shape, as a function of the number of determinants."""
    out = []
    for nd in n_dets:
        d, r_host = wl.co(M=walkers, n_det=nd)
        s = qb.QmcSystem(d, 0)
        r = torch.from_numpy(r_host).cuda()
        s.metropolis(r, float(d.extra.get("step", 0.2)), 20, seed=1)
        lp = torch.empty(walkers, dtype=torch.float64, device="cuda")
        sg, el = torch.empty_like(lp), torch.empty_like(lp)
        t_tab = _time(lambda: s.local_energy(r, lp, sg, el))
        t_exp = _time(lambda: s.local_energy_explicit(r, lp, sg, el), reps=3, warm=1)
        s.close()
        # the same with the inverse backflow transformation (F.8/F.9 tables against every determinant explicit)
        d_bf = copy.copy(d)
        d_bf.backflow_w = 0.05
        s = qb.QmcSystem(d_bf, 0)
        t_btab = _time(lambda: s.local_energy(r, lp, sg, el), reps=5)
        t_bexp = _time(lambda: s.local_energy_explicit(r, lp, sg, el), reps=2, warm=1)
        s.close()
        out.append(dict(n_det=nd, walkers=walkers, tab_ms=1e3 * t_tab, exp_ms=1e3 * t_exp, btab_ms=1e3 * t_btab,
                        bexp_ms=1e3 * t_bexp))
    return out


def fig10(points=(1000, 32768)):
    """The workload of PAPER.md:313-321 (Fig. 10): the kinetic energy by the trace formulas on the four molecules,
    ground-state determinant only, with and without backflow.  Here: the whole E_L call (kinetic + potential)."""
    out = []
    for name in ("H2", "LiH", "Li2", "CO"):
        for M in points:
            d, r_host = wl.CONFIGS[name](M=M)
            d = copy.copy(d)
            d.det_up, d.det_dn, d.ci_coeff = d.det_up[:1], d.det_dn[:1], d.ci_coeff[:1]
            r = torch.from_numpy(r_host).cuda()
            lp = torch.empty(M, dtype=torch.float64, device="cuda")
            sg, el = torch.empty_like(lp), torch.empty_like(lp)
            row = dict(config=name, points=M)
            for key, w in (("plain_ms", 0.0), ("bf_ms", 0.05)):
                d.backflow_w = w
                s = qb.QmcSystem(d, 0)
                row[key] = 1e3 * _time(lambda: s.local_energy(r, lp, sg, el))
                s.close()
            out.append(row)
    return out


def scan(n_geom, peak):
    """BASELINE configs[4]: per geometry 50 sweeps with E_L after every sweep."""
    out = []
    t_total = 0.0
    for d, r_host in wl.co_scan(n_geom=n_geom):
        s = qb.QmcSystem(d, 0)
        M = r_host.shape[2]
        r = torch.from_numpy(r_host).cuda()
        sweeps, step = int(d.extra["sweeps"]), float(d.extra["step"])
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        res = s.metropolis(r, step, sweeps, seed=5, want_eloc_acc=True)
        mean, err = qb.batch_stats(res["eloc_acc"] / sweeps)
        b.record()
        torch.cuda.synchronize()
        t = a.elapsed_time(b) * 1e-3
        t_total += t
        flops = (s.model_flops(0) + s.model_flops(1)) * M * sweeps
        out.append(dict(R=float(d.extra["R"]), mean_E_L=mean, stderr=err, seconds=t, tflops=flops / t / 1e12,
                        frac=flops / t / 1e12 / peak, walkers=M, sweeps=sweeps))
        s.close()
    return out, t_total


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--scan-geometries", type=int, default=16)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("configs_report needs a CUDA device: the product path has no CPU fallback")
    peak = max(qb.fp64_peak(k, reps=5) for k in (0, 1, 3))
    rows = [measure("H2", *wl.h2(), peak), measure("LiH", *wl.lih(), peak), measure("Li2 (30 AOs)", *wl.li2(), peak),
            measure("Li2-28", *wl.li2(variant="28"), peak), measure("CO", *wl.co(), peak)]
    print(f"FP64 peak measured in this process (max of DFMA, two-register DFMA, DMMA): {peak:.1f} TFLOP/s")
    print("| config | N_e | N_AO | N_det | walkers | E_L call ms | M walker*E_L/s | model TFLOP/s | of peak | sweeps | "
          "Metropolis ms | M walker-steps/s | model TFLOP/s | of peak | sweeps + E_L eager ms | as one CUDA graph ms |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for x in rows:
        print(f"| {x['config']} | {x['n_e']} | {x['n_ao']} | {x['n_det']} | {x['walkers']} | {x['el_ms']:.3f} | "
              f"{x['el_rate'] / 1e6:.1f} | {x['el_tflops']:.2f} | {100 * x['el_frac']:.1f} % | {x['sweeps']} | "
              f"{x['met_ms']:.3f} | {x['met_rate'] / 1e6:.1f} | {x['met_tflops']:.2f} | {100 * x['met_frac']:.1f} % | "
              f"{x['pair_ms']:.3f} | {x['graph_ms']:.3f} |")
    print("\nParameter derivatives (eq. 6 factors), same sampled walkers, device time per call:")
    print("| config | walkers | E_L ms | n_param | E_L + O_p ms | E_L + fused eq. 6 gradient ms | orbital parameters (N_AO x N_MO + N_AO) | "
          "dC, dzeta ms | grad_R ln Psi ms | grad_R E_L ms |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for x in rows:
        print(f"| {x['config']} | {x['deriv_walkers']} | {x['el_d_ms']:.3f} | {x['n_param']} | {x['O_ms']:.3f} | {x['fuse_ms']:.3f} | "
              f"{x['n_ao']} x {x['n_mo']} + {x['n_ao']} | {x['orb_ms']:.3f} | {x['nuc_ms']:.3f} | {x['frc_ms']:.3f} |")
    print("\nAccelerated (excitation tables, F.6/F.7) vs explicit per-determinant E_L (PAPER.md:345-349, Fig. 11), CO shape:")
    print("| N_det | walkers | tables ms | explicit ms | explicit / tables | backflow: tables (F.8/F.9) ms | backflow: explicit ms | explicit / tables |")
    print("|---|---|---|---|---|---|---|---|")
    for x in fig11():
        print(f"| {x['n_det']} | {x['walkers']} | {x['tab_ms']:.3f} | {x['exp_ms']:.3f} | {x['exp_ms'] / x['tab_ms']:.1f} | "
              f"{x['btab_ms']:.3f} | {x['bexp_ms']:.3f} | {x['bexp_ms'] / x['btab_ms']:.1f} |")
    print("\nGround-state determinant only, with and without the inverse backflow (workload of PAPER.md:313-321, Fig. 10), "
          "E_L call, device time:")
    print("| config | points | E_L ms | E_L with backflow ms |")
    print("|---|---|---|---|")
    for x in fig10():
        print(f"| {x['config']} | {x['points']} | {x['plain_ms']:.4f} | {x['bf_ms']:.4f} |")
    if args.scan_geometries > 0:
        geo, t_total = scan(args.scan_geometries, peak)
        print(f"\nCO scan (500 determinants, {geo[0]['walkers']} walkers per geometry, {geo[0]['sweeps']} sweeps + E_L on every "
              f"sweep): {len(geo)} geometries in {t_total:.2f} s")
        print("| R (bohr) | mean E_L (Ha) | std error | seconds | model TFLOP/s | of peak |")
        print("|---|---|---|---|---|---|")
        for g in geo:
            print(f"| {g['R']:.2f} | {g['mean_E_L']:.5f} | {g['stderr']:.5f} | {g['seconds']:.3f} | {g['tflops']:.2f} | "
                  f"{100 * g['frac']:.1f} % |")


if __name__ == "__main__":
    main()
