"""A variational Monte Carlo optimisation loop on the GPU path (eq. 6), as an example of how the
calls fit together:

    python -m paper_2506_09743_b200.vmc_example [--config H2] [--walkers 65536] [--iterations 12]

Per iteration: equilibrate / decorrelate the walkers with qmc_metropolis, evaluate E_L and the logarithmic
derivatives O_p with qmc_log_derivatives, form the gradient estimator with qmc_energy_gradient, take one plain
gradient-descent step on the selected parameters and rebuild the handle (a qmc_system_t is immutable).  The paper
optimises with ADAM through PyTorch autograd; the optimiser is not part of the hot path, so this example keeps the
simplest one.  Optimised here: the Pade e-e parameter b and the three electron-nucleus parameters (the cusp
values a_par, a_anti stay fixed), for multi-determinant systems the CI coefficients, and with
--orbitals also the AO exponents zeta and the MO coefficients C (qmc_orbital_derivatives; the
paper finds the exponents the most rewarding parameters).  With --backflow W the wavefunction carries the
inverse backflow transformation and its weight is optimised with b and the CI coefficients.
There is no CPU fallback: without a GPU this raises.
"""
from __future__ import annotations

import argparse
import copy

import numpy as np
import torch

from . import binding as qb
from . import workloads as wl

N_JASTROW = 6  # (a_par, a_anti, b, en_w0, en_w1, en_w2) precede the CI coefficients in theta (no e-e-n terms here)


def get_theta(d):
    """theta in the order of qmc_log_derivatives; a backflow wavefunction carries its weight w as the last entry"""
    th = np.concatenate([[d.jastrow_a_par, d.jastrow_a_anti, d.jastrow_b, d.jastrow_en_w0, d.jastrow_en_w1,
                          d.jastrow_en_w2], np.asarray(d.ci_coeff, np.float64)])
    return np.append(th, d.backflow_w) if d.backflow_w != 0.0 else th


def set_theta(d, theta):
    d2 = copy.copy(d)
    (d2.jastrow_a_par, d2.jastrow_a_anti, d2.jastrow_b, d2.jastrow_en_w0, d2.jastrow_en_w1,
     d2.jastrow_en_w2) = (float(t) for t in theta[:N_JASTROW])
    n_det = len(d.ci_coeff)
    d2.ci_coeff = np.array(theta[N_JASTROW:N_JASTROW + n_det], np.float64)
    if d.backflow_w != 0.0:
        d2.backflow_w = float(theta[N_JASTROW + n_det]) or 1e-12   # (0 would switch the transformation off)
    return d2


def optimise(d, r_host, iterations=12, lr=0.2, sweeps=20, step=0.4, seed=1, optimise_ci=True, verbose=True,
             optimise_orbitals=False, lr_orbitals=0.05):
    """Returns the list of (E_v, standard error, gradient norm) per iteration and the final description."""
    if not torch.cuda.is_available():
        raise RuntimeError("vmc_example needs a CUDA device: the product path has no CPU fallback")
    r = torch.from_numpy(r_host).cuda()
    bf = d.backflow_w != 0.0
    mask = np.zeros(N_JASTROW + len(d.ci_coeff) + (1 if bf else 0), bool)
    mask[2:N_JASTROW] = True                      # b and the electron-nucleus kernel
    if optimise_ci and len(d.ci_coeff) > 1:
        mask[N_JASTROW + 1:N_JASTROW + len(d.ci_coeff)] = True   # d_0 fixes the normalisation
    if bf:                                        # backflow wavefunction: its weight is a parameter; this
        mask[3:N_JASTROW] = False                 # example then leaves the e-n kernel alone (b, CI and w move)
        mask[-1] = True
    history = []
    for it in range(iterations):
        s = qb.QmcSystem(d, 0)
        s.metropolis(r, step, sweeps, seed=seed, sweep_offset=it * sweeps)   # sample |Psi_theta|^2
        lp, sg, el, O = s.log_derivatives(r)
        e_v, grad = qb.energy_gradient(el, O)
        _, err = qb.batch_stats(el)
        history.append((e_v, err, float(np.linalg.norm(grad[mask]))))
        if verbose:
            print(f"iteration {it:2d}: E_v = {e_v:+.5f} +- {err:.5f} Ha   |grad| = {history[-1][2]:.4f}   "
                  f"b = {d.jastrow_b:.4f}  en = ({d.jastrow_en_w0:+.4f}, {d.jastrow_en_w1:+.4f}, {d.jastrow_en_w2:.4f})"
                  + (f"  backflow w = {d.backflow_w:+.4f}" if bf else ""))
        if optimise_orbitals:   # eq. 6 with O = d ln Psi / d C and d ln Psi / d zeta, same E_L
            dC, dz = s.orbital_derivatives(r, d.n_ao, d.n_mo)
            _, g_C = qb.energy_gradient(el, dC.view(dC.shape[0], -1))
            _, g_z = qb.energy_gradient(el, dz)
            d = copy.copy(d)
            d.mo_coeff = np.asarray(d.mo_coeff, np.float64) - lr_orbitals * g_C.reshape(d.n_ao, d.n_mo)
            d.ao_zeta = np.maximum(np.asarray(d.ao_zeta, np.float64) - lr_orbitals * g_z, 0.1)
            del dC, dz
        theta = get_theta(d)
        theta[mask] -= lr * grad[mask]
        theta[2] = max(theta[2], 0.05)            # keep the Pade denominators positive
        theta[5] = max(theta[5], 0.05)
        d = set_theta(d, theta)
        s.close()
    return history, d


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="H2", choices=sorted(wl.CONFIGS))
    ap.add_argument("--walkers", type=int, default=65536)
    ap.add_argument("--iterations", type=int, default=12)
    ap.add_argument("--lr", type=float, default=0.2)
    ap.add_argument("--orbitals", action="store_true", help="also optimise AO exponents and MO coefficients")
    ap.add_argument("--backflow", type=float, default=0.0, help="initial weight w of the inverse backflow kernel (0 = none)")
    args = ap.parse_args()
    d, r = wl.CONFIGS[args.config](M=args.walkers)
    d = copy.copy(d)
    d.jastrow_en_w2 = 1.0                          # the e-n kernel starts switched off (w0 = w1 = 0) with D = 1 + r
    d.backflow_w = args.backflow
    optimise(d, r, iterations=args.iterations, lr=args.lr, step=float(d.extra.get("step", 0.4)),
             optimise_orbitals=args.orbitals)


if __name__ == "__main__":
    main()
