"""Pins of the CPU oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) P1-P17).  CPU only."""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import binding as ob
from paper_2506_09743_b200 import workloads as wl
from tests.helpers import atom_system, hydrogenic_set, soa

GOLD = os.path.join(os.path.dirname(__file__), "golden")
rng0 = np.random.default_rng(12345)


def _rand_pos(M, n_e, scale=1.0, rmin=0.0, seed=0):
    rng = np.random.default_rng(seed)
    r = rng.standard_normal((M, n_e, 3)) * scale
    if rmin > 0:
        nrm = np.linalg.norm(r, axis=2, keepdims=True)
        r = r * np.maximum(nrm, rmin) / nrm
    return r


# closed-form values the paper / textbook quantum mechanics fix (tests/golden/cusp_and_hydrogenic.txt, with citations)
from tests.helpers import golden_values  # noqa: E402
GOLDEN = golden_values("cusp_and_hydrogenic.txt")


# ---------------------------------------------------------------- P1, P2
def test_P1_hydrogen_1s_exact():
    d = atom_system(1, [(1, 0, 0, 1.0)], [[1.0]], 1, 0)
    r = _rand_pos(200, 1, 2.0)
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    assert np.max(np.abs(el - GOLDEN["E_n1"])) < 1e-12
    # normalised 1s: psi = e^{-r}/sqrt(pi)
    rr = np.linalg.norm(r[:, 0], axis=1)
    assert np.max(np.abs(lp - (-rr - 0.5 * math.log(math.pi)))) < 1e-13
    assert np.all(sg == 1.0)


@pytest.mark.parametrize("Z,zeta", [(1, 0.8), (2, 1.7), (3, 3.4)])
def test_P2_hydrogenlike_wrong_zeta(Z, zeta):
    d = atom_system(Z, [(1, 0, 0, zeta)], [[1.0]], 1, 0, xyz=(0.3, -0.2, 0.5))
    r = _rand_pos(100, 1, 1.5, seed=1) + np.array([0.3, -0.2, 0.5])
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    rr = np.linalg.norm(r[:, 0] - np.array([0.3, -0.2, 0.5]), axis=1)
    ref = -zeta ** 2 / 2 + (zeta - Z) / rr
    assert np.max(np.abs(el - ref) / np.maximum(1, np.abs(ref))) < 1e-12


# ---------------------------------------------------------------- P3, P4
@pytest.mark.parametrize("Z", [1, 3])
def test_P3_hydrogenic_2p_3d_every_harmonic(Z):
    r = _rand_pos(50, 1, 3.0, rmin=0.05, seed=2)
    for m in range(3):
        d = atom_system(Z, [(2, 1, m, Z / 2)], [[1.0]], 1, 0)
        _, _, el = ob.local_energy(ob.OracleSystem(d), soa(r))
        assert np.max(np.abs(el - Z * Z * GOLDEN["E_n2"])) < 1e-11 * Z * Z
    for m in range(5):
        d = atom_system(Z, [(3, 2, m, Z / 3)], [[1.0]], 1, 0)
        _, _, el = ob.local_energy(ob.OracleSystem(d), soa(r))
        assert np.max(np.abs(el - Z * Z * GOLDEN["E_n3"])) < 1e-11 * Z * Z


@pytest.mark.parametrize("Z", [1, 2])
def test_P4_hydrogenic_2s_as_mo(Z):
    # psi_2s ~ (2 - Z r) e^{-Z r/2} = 2*[1s-type, zeta Z/2] - Z*[2s-type r e^{-Z r /2}]
    d = atom_system(Z, [(1, 0, 0, Z / 2), (2, 0, 0, Z / 2)], [[2.0], [-float(Z)]], 1, 0, norm=[1.0, 1.0])
    r = _rand_pos(100, 1, 3.0, rmin=0.05, seed=3)
    rr = np.linalg.norm(r[:, 0], axis=1)
    keep = np.abs(2 - Z * rr) > 1e-2  # away from the radial node
    _, _, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    assert np.max(np.abs(el[keep] + Z * Z / 8)) < 1e-10


def test_3s_type_radial_power_two():
    # k = 2 radial factor (3s-type AO r^2 e^{-zeta r}): E_L = -zeta^2/2 + (3 zeta - Z)/r - 3/r^2 ... closed form
    # lap(r^2 e^{-z r}) / (r^2 e^{-z r}) = z^2 - 2 z (k+1)/r + k(k+1)/r^2 with k=2
    Z, z = 1.0, 0.7
    d = atom_system(Z, [(3, 0, 0, z)], [[1.0]], 1, 0)
    r = _rand_pos(50, 1, 3.0, rmin=0.2, seed=4)
    rr = np.linalg.norm(r[:, 0], axis=1)
    ref = -0.5 * (z * z - 6 * z / rr + 6 / rr ** 2) - Z / rr
    _, _, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    assert np.max(np.abs(el - ref) / np.maximum(1, np.abs(ref))) < 1e-12


# ---------------------------------------------------------------- normalisation (Q2) by quadrature
@pytest.mark.parametrize("n,l,m,zeta", [(1, 0, 0, 1.24), (2, 0, 0, 0.9), (2, 1, 0, 1.3), (2, 1, 2, 2.0),
                                        (3, 2, 0, 1.1), (3, 2, 3, 0.8), (3, 2, 4, 1.7), (3, 2, 1, 1.0)])
def test_sto_normalisation_integrates_to_one(n, l, m, zeta):
    d = atom_system(1, [(n, l, m, zeta)], [[1.0]], 1, 0)
    o = ob.OracleSystem(d)
    # Gauss-Laguerre in r (weight e^{-2 zeta r} absorbed numerically), Gauss-Legendre x uniform in angles
    xr, wr = np.polynomial.laguerre.laggauss(40)
    rr = xr / (2 * zeta)
    wrr = wr * np.exp(xr) / (2 * zeta)
    ct, wct = np.polynomial.legendre.leggauss(16)
    nphi = 16
    ph = (np.arange(nphi) + 0.5) * 2 * math.pi / nphi
    tot = 0.0
    for ri, wi in zip(rr, wrr):
        for c, wc in zip(ct, wct):
            s = math.sqrt(1 - c * c)
            for p in ph:
                v = ob.ao_eval(o, 0, [ri * s * math.cos(p), ri * s * math.sin(p), ri * c])[0]
                tot += wi * wc * (2 * math.pi / nphi) * ri * ri * v * v
    assert abs(tot - 1.0) < 1e-9


def test_P15_h2_overlap_and_mo_coefficient():
    d, _ = wl.h2(M=4)
    o = ob.OracleSystem(d)
    # overlap of the two normalised 1s STOs by quadrature in prolate spheroidal coordinates
    R, zeta = 1.4, 1.24
    xm, wm = np.polynomial.laguerre.laggauss(40)  # mu = 1 + x/(zeta R)
    nu, wn = np.polynomial.legendre.leggauss(24)
    S = 0.0
    for x, w in zip(xm, wm):
        mu = 1 + x / (zeta * R)
        for v, wv in zip(nu, wn):
            rho = (R / 2) * math.sqrt((mu * mu - 1) * (1 - v * v))
            z = (R / 2) * mu * v
            fa = ob.ao_eval(o, 0, [rho, 0.0, z])[0]
            fb = ob.ao_eval(o, 1, [rho, 0.0, z])[0]
            jac = (R / 2) ** 3 * (mu * mu - v * v) * 2 * math.pi
            S += w * math.exp(x) / (zeta * R) * wv * jac * fa * fb
    assert abs(S - 0.65917696731845) < 1e-9
    assert abs(d.mo_coeff[0, 0] - 0.54895740413533) < 1e-12
    assert abs(d.extra["overlap"] - S) < 1e-9


# ---------------------------------------------------------------- P5, P6
@pytest.mark.parametrize("n", [2, 3, 4, 5, 6, 7])
def test_P5_same_spin_hydrogenic_determinant(n):
    Z = 2.0
    aos, C, e = hydrogenic_set(Z)
    d = atom_system(Z, aos, C[:, :n], n, 0, norm=np.ones(len(aos)))
    r = _rand_pos(40, n, 2.5, rmin=0.1, seed=10 + n)
    lp, sg, el, parts = ob.local_energy(ob.OracleSystem(d), soa(r), parts=True)
    vee = np.zeros(len(r))
    for i, j in itertools.combinations(range(n), 2):
        vee += 1 / np.linalg.norm(r[:, i] - r[:, j], axis=1)
    ref = e[:n].sum() + vee
    ok = lp > np.max(lp) - 25  # drop walkers sitting on a node
    assert ok.sum() > 20
    assert np.max(np.abs(el[ok] - ref[ok]) / np.maximum(1, np.abs(ref[ok]))) < 1e-9
    assert np.allclose(parts[:, 1], vee, rtol=1e-13)


def test_P5_both_spins():
    Z = 3.0
    aos, C, e = hydrogenic_set(Z)
    d = atom_system(Z, aos, C[:, :5], 3, 2, norm=np.ones(len(aos)),
                    det_up=[[0, 2, 4]], det_dn=[[1, 3]])
    r = _rand_pos(40, 5, 1.5, rmin=0.1, seed=20)
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    vee = sum(1 / np.linalg.norm(r[:, i] - r[:, j], axis=1) for i, j in itertools.combinations(range(5), 2))
    ref = e[[0, 2, 4]].sum() + e[[1, 3]].sum() + vee
    ok = lp > np.max(lp) - 25
    assert np.max(np.abs(el[ok] - ref[ok]) / np.maximum(1, np.abs(ref[ok]))) < 1e-9


def test_P6_ci_degenerate_and_nondegenerate():
    Z = 2.0
    aos, C, e = hydrogenic_set(Z)
    # MOs: 0 1s, 1 2s, 2 2px, 3 2py, 4 2pz, 5 3dxy, 6 3dz2 ...
    # reference up = (1s, 2px), dn = (1s); substitutions 2px->2py, 2px->2pz (degenerate), weights arbitrary
    det_up = [[0, 2], [0, 3], [0, 4]]
    det_dn = [[0], [0], [0]]
    ci = [0.7, -0.4, 0.55]
    d = atom_system(Z, aos, C[:, :7], 2, 1, det_up=det_up, det_dn=det_dn, ci=ci, norm=np.ones(len(aos)))
    r = _rand_pos(60, 3, 1.5, rmin=0.1, seed=21)
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    vee = sum(1 / np.linalg.norm(r[:, i] - r[:, j], axis=1) for i, j in itertools.combinations(range(3), 2))
    ref = (e[0] + e[2] + e[0]) + vee
    ok = lp > np.max(lp) - 25
    assert np.max(np.abs(el[ok] - ref[ok]) / np.maximum(1, np.abs(ref[ok]))) < 1e-9
    # non-degenerate: E_L = sum d_n D_n E_n / sum d_n D_n + V_ee with D_n from single-determinant runs
    det_up = [[0, 2], [1, 2], [0, 5], [5, 6]]
    det_dn = [[0], [0], [1], [0]]
    ci = [0.8, 0.3, -0.5, 0.25]
    En = [e[0] + e[2] + e[0], e[1] + e[2] + e[0], e[0] + e[5] + e[1], e[5] + e[6] + e[0]]
    d = atom_system(Z, aos, C[:, :7], 2, 1, det_up=det_up, det_dn=det_dn, ci=ci, norm=np.ones(len(aos)))
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    num = np.zeros(len(r)); den = np.zeros(len(r))
    for k in range(4):
        dk = atom_system(Z, aos, C[:, :7], 2, 1, det_up=[det_up[k]], det_dn=[det_dn[k]], norm=np.ones(len(aos)))
        lpk, sgk, _ = ob.local_energy(ob.OracleSystem(dk), soa(r))
        Dk = sgk * np.exp(lpk)
        num += ci[k] * Dk * En[k]; den += ci[k] * Dk
    ref = num / den + vee
    ok = np.abs(den) > 1e-3 * np.max(np.abs(den))
    assert np.max(np.abs(el[ok] - ref[ok]) / np.maximum(1, np.abs(ref[ok]))) < 1e-8


# ---------------------------------------------------------------- P7
@pytest.mark.parametrize("a,b", [(0.5, 1.0), (0.37, 0.6)])
def test_P7_helium_like_with_pade_closed_form(a, b):
    Z, zeta = 2.0, 1.6875
    d = atom_system(Z, [(1, 0, 0, zeta)], [[1.0]], 1, 1, a_par=0.25, a_anti=a, b=b)
    r = _rand_pos(200, 2, 1.0, rmin=0.05, seed=30)
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(r))
    r1, r2 = r[:, 0], r[:, 1]
    n1, n2 = np.linalg.norm(r1, axis=1), np.linalg.norm(r2, axis=1)
    d12 = r1 - r2
    r12 = np.linalg.norm(d12, axis=1)
    den = 1 + b * r12
    u = a * r12 / den; u1 = a / den ** 2; u2 = -2 * a * b / den ** 3
    hat = np.einsum("ij,ij->i", d12 / r12[:, None], r1 / n1[:, None] - r2 / n2[:, None])
    ref = -zeta ** 2 + (zeta - Z) * (1 / n1 + 1 / n2) + 1 / r12 - (u2 + 2 * u1 / r12) - u1 ** 2 + zeta * u1 * hat
    assert np.max(np.abs(el - ref) / np.maximum(1, np.abs(ref))) < 1e-12
    # log psi = 2 log N - zeta (r1+r2) + u
    N = zeta ** 1.5 / math.sqrt(math.pi)
    assert np.max(np.abs(lp - (2 * math.log(N) - zeta * (n1 + n2) + u))) < 1e-12


def test_parallel_spin_jastrow_uses_a_par():
    # two same-spin electrons in 1s / 2pz hydrogenic orbitals; changing a_anti must not matter, a_par must
    Z = 1.0
    aos, C, e = hydrogenic_set(Z)
    r = _rand_pos(10, 2, 2.0, rmin=0.2, seed=31)
    out = []
    for ap, aa in [(0.25, 0.5), (0.25, 0.9), (0.4, 0.5)]:
        d = atom_system(Z, aos, C[:, [0, 4]], 2, 0, norm=np.ones(len(aos)), a_par=ap, a_anti=aa)
        out.append(ob.local_energy(ob.OracleSystem(d), soa(r))[2])
    assert np.allclose(out[0], out[1], rtol=0, atol=0)
    assert np.max(np.abs(out[0] - out[2])) > 1e-3


# ---------------------------------------------------------------- P8 finite differences
def _fd_check(d, r_soa, h=1e-4, nwalk=6, tol=1e-6):
    o = ob.OracleSystem(d)
    lp, sg, el, parts = ob.local_energy(o, r_soa, parts=True)
    n_e = d.n_e
    worst = 0.0
    for w in range(nwalk):
        r = r_soa[:, :, w].copy()  # [n_e,3]
        psi0 = ob.psi_plain(o, r)
        assert abs(math.log(abs(psi0)) - lp[w]) < 1e-11 and np.sign(psi0) == sg[w]

        def lap(hh):
            tot, scale = 0.0, 0.0
            for i in range(n_e):
                acc = 0.0
                for c in range(3):
                    rp = r.copy(); rp[i, c] += hh
                    rm = r.copy(); rm[i, c] -= hh
                    acc += (ob.psi_plain(o, rp) - 2 * psi0 + ob.psi_plain(o, rm)) / (hh * hh)
                tot += acc / psi0
                scale += abs(acc / psi0)
            return tot, scale
        l1, scale = lap(h)
        l2, _ = lap(h / 2)
        rich = (4 * l2 - l1) / 3  # Richardson: removes the h^2 truncation term
        kin_fd = -0.5 * rich
        err = abs(kin_fd - parts[w, 0]) / max(1.0, scale)
        worst = max(worst, err)
    assert worst < tol, worst


def _keep_away(d, r_soa, rmin=0.3):
    """walkers whose electrons are all >= rmin from every nucleus (Q17)"""
    r = r_soa.transpose(2, 0, 1)  # [M,n_e,3]
    dist = np.linalg.norm(r[:, :, None, :] - d.atom_xyz[None, None], axis=3)
    return np.where(dist.min(axis=(1, 2)) > rmin)[0]


@pytest.mark.parametrize("name", ["H2", "LiH", "Li2", "CO"])
def test_P8_finite_differences_configs(name):
    d, r = wl.CONFIGS[name](M=64)
    o = ob.OracleSystem(d)
    lp, _, _ = ob.local_energy(o, r)
    idx = _keep_away(d, r)
    idx = idx[np.argsort(-lp[idx])][:4]  # well away from nodes
    _fd_check(d, np.ascontiguousarray(r[:, :, idx]), nwalk=len(idx), tol=2e-6)


def test_P8_ao_derivatives_vs_fd():
    d, _ = wl.co(M=2)
    o = ob.OracleSystem(d)
    rng = np.random.default_rng(5)
    h = 1e-4
    for ao in range(d.n_ao):
        a = d.ao_atom[ao]
        x = d.atom_xyz[a] + rng.standard_normal(3) * 0.6 + 0.35
        v = ob.ao_eval(o, ao, x)
        g = np.zeros(3); lap = 0.0
        for c in range(3):
            e = np.zeros(3); e[c] = h
            p, m = ob.ao_eval(o, ao, x + e)[0], ob.ao_eval(o, ao, x - e)[0]
            p2, m2 = ob.ao_eval(o, ao, x + e / 2)[0], ob.ao_eval(o, ao, x - e / 2)[0]
            g1, g2 = (p - m) / (2 * h), (p2 - m2) / h
            g[c] = (4 * g2 - g1) / 3
            l1, l2 = (p - 2 * v[0] + m) / h ** 2, (p2 - 2 * v[0] + m2) / (h / 2) ** 2
            lap += (4 * l2 - l1) / 3
        sc = max(1.0, abs(v[0]) * d.ao_zeta[ao] ** 2)
        assert np.max(np.abs(g - v[1:4])) < 1e-7 * sc, (ao, g, v)
        assert abs(lap - v[4]) < 2e-6 * sc, (ao, lap, v[4])


# ---------------------------------------------------------------- P9 antisymmetry
@pytest.mark.parametrize("name", ["LiH", "Li2", "CO"])
def test_P9_same_spin_exchange(name):
    d, r = wl.CONFIGS[name](M=32)
    o = ob.OracleSystem(d)
    lp, sg, el = ob.local_energy(o, r)
    for (i, j) in [(0, 1), (d.n_up, d.n_up + 1)]:
        r2 = r.copy()
        r2[[i, j]] = r2[[j, i]]
        lp2, sg2, el2 = ob.local_energy(o, r2)
        assert np.all(sg2 == -sg)
        assert np.max(np.abs(lp2 - lp)) < 1e-11
        assert np.max(np.abs(el2 - el) / np.maximum(1, np.abs(el))) < 1e-9
    # opposite-spin exchange is NOT a symmetry of the spin-assigned function
    r3 = r.copy(); r3[[0, d.n_up]] = r3[[d.n_up, 0]]
    lp3, _, _ = ob.local_energy(o, r3)
    assert np.max(np.abs(lp3 - lp)) > 1e-3


def test_pauli_zero_at_same_spin_coalescence():
    # the wave function vanishes when two same-spin electrons coincide
    d, r = wl.li2(M=4)
    o = ob.OracleSystem(d)
    base = ob.local_energy(o, r)[0]
    r2 = r.copy(); r2[1] = r2[0] + 1e-9
    lp2 = ob.local_energy(o, r2)[0]
    assert np.all(lp2 < base - 12)


# ---------------------------------------------------------------- P10 Leibniz
def _leibniz(A):
    n = A.shape[0]
    tot = 0.0
    for perm in itertools.permutations(range(n)):
        sgn = 1
        for i in range(n):
            for j in range(i + 1, n):
                if perm[i] > perm[j]:
                    sgn = -sgn
        p = 1.0
        for i in range(n):
            p *= A[i, perm[i]]
        tot += sgn * p
    return tot


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_P10_determinant_vs_permutation_sum(n):
    rng = np.random.default_rng(n)
    for _ in range(10):
        A = rng.standard_normal((n, n))
        dd, inv = ob.det_inv(A)
        ref = _leibniz(A)
        assert abs(dd - ref) < 1e-13 * max(1.0, abs(ref))
        assert np.max(np.abs(inv @ A - np.eye(n))) < 1e-11
    # a matrix that needs pivoting (zero leading element)
    A = rng.standard_normal((n, n)); A[0, 0] = 0.0
    if n > 1:
        assert abs(ob.det_inv(A)[0] - _leibniz(A)) < 1e-13


# ---------------------------------------------------------------- P11 nuclear repulsion
def test_P11_nuclear_repulsion():
    for fn, ref in [(wl.h2, 1 / 1.4), (wl.lih, 3 / 3.015), (wl.li2, 9 / 5.051), (wl.co, 48 / 2.132)]:
        d, r = fn(M=2)
        parts = ob.local_energy(ob.OracleSystem(d), r, parts=True)[3]
        assert np.max(np.abs(parts[:, 3] - ref)) < 1e-14 * max(1, ref)
    assert abs(1 / 1.4 - 0.7142857142857143) < 1e-15


def test_potential_terms_brute_force():
    d, r = wl.co(M=8)
    parts = ob.local_energy(ob.OracleSystem(d), r, parts=True)[3]
    rr = r.transpose(2, 0, 1)
    for w in range(8):
        ven = -sum(d.atom_Z[a] / np.linalg.norm(rr[w, i] - d.atom_xyz[a]) for i in range(14) for a in range(2))
        vee = sum(1 / np.linalg.norm(rr[w, i] - rr[w, j]) for i in range(14) for j in range(i))
        assert abs(parts[w, 2] - ven) < 1e-12 * abs(ven) and abs(parts[w, 1] - vee) < 1e-12 * abs(vee)


# ---------------------------------------------------------------- P12 cusps
def test_P12_electron_electron_cusp_finite():
    Z, zeta = 2.0, 1.7
    out = {}
    for label, a in [("exact", GOLDEN["cusp_antiparallel"]), ("off", 0.4)]:
        d = atom_system(Z, [(1, 0, 0, zeta)], [[1.0]], 1, 1, a_anti=a, b=1.0)
        o = ob.OracleSystem(d)
        vals = []
        for eps in [1e-2, 1e-3, 1e-4, 1e-5, 1e-6]:
            r = np.array([[[0.4, 0.3, 0.2], [0.4 + eps, 0.3, 0.2]]])
            vals.append(ob.local_energy(o, soa(r))[2][0])
        out[label] = np.array(vals)
    assert np.all(np.abs(out["exact"]) < 50)
    assert abs(out["exact"][-1] - out["exact"][-2]) < 1e-3  # converges
    # perturbed cusp diverges like (1 - 2a)/r
    assert abs(out["off"][-1] - (1 - 2 * 0.4) / 1e-6) < 0.01 * (0.2 / 1e-6)
    # parallel spins (a = 1/4): antisymmetric pair 1s/2pz
    aos, C, e = hydrogenic_set(1.0)
    for a, finite in [(GOLDEN["cusp_parallel"], True), (0.15, False)]:
        d = atom_system(1.0, aos, C[:, [0, 4]], 2, 0, norm=np.ones(len(aos)), a_par=a)
        o = ob.OracleSystem(d)
        vals = [ob.local_energy(o, soa(np.array([[[0.4, 0.3, 0.2], [0.4, 0.3, 0.2 + eps]]])))[2][0]
                for eps in [1e-3, 1e-4, 1e-5]]
        if finite:
            assert max(abs(v) for v in vals) < 50 and abs(vals[-1] - vals[-2]) < 1e-2
        else:
            assert abs(vals[-1] - (1 - 4 * a) / 1e-5) < 0.02 * (1 - 4 * a) / 1e-5


def test_electron_nucleus_cusp_finite_energy():
    # STOs give finite E_L at electron-nucleus coalescence when zeta = Z (1s)
    d = atom_system(3.0, [(1, 0, 0, 3.0)], [[1.0]], 1, 0)
    o = ob.OracleSystem(d)
    vals = [ob.local_energy(o, soa(np.array([[[eps, 0, 0]]])))[2][0] for eps in [1e-2, 1e-4, 1e-6]]
    assert np.max(np.abs(np.array(vals) + 4.5)) < 1e-9


# ---------------------------------------------------------------- P13 SD enumerator
def test_P13_sd_counts_match_paper():
    rows = [l.split() for l in open(os.path.join(GOLD, "sd_counts.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 5
    for n_el, n_orb, n_det in rows:
        assert wl.sd_count(int(n_el), int(n_orb)) == int(n_det)


def test_selected_determinants_structure():
    for fn, nd in [(wl.li2, 20), (wl.co, 100)]:
        d, _ = fn(M=2)
        assert d.det_up.shape == (nd, d.n_up)
        ref = np.arange(d.n_up)
        seen = set()
        ks = set()
        for n in range(nd):
            key = (tuple(d.det_up[n]), tuple(d.det_dn[n]))
            assert key not in seen
            seen.add(key)
            for lst in key:
                assert len(set(lst)) == len(lst) and max(lst) < d.n_mo
            ks.add((int((d.det_up[n] != ref).sum()), int((d.det_dn[n] != ref).sum())))
        assert ks == {(0, 0), (1, 0), (0, 1), (1, 1), (2, 0), (0, 2)}


# ---------------------------------------------------------------- P14 identities behind the fast path
def test_P14_trace_identities_random_matrices():
    rng = np.random.default_rng(7)
    n, nv = 6, 5
    for trial in range(20):
        A0 = rng.standard_normal((n, n)); Av = rng.standard_normal((n, nv))
        B0 = rng.standard_normal((n, n)); Bv = rng.standard_normal((n, nv))
        k = 1 + trial % 3
        p = rng.choice(n, k, replace=False); q = rng.choice(nv, k, replace=False)
        AX, BX = A0.copy(), B0.copy()
        AX[:, p] = Av[:, q]; BX[:, p] = Bv[:, q]
        d0, A0i = ob.det_inv(A0)
        dX, AXi = ob.det_inv(AX)
        T = A0i @ Av
        Mtab = A0i @ Bv - (A0i @ B0) @ T
        Tpq = T[np.ix_(p, q)]
        # reading Q8: D_X / D_0 = det T[p,q]
        assert abs(dX / d0 - np.linalg.det(Tpq)) < 1e-10 * max(1, abs(dX / d0))
        # F.6 / F.7 in table form
        lhs = np.trace(AXi @ BX)
        rhs = np.trace(A0i @ B0) + np.trace(np.linalg.inv(Tpq) @ Mtab[np.ix_(p, q)])
        assert abs(lhs - rhs) < 1e-9 * max(1, abs(lhs))
        # H.10
        P = np.zeros((n, n)); P[p, p] = 1
        W = A0i @ AX
        Tm = np.zeros((n, n)); Tm[np.ix_(p, p)] = np.linalg.inv(W[np.ix_(p, p)])
        assert np.max(np.abs(AXi - (A0i - (W - np.eye(n)) @ Tm @ A0i))) < 1e-8
    # G.5 / G.6: row-local derivative => (Tr)^2 = Tr(()^2)
    A = rng.standard_normal((n, n)); Ai = np.linalg.inv(A)
    dA = np.zeros((n, n)); dA[2] = rng.standard_normal(n)
    X = Ai @ dA
    assert abs(np.trace(X) ** 2 - np.trace(X @ X)) < 1e-12


# ---------------------------------------------------------------- P16 Philox + normals
def test_P16_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    for row in rows:
        v = [int(x, 16) for x in row]
        out = ob.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_P16_uniform_mapping_and_counter_layout():
    # walker_draws must be Philox(ctr=(w, sweep, j, 0), key=(seed lo, seed hi)) + the stated 53-bit mapping
    seed, w, sweep = 0x123456789ABCDEF0, 77, 5
    z, u = ob.walker_draws(seed, w, sweep, 6)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for j in range(3):
        x = [int(t) for t in ob.philox([w, sweep, j, 0], key)]
        u1 = (((x[0] << 32 | x[1]) >> 11) + 0.5) * 2.0 ** -53
        u2 = (((x[2] << 32 | x[3]) >> 11) + 0.5) * 2.0 ** -53
        rho = math.sqrt(-2 * math.log(u1))
        assert abs(z[2 * j] - rho * math.cos(2 * math.pi * u2)) < 1e-15 * max(1, rho)
        assert abs(z[2 * j + 1] - rho * math.sin(2 * math.pi * u2)) < 1e-15 * max(1, rho)
    x = [int(t) for t in ob.philox([w, sweep, 0xFFFFFFFF, 0], key)]
    assert u == (((x[0] << 32 | x[1]) >> 11) + 0.5) * 2.0 ** -53
    assert 0.0 < u < 1.0


def test_P16_normal_moments_and_ks():
    from scipy import stats
    zs = np.concatenate([ob.walker_draws(42, w, s, 42)[0] for w in range(400) for s in range(3)])
    assert abs(zs.mean()) < 4 / math.sqrt(len(zs))
    assert abs(zs.var() - 1) < 0.03
    assert stats.kstest(zs, "norm").pvalue > 1e-3
    us = np.array([ob.walker_draws(42, w, 0, 2)[1] for w in range(4000)])
    assert stats.kstest(us, "uniform").pvalue > 1e-3


# ---------------------------------------------------------------- P17 sampler sanity
def test_P17_metropolis_hydrogen_atom():
    d = atom_system(1, [(1, 0, 0, 1.0)], [[1.0]], 1, 0)
    o = ob.OracleSystem(d)
    M = 6000
    r0 = soa(np.random.default_rng(3).standard_normal((M, 1, 3)))
    out = ob.metropolis(o, r0, 0.5, 150, seed=9, threads=8)
    rr = np.linalg.norm(out["r"][0], axis=0)
    assert abs(rr.mean() - 1.5) < 0.05          # <r> of the 1s density
    assert abs((rr ** 2).mean() - 3.0) < 0.2    # <r^2> = 3
    acc = out["accept"].mean()
    assert 0.3 < acc < 0.95
    # decisions are exactly the sign of the margin
    assert np.array_equal(out["accept"] == 1, out["margin"] > 0)
    lp, sg, el = ob.local_energy(o, out["r"])
    assert np.max(np.abs(el + 0.5)) < 1e-12 and np.max(np.abs(lp - out["logpsi"])) < 1e-13


def test_metropolis_resumable_and_partition_independent():
    d, r = wl.lih(M=64)
    o = ob.OracleSystem(d)
    a = ob.metropolis(o, r, 0.3, 6, seed=11)
    b1 = ob.metropolis(o, r, 0.3, 2, seed=11, sweep_offset=0)
    b2 = ob.metropolis(o, b1["r"], 0.3, 4, seed=11, sweep_offset=2, threads=3)
    assert np.array_equal(a["r"], b2["r"]) and np.array_equal(a["accept"][2:], b2["accept"])
    assert np.array_equal(a["logpsi"], b2["logpsi"])


def test_metropolis_eloc_acc():
    d, r = wl.lih(M=16)
    o = ob.OracleSystem(d)
    out1 = ob.metropolis(o, r, 0.3, 1, seed=5, want_eloc_acc=True)
    el = ob.local_energy(o, out1["r"])[2]
    assert np.allclose(out1["eloc_acc"], el, rtol=1e-14)


def test_batch_stats():
    x = np.random.default_rng(1).standard_normal(10001) * 3 + 1e6
    m, s = ob.batch_stats(x)
    assert abs(m - math.fsum(x) / len(x)) < 1e-9
    assert abs(s - x.std(ddof=1) / math.sqrt(len(x))) < 1e-12


# ---------------------------------------------------------------- parameter derivatives (eq. 6)
def _with_param(d, p, value):
    """copy of the system with parameter p of theta = (a_par, a_anti, b, en_w0, en_w1, en_w2, d_0 ...) set to value"""
    import copy
    d2 = copy.copy(d)
    if p == 0:
        d2.jastrow_a_par = value
    elif p == 1:
        d2.jastrow_a_anti = value
    elif p == 2:
        d2.jastrow_b = value
    elif p == 3:
        d2.jastrow_en_w0 = value
    elif p == 4:
        d2.jastrow_en_w1 = value
    elif p == 5:
        d2.jastrow_en_w2 = value
    else:
        ci = np.array(d.ci_coeff, np.float64, copy=True)
        ci[p - NJ] = value
        d2.ci_coeff = ci
    return d2


NJ = 6  # Jastrow parameters ahead of the CI coefficients


def _param(d, p):
    jp = [d.jastrow_a_par, d.jastrow_a_anti, d.jastrow_b, d.jastrow_en_w0, d.jastrow_en_w1, d.jastrow_en_w2]
    return jp[p] if p < NJ else float(d.ci_coeff[p - NJ])


@pytest.mark.parametrize("name,M", [("H2", 12), ("LiH", 10), ("Li2", 8), ("CO", 5)])
def test_log_derivatives_vs_central_differences_of_log_psi(name, M):
    # the oracle's O_p against central differences of its own log|Psi| in EVERY parameter
    # (Richardson h, h/2): pins sign, pair bookkeeping (which a), the b derivative and D_n / Sigma
    d, r = wl.CONFIGS[name](M=M)
    d = _with_en(d, 0.35, -0.04, 0.9)  # all six Jastrow parameters active
    O = ob.log_derivatives(ob.OracleSystem(d), r)
    assert O.shape == (M, NJ + len(d.ci_coeff))
    params = list(range(NJ)) + list(range(NJ, O.shape[1], max(1, (O.shape[1] - NJ) // 7)))
    for p in params:
        t0 = _param(d, p)

        def cd(h):
            lp_p = ob.local_energy(ob.OracleSystem(_with_param(d, p, t0 + h)), r)[0]
            lp_m = ob.local_energy(ob.OracleSystem(_with_param(d, p, t0 - h)), r)[0]
            return (lp_p - lp_m) / (2 * h)

        h = 1e-3 * max(1.0, abs(t0)) if p < NJ else 1e-3 * max(abs(t0), 1e-2)
        fd = (4 * cd(h / 2) - cd(h)) / 3
        assert np.max(np.abs(O[:, p] - fd) / np.maximum(1, np.abs(fd))) < 1e-7, (name, p)


def test_log_derivatives_sum_rule_and_helium_closed_form():
    # sum_n d_n O_n = 1 (Sigma is linear in d)
    d, r = wl.li2(M=20)
    O = ob.log_derivatives(ob.OracleSystem(d), r)
    assert np.max(np.abs(O[:, NJ:] @ np.asarray(d.ci_coeff) - 1.0)) < 1e-11
    # He-like 1s^2 + Pade: O_a_anti = r12/(1+b r12), O_b = -a r12^2/(1+b r12)^2, O_a_par = 0, O_d0 = 1/d0
    a, b = 0.37, 0.6
    d = atom_system(2.0, [(1, 0, 0, 1.6875)], [[1.0]], 1, 1, a_par=0.25, a_anti=a, b=b, ci=[0.8])
    rr = _rand_pos(50, 2, 1.0, rmin=0.05, seed=77)
    O = ob.log_derivatives(ob.OracleSystem(d), soa(rr))
    r12 = np.linalg.norm(rr[:, 0] - rr[:, 1], axis=1)
    assert np.max(np.abs(O[:, 0])) == 0.0
    assert np.max(np.abs(O[:, 1] - r12 / (1 + b * r12))) < 1e-14
    assert np.max(np.abs(O[:, 2] + a * r12 ** 2 / (1 + b * r12) ** 2)) < 1e-14
    assert np.max(np.abs(O[:, NJ] - 1 / 0.8)) < 1e-13
    # e-n kernel switched off (w = 0): dK/dw0 = r, dK/dw1 = r^2, dK/dw2 = 0 summed over both electrons
    n1, n2 = np.linalg.norm(rr[:, 0], axis=1), np.linalg.norm(rr[:, 1], axis=1)
    assert np.max(np.abs(O[:, 3] - (n1 + n2))) < 1e-13 and np.max(np.abs(O[:, 4] - (n1 ** 2 + n2 ** 2))) < 1e-13
    assert np.max(np.abs(O[:, 5])) == 0.0
    # three same-spin electrons: only a_par pairs contribute
    aos, C, e = hydrogenic_set(1.0)
    d = atom_system(1.0, aos, C[:, [0, 2, 4]], 3, 0, norm=np.ones(len(aos)), a_par=0.25, a_anti=0.5, b=0.9)
    rr = _rand_pos(20, 3, 2.0, rmin=0.2, seed=78)
    O = ob.log_derivatives(ob.OracleSystem(d), soa(rr))
    s = sum(np.linalg.norm(rr[:, i] - rr[:, j], axis=1) / (1 + 0.9 * np.linalg.norm(rr[:, i] - rr[:, j], axis=1))
            for i in range(3) for j in range(i))
    assert np.max(np.abs(O[:, 0] - s)) < 1e-13 and np.max(np.abs(O[:, 1])) == 0.0


def test_energy_gradient_estimator():
    rng = np.random.default_rng(5)
    M, n_p = 1000, 7
    e = rng.standard_normal(M) * 3 - 10
    O = rng.standard_normal((M, n_p))
    ev, g = ob.energy_gradient(e, O)
    assert abs(ev - math.fsum(e) / M) < 1e-13
    ref = np.array([2 * math.fsum(O[:, p] * (e - math.fsum(e) / M)) / M for p in range(n_p)])
    assert np.max(np.abs(g - ref)) < 1e-13
    # an exact eigenfunction has E_L constant, so the estimator vanishes identically whatever O is (eq. 6):
    # hydrogen atom, exact 1s, two "determinants" that are the same orbital
    d = atom_system(1, [(1, 0, 0, 1.0)], [[1.0]], 1, 0, det_up=[[0], [0]], det_dn=np.zeros((2, 0), np.int32), ci=[0.7, 0.2])
    r = soa(_rand_pos(64, 1, 2.0, rmin=0.1, seed=6))
    o = ob.OracleSystem(d)
    el = ob.local_energy(o, r)[2]
    ev, g = ob.energy_gradient(el, ob.log_derivatives(o, r))
    assert abs(ev + 0.5) < 1e-12 and np.max(np.abs(g)) < 1e-11


def test_energy_gradient_estimator_reproduces_dE_dzeta_of_the_hydrogen_atom():
    # Physical pin of eq. 6's prefactor 2/M and sign: hydrogen atom, trial function N e^{-zeta r}:
    #   E(zeta) = zeta^2/2 - zeta  =>  dE/dzeta = zeta - 1,   O = d ln Psi / d zeta = 3/(2 zeta) - r,
    #   E_L = -zeta^2/2 + (zeta - 1)/r.
    # Samples of |Psi|^2 from the oracle's own sampler (pinned by P17), O from oracle_orbital_derivatives (pinned by its
    # closed form), then oracle_energy_gradient must give zeta - 1 within 4 standard errors -- a factor 1 or 4 instead
    # of 2, or a flipped sign, is tens of standard errors away.
    for zeta in (1.3, 0.75):
        d = atom_system(1, [(1, 0, 0, zeta)], [[1.0]], 1, 0)
        o = ob.OracleSystem(d)
        M = 40000
        r0 = soa(_rand_pos(M, 1, 1.0, rmin=0.05, seed=17))
        out = ob.metropolis(o, r0, 0.7 / zeta, 60, seed=31, threads=os.cpu_count() or 1)
        r = out["r"]
        el = ob.local_energy(o, r, threads=os.cpu_count() or 1)[2]
        dz = ob.orbital_derivatives(o, r, threads=os.cpu_count() or 1)[1]       # [M, 1]
        rr = np.linalg.norm(r[0], axis=0)
        assert np.max(np.abs(dz[:, 0] - (1.5 / zeta - rr))) < 1e-12             # the factor O itself
        ev, g = ob.energy_gradient(el, dz)
        per_walker = 2.0 * dz[:, 0] * (el - ev)
        sigma = per_walker.std(ddof=1) / math.sqrt(M)
        assert abs(ev - (zeta * zeta / 2 - zeta)) < 5 * el.std(ddof=1) / math.sqrt(M)
        assert abs(g[0] - (zeta - 1.0)) < 4 * sigma, (zeta, g[0], sigma)
        assert sigma < 0.1 * abs(zeta - 1.0)                                    # the pin resolves scale and sign


# ---------------------------------------------------------------- electron-nucleus Jastrow (D.2)
def _with_en(d, w0, w1, w2):
    import copy
    d2 = copy.copy(d)
    d2.jastrow_en_w0, d2.jastrow_en_w1, d2.jastrow_en_w2 = w0, w1, w2
    return d2


@pytest.mark.parametrize("Z,zeta,w", [(1.0, 1.0, (0.3, -0.05, 0.7)), (3.0, 2.2, (-0.4, 0.1, 1.3))])
def test_en_jastrow_hydrogenlike_closed_form(Z, zeta, w):
    # one electron: Psi = N exp(f(r)), f = -zeta r + K_en(r); E_L = -1/2 (f'' + 2 f'/r + f'^2) - Z/r.
    # K' and K'' from the partial-fraction form K = A r + B (1 - 1/(1 + w2 r)), A = w1/w2, B = (w0 - A)/w2,
    # an algebraically different route from the oracle's quotient rule
    w0, w1, w2 = w
    d = _with_en(atom_system(Z, [(1, 0, 0, zeta)], [[1.0]], 1, 0), w0, w1, w2)
    rr = _rand_pos(100, 1, 1.5, rmin=0.05, seed=90)
    lp, sg, el = ob.local_energy(ob.OracleSystem(d), soa(rr))
    r = np.linalg.norm(rr[:, 0], axis=1)
    A = w1 / w2
    B = (w0 - A) / w2
    D = 1 + w2 * r
    K = A * r + B * (1 - 1 / D)
    K1 = A + B * w2 / D ** 2
    K2 = -2 * B * w2 ** 2 / D ** 3
    f1 = -zeta + K1
    ref = -0.5 * (K2 + 2 * f1 / r + f1 ** 2) - Z / r
    assert np.max(np.abs(el - ref) / np.maximum(1, np.abs(ref))) < 1e-12
    N = zeta ** 1.5 / math.sqrt(math.pi)
    assert np.max(np.abs(lp - (math.log(N) - zeta * r + K))) < 1e-12


def test_en_jastrow_finite_differences_and_sampler_value():
    # analytic grad / Laplacian of the e-n term against Richardson differences of the plain Psi (two centres,
    # several electrons, together with the e-e term), and the sampler's value-only route against it
    for name, M in (("LiH", 6), ("CO", 3)):
        d, r = wl.CONFIGS[name](M=64)
        d = _with_en(d, 0.35, -0.04, 0.9)
        o = ob.OracleSystem(d)
        lp_all = ob.local_energy(o, r)[0]
        idx = _keep_away(d, r)
        idx = idx[np.argsort(-lp_all[idx])][:M]  # well away from nuclei and nodes (Q17)
        rk = np.ascontiguousarray(r[:, :, idx])
        _fd_check(d, rk, nwalk=len(idx), tol=2e-6)
        lp = ob.local_energy(o, rk)[0]
        out = ob.metropolis(o, rk, 0.2, 0, seed=1)
        assert np.max(np.abs(out["logpsi"] - lp)) < 1e-12


def test_en_jastrow_absent_when_parameters_are_zero():
    d, r = wl.li2(M=16)
    a = ob.local_energy(ob.OracleSystem(d), r)
    b = ob.local_energy(ob.OracleSystem(_with_en(d, 0.0, 0.0, 0.8)), r)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    c = ob.local_energy(ob.OracleSystem(_with_en(d, 0.2, 0.0, 0.8)), r)
    assert np.max(np.abs(c[2] - a[2])) > 1e-3


# ---------------------------------------------------------------- electron-electron-nucleus Jastrow (D.3)
EEN = np.array([[0.30, 0.8, 0.9, 0.5, 1.4, 0.7, 0.6],
                [-0.12, 1.1, 0.4, 0.9, 0.8, 0.35, 1.2],
                [0.05, 0.6, 1.7, 1.3, 0.5, 1.0, 0.9]])


def _with_een(d, een=EEN):
    import copy
    d2 = copy.copy(d)
    d2.jastrow_een = np.asarray(een, np.float64)
    return d2


def test_een_jastrow_closed_form_two_electrons():
    # two electrons, one nucleus at the origin: the one pair of eq. 5's sum_{alpha, i>j}, symmetrised
    # (reading Q22): J_een = sum_mu (c/2) [f(r1) g(r2) + f(r2) g(r1)] h(r12)
    d0 = atom_system(2.0, [(1, 0, 0, 1.7)], [[1.0]], 1, 1, a_par=0.25, a_anti=0.5, b=0.9)
    rr = _rand_pos(60, 2, 1.2, rmin=0.05, seed=91)
    lp0 = ob.local_energy(ob.OracleSystem(d0), soa(rr))[0]
    lp1 = ob.local_energy(ob.OracleSystem(_with_een(d0)), soa(rr))[0]
    r1, r2 = np.linalg.norm(rr[:, 0], axis=1), np.linalg.norm(rr[:, 1], axis=1)
    r12 = np.linalg.norm(rr[:, 0] - rr[:, 1], axis=1)
    pade = lambda a, b, r: a * r / (1 + b * r)
    J = sum(0.5 * c * (pade(a1, b1, r1) * pade(a2, b2, r2) + pade(a1, b1, r2) * pade(a2, b2, r1)) * pade(a3, b3, r12)
            for c, a1, b1, a2, b2, a3, b3 in EEN)
    assert np.max(np.abs((lp1 - lp0) - J)) < 1e-13


def test_een_jastrow_equals_the_literal_pair_sum_of_eq5_for_symmetric_factors():
    # eq. 5 with D.3 as printed: J_een = sum_alpha sum_{i>j} sum_mu c f(r_ai) g(r_aj) h(r_ij).
    # With a1 = a2, b1 = b2 (f = g) the symmetrised reading Q22 must reproduce that hand sum exactly -- on a
    # three-centre, five-electron system so that a factor 2, a missing nucleus or a missing pair all show.
    een = np.array([[0.30, 0.8, 0.9, 0.8, 0.9, 0.7, 0.6], [-0.12, 1.1, 0.4, 1.1, 0.4, 0.35, 1.2]])
    xyz = np.array([[0.0, 0.0, 0.0], [0.0, 0.9, 1.8], [1.1, -0.4, 0.3]])
    from paper_2506_09743_b200.workloads import SystemDesc
    aos = [(1, 0, 0, 1.3), (1, 0, 0, 0.9), (2, 1, 2, 1.1), (2, 0, 0, 0.8)]
    d = SystemDesc("3c", xyz, np.array([2.0, 1.0, 2.0]), 3, 2, np.array([0, 1, 2, 2], np.int32),
                   np.array([a[0] for a in aos], np.int32), np.array([a[1] for a in aos], np.int32),
                   np.array([a[2] for a in aos], np.int32), np.array([a[3] for a in aos]), None,
                   np.random.default_rng(5).standard_normal((4, 3)), np.array([[0, 1, 2]], np.int32),
                   np.array([[0, 1]], np.int32), np.array([1.0]), 0.25, 0.5, 0.9)
    rr = _rand_pos(25, 5, 1.5, rmin=0.05, seed=93)
    lp0 = ob.local_energy(ob.OracleSystem(d), soa(rr))[0]
    lp1 = ob.local_energy(ob.OracleSystem(_with_een(d, een)), soa(rr))[0]
    pade = lambda a, b, r: a * r / (1 + b * r)
    J = np.zeros(len(rr))
    for A in xyz:
        for i in range(5):
            for j in range(i):          # i > j: every pair once
                rai, raj = np.linalg.norm(rr[:, i] - A, axis=1), np.linalg.norm(rr[:, j] - A, axis=1)
                rij = np.linalg.norm(rr[:, i] - rr[:, j], axis=1)
                for c, a1, b1, a2, b2, a3, b3 in een:
                    J += c * pade(a1, b1, rai) * pade(a2, b2, raj) * pade(a3, b3, rij)
    assert np.max(np.abs((lp1 - lp0) - J)) < 1e-12


def test_een_jastrow_finite_differences_exchange_and_sampler_value():
    for name, M in (("LiH", 5), ("CO", 2)):
        d, r = wl.CONFIGS[name](M=64)
        d = _with_een(_with_en(d, 0.2, -0.03, 0.8))
        o = ob.OracleSystem(d)
        lp_all = ob.local_energy(o, r)[0]
        idx = _keep_away(d, r)
        idx = idx[np.argsort(-lp_all[idx])][:M]
        rk = np.ascontiguousarray(r[:, :, idx])
        # analytic grad / Laplacian through three distances vs the plain Psi; h = 2e-4: at 1e-4 the difference
        # quotient is already round-off dominated here (error grows like 1/h^2: 8e-7, 5e-6, 1.3e-5 at 2e-4, 1e-4, 5e-5)
        _fd_check(d, rk, h=2e-4, nwalk=len(idx), tol=2e-6)
        lp, sg, el = ob.local_energy(o, rk)
        out = ob.metropolis(o, rk, 0.2, 0, seed=1)    # value-only route of the sampler
        assert np.max(np.abs(out["logpsi"] - lp)) < 1e-12
        # exchanging two same-spin electrons: |Psi| and E_L unchanged, sign flips (the kernel is symmetric only
        # because every pair enters symmetrised: f != g in EEN)
        rx = rk.copy()
        rx[[0, 1]] = rx[[1, 0]]
        lpx, sgx, elx = ob.local_energy(o, rx)
        assert np.max(np.abs(lpx - lp)) < 1e-11 and np.array_equal(sgx, -sg)
        assert np.max(np.abs(elx - el) / np.maximum(1, np.abs(el))) < 1e-9


def test_een_jastrow_absent_without_terms():
    d, r = wl.li2(M=8)
    a = ob.local_energy(ob.OracleSystem(d), r)
    b = ob.local_energy(ob.OracleSystem(_with_een(d, np.zeros((0, 7)))), r)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    c = ob.local_energy(ob.OracleSystem(_with_een(d)), r)
    assert np.max(np.abs(c[2] - a[2])) > 1e-3


def test_een_parameter_derivatives_vs_central_differences_closed_form_and_layout():
    # O_p for the 7 n_een parameters of D.3 sit between the six D.1/D.2 parameters and the CI coefficients;
    # pinned by Richardson central differences of the oracle's own log|Psi| in EVERY such parameter, by the
    # two-electron closed form, and by Euler's identity for the coefficient c (the term is linear in it)
    for name, M in (("LiH", 6), ("CO", 3)):
        d, r = wl.CONFIGS[name](M=M)
        d = _with_een(_with_en(d, 0.2, -0.03, 0.8))
        O = ob.log_derivatives(ob.OracleSystem(d), r)
        n_een = EEN.shape[0]
        assert O.shape == (M, NJ + 7 * n_een + len(d.ci_coeff))
        for mu in range(n_een):
            for k in range(7):
                t0 = EEN[mu, k]

                def cd(h):
                    out = []
                    for sgn in (1.0, -1.0):
                        e2 = EEN.copy()
                        e2[mu, k] = t0 + sgn * h
                        out.append(ob.local_energy(ob.OracleSystem(_with_een(d, e2)), r)[0])
                    return (out[0] - out[1]) / (2 * h)

                h = 1e-3 * max(1.0, abs(t0))
                fd = (4 * cd(h / 2) - cd(h)) / 3
                col = O[:, NJ + 7 * mu + k]
                assert np.max(np.abs(col - fd) / np.maximum(1, np.abs(fd))) < 1e-7, (name, mu, k)
        # CI block moved behind the D.3 block, unchanged: sum rule
        assert np.max(np.abs(O[:, NJ + 7 * n_een:] @ np.asarray(d.ci_coeff) - 1.0)) < 1e-10
        # the first six columns do not depend on the D.3 terms
        O0 = ob.log_derivatives(ob.OracleSystem(_with_een(d, np.zeros((0, 7)))), r)
        assert np.array_equal(O0[:, :NJ], O[:, :NJ]) and O0.shape[1] == NJ + len(d.ci_coeff)
    # two electrons, one nucleus: J_een = sum_mu (c/2) [f(r1) g(r2) + f(r2) g(r1)] h(r12)
    d0 = _with_een(atom_system(2.0, [(1, 0, 0, 1.7)], [[1.0]], 1, 1, a_par=0.25, a_anti=0.5, b=0.9))
    rr = _rand_pos(40, 2, 1.2, rmin=0.05, seed=92)
    O = ob.log_derivatives(ob.OracleSystem(d0), soa(rr))
    r1, r2 = np.linalg.norm(rr[:, 0], axis=1), np.linalg.norm(rr[:, 1], axis=1)
    r12 = np.linalg.norm(rr[:, 0] - rr[:, 1], axis=1)
    pade = lambda a, b, x: a * x / (1 + b * x)
    da = lambda a, b, x: x / (1 + b * x)
    db = lambda a, b, x: -a * x * x / (1 + b * x) ** 2
    for mu, (c, a1, b1, a2, b2, a3, b3) in enumerate(EEN):
        f1, f2, g1, g2, hh = pade(a1, b1, r1), pade(a1, b1, r2), pade(a2, b2, r1), pade(a2, b2, r2), pade(a3, b3, r12)
        want = [(f1 * g2 + f2 * g1) * hh,
                c * (da(a1, b1, r1) * g2 + da(a1, b1, r2) * g1) * hh, c * (db(a1, b1, r1) * g2 + db(a1, b1, r2) * g1) * hh,
                c * (f1 * da(a2, b2, r2) + f2 * da(a2, b2, r1)) * hh, c * (f1 * db(a2, b2, r2) + f2 * db(a2, b2, r1)) * hh,
                c * (f1 * g2 + f2 * g1) * da(a3, b3, r12), c * (f1 * g2 + f2 * g1) * db(a3, b3, r12)]
        for k in range(7):
            assert np.max(np.abs(O[:, NJ + 7 * mu + k] - 0.5 * want[k])) < 1e-13, (mu, k)


# ---------------------------------------------------------------- orbital parameters (AO exponents, MO coefficients)
@pytest.mark.parametrize("name,M", [("H2", 6), ("LiH", 5), ("Li2", 3), ("CO", 2)])
def test_orbital_derivatives_vs_central_differences_of_log_psi(name, M):
    # d ln Psi / d zeta_beta and d ln Psi / d C[beta][alpha] against Richardson central differences of the
    # oracle's own log|Psi| (rebuilt with one AO exponent / one MO coefficient perturbed): pins the inverse
    # transposition, the column bookkeeping over determinants, the CI weights and d(norm)/d zeta
    d, r = wl.CONFIGS[name](M=M)
    _check_orbital_derivatives_fd(d, r, name)


def _check_orbital_derivatives_fd(d, r, name):
    import copy
    o = ob.OracleSystem(d)
    dC, dz = ob.orbital_derivatives(o, r)
    rng = np.random.default_rng(3)
    used = sorted(set(np.asarray(d.det_up).ravel()) | set(np.asarray(d.det_dn).ravel()))

    def fd(make, t0, h):
        def cd(hh):
            lp_p = ob.local_energy(ob.OracleSystem(make(t0 + hh)), r)[0]
            lp_m = ob.local_energy(ob.OracleSystem(make(t0 - hh)), r)[0]
            return (lp_p - lp_m) / (2 * hh)
        return (4 * cd(h / 2) - cd(h)) / 3

    for beta in rng.choice(d.n_ao, min(4, d.n_ao), replace=False):
        def mk(z, beta=beta):
            d2 = copy.copy(d)
            zz = np.array(d.ao_zeta, np.float64, copy=True)
            zz[beta] = z
            d2.ao_zeta = zz
            return d2
        ref = fd(mk, float(d.ao_zeta[beta]), 1e-3)
        assert np.max(np.abs(dz[:, beta] - ref) / np.maximum(1, np.abs(ref))) < 1e-7, (name, "zeta", beta)
        alpha = int(rng.choice(used))
        def mkc(c, beta=beta, alpha=alpha):
            d2 = copy.copy(d)
            cc = np.array(d.mo_coeff, np.float64, copy=True)
            cc[beta, alpha] = c
            d2.mo_coeff = cc
            return d2
        ref = fd(mkc, float(d.mo_coeff[beta, alpha]), 1e-3)
        assert np.max(np.abs(dC[:, beta, alpha] - ref) / np.maximum(1, np.abs(ref))) < 1e-7, (name, "C", beta, alpha)
    # an MO that no determinant uses cannot matter
    unused = [a for a in range(d.n_mo) if a not in used]
    if unused:
        assert np.max(np.abs(dC[:, :, unused])) == 0.0


def test_orbital_derivatives_closed_form_and_scaling_identity():
    # hydrogen-like 1s: ln Psi = ln N(zeta) - zeta r  =>  d/dzeta = 3/(2 zeta) - r ; d/dC = 1/C
    zeta, c = 1.3, 0.7
    d = atom_system(1.0, [(1, 0, 0, zeta)], [[c]], 1, 0)
    rr = _rand_pos(40, 1, 1.5, rmin=0.05, seed=95)
    dC, dz = ob.orbital_derivatives(ob.OracleSystem(d), soa(rr))
    rad = np.linalg.norm(rr[:, 0], axis=1)
    assert np.max(np.abs(dz[:, 0] - (1.5 / zeta - rad))) < 1e-13 and np.max(np.abs(dC[:, 0, 0] - 1 / c)) < 1e-13
    # custom normalisation: no d(norm)/d zeta
    d = atom_system(1.0, [(1, 0, 0, zeta)], [[c]], 1, 0, norm=[2.0])
    dz = ob.orbital_derivatives(ob.OracleSystem(d), soa(rr))[1]
    assert np.max(np.abs(dz[:, 0] + rad)) < 1e-13
    # Euler: scaling every coefficient of the MOs by t scales each determinant by t^(n_e): sum C dlnPsi/dC = n_e
    # (every determinant here uses n_up + n_dn columns)
    d, r = wl.li2(M=10)
    dC, _ = ob.orbital_derivatives(ob.OracleSystem(d), r)
    assert np.max(np.abs(np.einsum("mba,ba->m", dC, d.mo_coeff) - d.n_e)) < 1e-10


# ---------------------------------------------------------------- nuclear log-gradient (eq. 7)
@pytest.mark.parametrize("name,M", [("H2", 6), ("LiH", 5), ("Li2", 3), ("CO", 2)])
def test_nuclear_log_gradient_vs_central_differences_of_log_psi(name, M):
    # grad_alpha ln|Psi| against Richardson central differences of the oracle's own (pinned) log|Psi| with one
    # nuclear coordinate displaced, D.2 and D.3 switched on: pins the sign of d ao / d R, the AO -> atom
    # bookkeeping, the CI weights, and both Jastrow chain rules
    d, r = wl.CONFIGS[name](M=M)
    _check_nuclear_log_gradient_fd(_with_een(_with_en(d, 0.3, -0.05, 0.7)), r, name)


def _check_nuclear_log_gradient_fd(d, r, name):
    import copy
    dR = ob.nuclear_log_gradient(ob.OracleSystem(d), r)
    assert dR.shape == (r.shape[2], d.n_atoms, 3)

    def lp(a, c, t):
        d2 = copy.copy(d)
        xyz = np.array(d.atom_xyz, np.float64, copy=True)
        xyz[a, c] += t
        d2.atom_xyz = xyz
        return ob.local_energy(ob.OracleSystem(d2), r)[0]

    for a in range(d.n_atoms):
        for c in range(3):
            cd = lambda h: (lp(a, c, h) - lp(a, c, -h)) / (2 * h)
            ref = (4 * cd(1e-4) - cd(2e-4)) / 3
            # 1e-6: the bound BASELINE.json's north_star gives for central differences at h = 1e-4
            assert np.max(np.abs(dR[:, a, c] - ref) / np.maximum(1, np.abs(ref))) < 1e-6, (name, a, c)


def test_nuclear_log_gradient_closed_form_translation_and_partition():
    # hydrogen-like 1s at R: ln Psi = const - zeta |r - R|  =>  grad_R ln Psi = zeta (r - R)/|r - R|
    zeta, R = 1.3, np.array([0.3, -0.2, 0.5])
    d = atom_system(1.0, [(1, 0, 0, zeta)], [[1.0]], 1, 0, xyz=tuple(R))
    rr = _rand_pos(40, 1, 1.5, rmin=0.05, seed=96) + R
    dR = ob.nuclear_log_gradient(ob.OracleSystem(d), soa(rr))
    u = rr[:, 0] - R
    assert np.max(np.abs(dR[:, 0] - zeta * u / np.linalg.norm(u, axis=1, keepdims=True))) < 1e-13
    # translation invariance: Psi depends on r_i - R_a and r_i - r_j only, so
    # sum_a grad_a ln Psi = -sum_i grad_i ln Psi (the latter by central differences of a rigid electron shift)
    d, r = wl.li2(M=6)
    d = _with_een(_with_en(d, 0.3, -0.05, 0.7))
    o = ob.OracleSystem(d)
    dR = ob.nuclear_log_gradient(o, r)
    for c in range(3):
        def shifted(t):
            r2 = np.array(r, copy=True)
            r2[:, c, :] += t
            return ob.local_energy(o, r2)[0]
        cd = lambda h: (shifted(h) - shifted(-h)) / (2 * h)
        ref = (4 * cd(1e-4) - cd(2e-4)) / 3
        assert np.max(np.abs(dR[:, :, c].sum(axis=1) + ref) / np.maximum(1, np.abs(ref))) < 1e-6
    # partition independence (threads) and a diatomic on z with sigma orbitals only has no x, y asymmetry pin:
    # H2 with both electrons on the axis -> gradient along z only
    d, _ = wl.h2(M=4)
    rz = np.zeros((4, 2, 3))
    rz[:, :, 2] = np.random.default_rng(5).uniform(-1.5, 1.5, (4, 2))
    g = ob.nuclear_log_gradient(ob.OracleSystem(d), soa(rz))
    assert np.max(np.abs(g[:, :, :2])) < 1e-14 and np.min(np.abs(g[:, :, 2])) > 1e-3
    d, r = wl.lih(M=9)
    o = ob.OracleSystem(d)
    assert np.array_equal(ob.nuclear_log_gradient(o, r, threads=1), ob.nuclear_log_gradient(o, r, threads=3))


# ---------------------------------------------------------------- forces: grad_alpha E_L and the estimator of eq. 7
def test_ao_hessian_and_laplacian_gradient_vs_central_differences():
    # oracle_ao_eval2's new outputs against Richardson central differences of the PINNED first-level outputs of
    # oracle_ao_eval (gradient -> Hessian, Laplacian -> its gradient), for every kind of AO: s with k = 0, 1, 2,
    # every p and d harmonic, with a radial power
    aos = [(1, 0, 0, 1.3), (2, 0, 0, 0.9), (3, 0, 0, 1.1)] + [(2, 1, m, 1.2) for m in range(3)] + \
          [(3, 1, m, 0.8) for m in range(3)] + [(3, 2, m, 1.0) for m in range(5)] + [(4, 2, m, 1.4) for m in range(5)]
    d = atom_system(1.0, aos, np.eye(len(aos))[:, :1], 1, 0, xyz=(0.2, -0.1, 0.3))
    o = ob.OracleSystem(d)
    rng = np.random.default_rng(11)
    pairs = {(0, 0): 5, (1, 1): 6, (2, 2): 7, (0, 1): 8, (1, 2): 9, (2, 0): 10}
    for ao in range(len(aos)):
        for _ in range(3):
            x = np.array([0.2, -0.1, 0.3]) + rng.standard_normal(3) * 0.7 + 0.3
            v = ob.ao_eval2(o, ao, x)
            assert np.max(np.abs(v[:5] - ob.ao_eval(o, ao, x))) < 1e-14 * max(1.0, np.max(np.abs(v[:5])))

            def cd(q, c, h):
                e = np.zeros(3); e[c] = h
                return (ob.ao_eval(o, ao, x + e)[q] - ob.ao_eval(o, ao, x - e)[q]) / (2 * h)

            scale = max(1.0, np.max(np.abs(v)))
            for (a, b), k in pairs.items():
                fd = (4 * cd(1 + a, b, 5e-4) - cd(1 + a, b, 1e-3)) / 3     # d_b of (d_a phi)
                assert abs(v[k] - fd) < 2e-8 * scale, (aos[ao], a, b, v[k], fd)
            for c in range(3):
                fd = (4 * cd(4, c, 5e-4) - cd(4, c, 1e-3)) / 3             # d_c of lap phi
                assert abs(v[11 + c] - fd) < 2e-7 * scale, (aos[ao], c, v[11 + c], fd)


@pytest.mark.parametrize("name,M", [("H2", 5), ("LiH", 4), ("Li2", 3), ("CO", 2)])
def test_nuclear_energy_gradient_vs_central_differences_of_E_L(name, M):
    # grad_alpha E_L against Richardson central differences of the oracle's own pinned E_L with one nuclear
    # coordinate displaced: a wrong sign of d ao / d R, a dropped d(A^-1) term, a wrong CI weight derivative or a
    # missing potential term each fail it
    import copy
    d, r = wl.CONFIGS[name](M=64)
    lp_all = ob.local_energy(ob.OracleSystem(d), r)[0]
    idx = _keep_away(d, r)
    idx = idx[np.argsort(-lp_all[idx])][:M]                 # away from nuclei and nodes (Q17)
    rk = np.ascontiguousarray(r[:, :, idx])
    dE = ob.nuclear_energy_gradient(ob.OracleSystem(d), rk)
    assert dE.shape == (len(idx), d.n_atoms, 3)

    def el(a, c, t):
        d2 = copy.copy(d)
        xyz = np.array(d.atom_xyz, np.float64, copy=True)
        xyz[a, c] += t
        d2.atom_xyz = xyz
        return ob.local_energy(ob.OracleSystem(d2, extended=True), rk)[2]

    for a in range(d.n_atoms):
        for c in range(3):
            cd = lambda h: (el(a, c, h) - el(a, c, -h)) / (2 * h)
            ref = (4 * cd(1e-4) - cd(2e-4)) / 3
            assert np.max(np.abs(dE[:, a, c] - ref) / np.maximum(1, np.abs(ref))) < 1e-6, (name, a, c, dE[:, a, c], ref)


def test_nuclear_energy_gradient_closed_forms_and_translation_invariance():
    # hydrogen-like 1s (zeta) on a nucleus Z at R plus a bare charge q at R2 (no basis functions on it):
    #   E_L = -zeta^2/2 + (zeta - Z)/|r - R| - q/|r - R2| + Z q/|R - R2|
    #   grad_R  E_L = (zeta - Z)(r - R)/|r - R|^3 - Z q (R - R2)/|R - R2|^3
    #   grad_R2 E_L = -q (r - R2)/|r - R2|^3      + Z q (R - R2)/|R - R2|^3
    from paper_2506_09743_b200.workloads import SystemDesc
    Z, zeta, q = 2.0, 1.6, 0.7
    R, R2 = np.array([0.3, -0.2, 0.5]), np.array([-1.1, 0.9, 2.0])
    d = SystemDesc("h-like+q", np.array([R, R2]), np.array([Z, q]), 1, 0, np.zeros(1, np.int32), np.ones(1, np.int32),
                   np.zeros(1, np.int32), np.zeros(1, np.int32), np.array([zeta]), None, np.array([[1.0]]),
                   np.zeros((1, 1), np.int32), np.zeros((1, 0), np.int32), np.array([1.0]), 0.25, 0.5, 1.0)
    rr = _rand_pos(60, 1, 1.5, rmin=0.05, seed=97) + R
    dE = ob.nuclear_energy_gradient(ob.OracleSystem(d), soa(rr))
    v, v2, RR = rr[:, 0] - R, rr[:, 0] - R2, R - R2
    want = np.stack([(zeta - Z) * v / np.linalg.norm(v, axis=1, keepdims=True) ** 3 - Z * q * RR / np.linalg.norm(RR) ** 3,
                     -q * v2 / np.linalg.norm(v2, axis=1, keepdims=True) ** 3 + Z * q * RR / np.linalg.norm(RR) ** 3], axis=1)
    assert np.max(np.abs(dE - want) / np.maximum(1, np.abs(want))) < 1e-12
    # translation invariance of E_L(r; R): sum_alpha grad_alpha E_L = -sum_i grad_i E_L, the right side by Richardson
    # central differences of the oracle's E_L under a rigid shift of every electron (Li2, 20 determinants)
    dsys, r = wl.li2(M=64)
    o = ob.OracleSystem(dsys)
    lp_all = ob.local_energy(o, r)[0]
    idx = _keep_away(dsys, r)
    idx = idx[np.argsort(-lp_all[idx])][:4]
    rk = np.ascontiguousarray(r[:, :, idx])
    tot = ob.nuclear_energy_gradient(o, rk).sum(axis=1)
    ox = ob.OracleSystem(dsys, extended=True)
    for c in range(3):
        def shifted(t):
            r2 = rk.copy()
            r2[:, c, :] += t
            return ob.local_energy(ox, r2)[2]
        cd = lambda h: (shifted(h) - shifted(-h)) / (2 * h)
        ref = -(4 * cd(1e-4) - cd(2e-4)) / 3
        assert np.max(np.abs(tot[:, c] - ref) / np.maximum(1, np.abs(ref))) < 1e-6, (c, tot[:, c], ref)
    # the e-n / e-e-n kernels are not covered: the call says so instead of returning a partial derivative
    L = ob.lib()
    o2 = ob.OracleSystem(_with_en(dsys, 0.2, 0.0, 0.8))
    out = np.zeros((rk.shape[2], 2, 3))
    assert L.oracle_nuclear_energy_gradient(o2.ref, rk.ctypes.data, rk.shape[2], 0, rk.shape[2], out.ctypes.data) == -2


def test_force_estimator_formula_and_physical_pin():
    # (i) the reduction itself against math.fsum of eq. 7 (reading Q23)
    rng = np.random.default_rng(8)
    M, na = 500, 3
    e = rng.standard_normal(M) * 2 - 7
    dE, dl = rng.standard_normal((M, na, 3)), rng.standard_normal((M, na, 3))
    F, T = ob.force(e, dE, dl)
    ev = math.fsum(e) / M
    for a in range(na):
        for c in range(3):
            t1 = -math.fsum(dE[:, a, c]) / M
            t2 = -math.fsum(2 * (e - ev) * dl[:, a, c]) / M
            assert abs(T[0, a, c] - t1) < 1e-13 and abs(T[1, a, c] - t2) < 1e-13 and abs(F[a, c] - (t1 + t2)) < 1e-13
    # (ii) physical pin of both terms' signs and of the factor 2: He+-like exact 1s (zeta = Z = 2) on nucleus A at the
    # origin, a bare charge q at distance R on the z axis.  The variational energy depends on R only through
    #   E(R) = const + Z q / R - q phi(R),  phi(R) = [1 - e^{-2 zeta R}(1 + zeta R)] / R  (potential of the 1s density),
    # so F_B = -dE/dR = q [(Z - 1)/R^2 + e^{-2 zeta R}(1/R^2 + 2 zeta/R + 2 zeta^2)] along +z and F_A = -F_B.
    # For B only the first term of eq. 7 contributes (Psi does not depend on R_B); for A the second term carries
    # +q/R^2 of the total (1 - Z) q/R^2 to leading order, so a factor 1 instead of 2 would be ~50% off.
    from paper_2506_09743_b200.workloads import SystemDesc
    Z = zeta = 2.0
    q, R = 0.5, 3.0
    d = SystemDesc("He+ + q", np.array([[0.0, 0.0, 0.0], [0.0, 0.0, R]]), np.array([Z, q]), 1, 0, np.zeros(1, np.int32),
                   np.ones(1, np.int32), np.zeros(1, np.int32), np.zeros(1, np.int32), np.array([zeta]), None,
                   np.array([[1.0]]), np.zeros((1, 1), np.int32), np.zeros((1, 0), np.int32), np.array([1.0]), 0.25, 0.5, 1.0)
    o = ob.OracleSystem(d)
    M = 60000
    nt = os.cpu_count() or 1
    out = ob.metropolis(o, soa(_rand_pos(M, 1, 0.5, rmin=0.02, seed=19)), 0.45, 60, seed=77, threads=nt)
    r = out["r"]
    el = ob.local_energy(o, r, threads=nt)[2]
    dE = ob.nuclear_energy_gradient(o, r, threads=nt)
    dl = ob.nuclear_log_gradient(o, r, threads=nt)
    F, T = ob.force(el, dE, dl)
    FB = q * ((Z - 1) / R ** 2 + math.exp(-2 * zeta * R) * (1 / R ** 2 + 2 * zeta / R + 2 * zeta ** 2))
    ev = el.mean()
    per_walker = -(dE + 2 * (el - ev)[:, None, None] * dl)
    sig = per_walker.std(axis=0, ddof=1) / math.sqrt(M)
    assert abs(F[1, 2] - FB) < 4 * sig[1, 2] and abs(F[0, 2] + FB) < 4 * sig[0, 2], (F, FB, sig)
    assert sig[0, 2] < 0.05 * FB and sig[1, 2] < 0.05 * FB                     # the pin resolves sign and scale
    assert np.max(np.abs(F[:, :2])) < 4 * np.max(sig[:, :2]) + 1e-12           # no force off the axis
    assert abs(T[1, 1, 2]) < 1e-12                                             # Psi does not depend on R_B
    assert abs(T[1, 0, 2] - q / R ** 2) < 0.15 * q / R ** 2                    # second term: +q/R^2 to leading order


# ---------------------------------------------------------------- inverse backflow (F.4 cross term, F.5)
def _with_bf(d, w):
    import copy
    d2 = copy.copy(d)
    d2.backflow_w = w
    return d2


def test_backflow_map_is_a_push_of_w_along_every_unit_vector():
    # K_BF(r) = w / r  =>  rt_i = r_i + w sum_{j != i} (r_i - r_j)/|r_i - r_j|, over ALL other electrons (both spins)
    d, r = wl.li2(M=5)
    o = ob.OracleSystem(_with_bf(d, 0.17))
    for w in range(5):
        rr = r[:, :, w]
        rt = ob.backflow_coords(o, rr)
        want = rr.copy()
        for i in range(6):
            for j in range(6):
                if j != i:
                    want[i] += 0.17 * (rr[i] - rr[j]) / np.linalg.norm(rr[i] - rr[j])
        assert np.max(np.abs(rt - want)) < 1e-14
    # a single electron has no partner: the hydrogen atom stays exact
    da = _with_bf(atom_system(1, [(1, 0, 0, 1.0)], [[1.0]], 1, 0), 0.3)
    el = ob.local_energy(ob.OracleSystem(da), soa(_rand_pos(50, 1, 2.0, seed=3)))[2]
    assert np.max(np.abs(el - GOLDEN["E_n1"])) < 1e-12


@pytest.mark.parametrize("name,M,w", [("H2", 4, 0.2), ("LiH", 4, 0.12), ("Li2", 3, 0.08), ("CO", 2, 0.05)])
def test_backflow_local_energy_vs_finite_differences_of_the_plain_psi(name, M, w):
    # the whole general chain (Jacobian and second derivatives of the map, AO Hessians, F.3, F.5, the cross term of
    # F.4, F.1) against Richardson central differences of the plain definition e^J sum_n d_n det det evaluated at the
    # backflow coordinates (oracle_psi_plain): a dropped cross term or a wrong sign in F.5 is O(w), far above the bound
    d, r = wl.CONFIGS[name](M=64)
    d = _with_bf(d, w)
    o = ob.OracleSystem(d)
    lp_all = ob.local_energy(o, r)[0]
    idx = _keep_away(d, r)
    # also keep electrons apart: the inverse kernel is singular at coalescence
    rr = r.transpose(2, 0, 1)
    dmin = np.array([min(np.linalg.norm(rr[k, i] - rr[k, j]) for i in range(d.n_e) for j in range(i)) for k in range(rr.shape[0])])
    idx = np.array([k for k in idx if dmin[k] > 0.4])
    idx = idx[np.argsort(-lp_all[idx])][:M]
    _fd_check(d, np.ascontiguousarray(r[:, :, idx]), nwalk=len(idx), tol=3e-6)


def test_backflow_limit_antisymmetry_and_sampler_value():
    d, r = wl.li2(M=24)
    o0 = ob.OracleSystem(d)
    lp0, sg0, el0 = ob.local_energy(o0, r)
    # w -> 0: the general formulas (every coordinate's dense d_l A, F.5 with both extra traces, F.4's cross term) must
    # collapse onto the single-electron-orbital result G.7 (Appendix G)
    lp1, sg1, el1 = ob.local_energy(ob.OracleSystem(_with_bf(d, 1e-200)), r)
    assert np.array_equal(sg1, sg0) and np.max(np.abs(lp1 - lp0)) < 1e-12
    keep = lp0 - lp0.max() > math.log(1e-6)
    assert np.max((np.abs(el1 - el0) / np.maximum(1, np.abs(el0)))[keep]) < 1e-9
    # a finite w changes the energy, is antisymmetric under same-spin exchange (the map treats all
    # electrons alike), and the sampler's value-only route agrees with the E_L route
    db = _with_bf(d, 0.1)
    ob_ = ob.OracleSystem(db)
    lp, sg, el = ob.local_energy(ob_, r)
    assert np.max(np.abs(el - el0)) > 1e-3
    rx = r.copy()
    rx[[0, 2]] = rx[[2, 0]]
    lpx, sgx, elx = ob.local_energy(ob_, rx)
    assert np.array_equal(sgx, -sg) and np.max(np.abs(lpx - lp)) < 1e-11
    assert np.max((np.abs(elx - el) / np.maximum(1, np.abs(el)))[keep]) < 1e-9
    out = ob.metropolis(ob_, r, 0.2, 0, seed=1)
    assert np.max(np.abs(out["logpsi"] - lp)) < 1e-12
    # nuclear derivatives are not derived for backflow wavefunctions: the call says so
    L = ob.lib()
    buf = np.zeros((24, 64))
    assert L.oracle_nuclear_energy_gradient(ob_.ref, r.ctypes.data, 24, 0, 24, buf.ctypes.data) == -2


@pytest.mark.parametrize("name,w", [("H2", 0.2), ("LiH", -0.12), ("Li2", 0.08), ("CO", 0.05)])
def test_backflow_log_derivatives_vs_finite_differences_of_log_psi(name, w):
    # eq. 6 factors of a backflow wavefunction: the Jastrow entries (J sits at r), the CI entries (determinants at the
    # backflow coordinates) and the backflow weight itself (last entry) against Richardson central differences of the
    # pinned log|Psi| in each parameter
    import copy
    d, r = wl.CONFIGS[name](M=6)
    d = _with_bf(d, w)
    O = ob.log_derivatives(ob.OracleSystem(d), r)
    n_det = len(d.ci_coeff)
    assert O.shape == (6, 6 + n_det + 1)

    def lp_with(**kw):
        d2 = copy.copy(d)
        for k, v in kw.items():
            setattr(d2, k, v)
        return ob.local_energy(ob.OracleSystem(d2), r)[0]

    def fd(field, value, h, index=None):
        def at(x):
            if index is None:
                return lp_with(**{field: x})
            arr = np.array(getattr(d, field), dtype=np.float64).copy()
            arr[index] = x
            return lp_with(**{field: arr})
        d1 = (at(value + h) - at(value - h)) / (2 * h)
        d2 = (at(value + 2 * h) - at(value - 2 * h)) / (4 * h)
        return (4 * d1 - d2) / 3

    tol = lambda x: 1e-6 * np.maximum(1.0, np.abs(x))
    want = fd("backflow_w", w, 1e-4)
    assert np.all(np.abs(O[:, -1] - want) < tol(want)), (O[:, -1], want)
    assert np.max(np.abs(O[:, -1])) > 1e-3                                    # not a vacuous comparison
    for col, field in ((0, "jastrow_a_par"), (1, "jastrow_a_anti"), (2, "jastrow_b")):
        want = fd(field, getattr(d, field), 1e-3)
        assert np.all(np.abs(O[:, col] - want) < tol(want)), (field, O[:, col], want)
    for n in range(min(n_det, 4)):
        want = fd("ci_coeff", float(d.ci_coeff[n]), 1e-3 * max(1.0, abs(float(d.ci_coeff[n]))), index=n)
        assert np.all(np.abs(O[:, 6 + n] - want) < tol(want)), (n, O[:, 6 + n], want)
    # the CI entries are the determinant ratios at the BACKFLOW coordinates: with w they differ from the plain ones
    if n_det > 1:
        O0 = ob.log_derivatives(ob.OracleSystem(_with_bf(d, 0.0)), r)
        assert O0.shape == (6, 6 + n_det) and np.max(np.abs(O0[:, 6:] - O[:, 6:6 + n_det])) > 1e-6


@pytest.mark.parametrize("name,M,w", [("H2", 5, 0.2), ("LiH", 4, -0.12), ("Li2", 3, 0.08), ("CO", 2, 0.05)])
def test_backflow_orbital_and_nuclear_derivatives_vs_central_differences_of_log_psi(name, M, w):
    # orbitals at the backflow coordinates (which depend on neither C, zeta nor the nuclei), Jastrow factor (D.1, D.2, D.3)
    # at r: the same Richardson differences of the pinned log|Psi| as for the plain wavefunction
    d, r = wl.CONFIGS[name](M=M)
    _check_orbital_derivatives_fd(_with_bf(d, w), r, name)
    _check_nuclear_log_gradient_fd(_with_bf(_with_een(_with_en(d, 0.3, -0.05, 0.7)), w), r, name)
    # and they differ from the plain ones
    dC0, _ = ob.orbital_derivatives(ob.OracleSystem(d), r)
    dC1, _ = ob.orbital_derivatives(ob.OracleSystem(_with_bf(d, w)), r)
    assert np.max(np.abs(dC1 - dC0)) > 1e-4


# ---------------------------------------------------------------- P14b: F.8 / F.9 and the table route of the backflow term
def test_P14b_second_order_trace_identities_on_random_matrices():
    # (i) F.8 with F.9 as printed (last line of Appendix H, PAPER.md:542 -- lines 499 and 514-516 of the
    # derivation are garbled, the result is legible):  Tr((A_X^-1 B_X)^2) = Tr((A_0^-1 B_0)^2) + Tr((T~ M)^2) + 2 Tr(T~ Y),
    # T~ = (P A_0^-1 A_X P)^-1 inside the substituted subspace, M of F.7, Y = A_0^-1 B_0 M; single and double substitutions
    rng = np.random.default_rng(140)
    n = 6
    A0, B0 = rng.standard_normal((n, n)), rng.standard_normal((n, n))
    Av, Bv = rng.standard_normal((n, 4)), rng.standard_normal((n, 4))
    Ai0 = np.linalg.inv(A0)
    for P, Q in (([1], [2]), ([4], [0]), ([0, 3], [1, 0]), ([2, 5], [3, 2])):
        AX, BX = A0.copy(), B0.copy()
        for p, q in zip(P, Q):
            AX[:, p] = Av[:, q]
            BX[:, p] = Bv[:, q]
        Tt = np.zeros((n, n))
        Tt[np.ix_(P, P)] = np.linalg.inv((Ai0 @ AX)[np.ix_(P, P)])
        M = Ai0 @ BX - Ai0 @ B0 @ Ai0 @ AX                                   # F.7
        Y = Ai0 @ B0 @ M                                                       # F.9
        lhs = np.trace(np.linalg.inv(AX) @ BX @ np.linalg.inv(AX) @ BX)
        rhs = np.trace(Ai0 @ B0 @ Ai0 @ B0) + np.trace(Tt @ M @ Tt @ M) + 2 * np.trace(Tt @ Y)   # F.8
        assert abs(lhs - rhs) < 1e-10 * max(1.0, abs(lhs)), (P, Q, lhs, rhs)
    # (ii) what the CUDA table route of the backflow kernel assembles, against brute force over the
    # 3 N_e coordinates: B_l = d_l A dense (rows of both spins couple through the Jacobian J of the backflow map),
    #   E2_X = sum_l (Tr(A^-1 d_l A)^up + Tr(..)^dn)^2 - sum_l Tr((A^-1 d_l A)^2)^up - (..)^dn
    # from per-spin tables T, E[q][p][l] (= M_l[p][q] of F.7 for B_l), Y2[q][p] (= sum_l Y_l[p][q] of F.9), division-free:
    #   R^up R^dn E2_X = R^up R^dn E2_0 + 2 R^dn t0.e~^up + 2 R^up t0.e~^dn + 2 e~^up.e~^dn + R^dn b^up + R^up b^dn
    n_up, n_dn, nv = 4, 3, 3
    ne = n_up + n_dn
    nc = 3 * ne
    J = rng.standard_normal((ne, 3, nc)) * 0.3
    for i in range(ne):
        for a in range(3):
            J[i, a, 3 * i + a] += 1.0
    spins = [(0, n_up), (n_up, n_dn)]
    A0s = [rng.standard_normal((m, m)) for _, m in spins]
    Avs = [rng.standard_normal((m, nv)) for _, m in spins]
    V0s = [rng.standard_normal((3, m, m)) for _, m in spins]
    Vvs = [rng.standard_normal((3, m, nv)) for _, m in spins]

    def brute(exc):
        t1, s2, D = np.zeros((2, nc)), np.zeros(2), np.zeros(2)
        for sp, (e0, m) in enumerate(spins):
            A, V = A0s[sp].copy(), V0s[sp].copy()
            for p, q in zip(*exc[sp]):
                A[:, p] = Avs[sp][:, q]
                V[:, :, p] = Vvs[sp][:, :, q]
            Ai = np.linalg.inv(A)
            D[sp] = np.linalg.det(A)
            for l in range(nc):
                G = Ai @ sum(V[a] * J[e0:e0 + m, a, l][:, None] for a in range(3))
                t1[sp, l] = np.trace(G)
                s2[sp] += np.trace(G @ G)
        return D, np.sum((t1[0] + t1[1]) ** 2) - s2[0] - s2[1]

    tab = []
    for sp, (e0, m) in enumerate(spins):
        rho = np.linalg.inv(A0s[sp])
        T = rho @ Avs[sp]
        W0 = np.array([V0s[sp][a] @ rho for a in range(3)])
        mm = np.array([Vvs[sp][a] - V0s[sp][a] @ T for a in range(3)])
        Js = J[e0:e0 + m]
        g0 = np.array([[W0[a][i][i] for a in range(3)] for i in range(m)])
        C = np.einsum('ial,jbl->iajb', Js, Js)
        tab.append(dict(T=T, t0=np.einsum('ial,ia->l', Js, g0), E=np.einsum('ial,aiq,pi->qpl', Js, mm, rho),
                        s0=np.einsum('iajb,aij,bji->', C, W0, W0), Y2=np.einsum('iajb,aij,bjq,pi->qp', C, W0, mm, rho),
                        D0=np.linalg.det(A0s[sp])))
    t0 = tab[0]['t0'] + tab[1]['t0']
    E2_0 = t0 @ t0 - tab[0]['s0'] - tab[1]['s0']
    cases = [(([], []), ([], [])), (([1], [2]), ([], [])), (([], []), ([0], [1])), (([2], [0]), ([1], [2])),
             (([0, 3], [1, 2]), ([], [])), (([1, 2], [0, 2]), ([0, 2], [0, 1])), (([0], [0]), ([1, 2], [1, 2]))]
    for exc in cases:
        R, et, b = [1.0, 1.0], [np.zeros(nc), np.zeros(nc)], [0.0, 0.0]
        for sp in range(2):
            P, Q = exc[sp]
            tb = tab[sp]
            if len(P) == 1:
                R[sp], et[sp], b[sp] = tb['T'][P[0], Q[0]], tb['E'][Q[0], P[0]], -2 * tb['Y2'][Q[0], P[0]]
            elif len(P) == 2:
                TPQ = tb['T'][np.ix_(P, Q)]
                R[sp] = np.linalg.det(TPQ)
                adj = np.array([[TPQ[1, 1], -TPQ[0, 1]], [-TPQ[1, 0], TPQ[0, 0]]])
                Ml = np.array([[tb['E'][Q[bb], P[aa]] for bb in range(2)] for aa in range(2)])
                Y2 = np.array([[tb['Y2'][Q[bb], P[aa]] for bb in range(2)] for aa in range(2)])
                et[sp] = sum(adj[bb, aa] * Ml[aa, bb] for aa in range(2) for bb in range(2))
                b[sp] = 2 * np.sum(Ml[0, 0] * Ml[1, 1] - Ml[0, 1] * Ml[1, 0]) - 2 * sum(adj[bb, aa] * Y2[aa, bb] for aa in range(2) for bb in range(2))
        got = R[0] * R[1] * E2_0 + 2 * R[1] * (t0 @ et[0]) + 2 * R[0] * (t0 @ et[1]) + 2 * (et[0] @ et[1]) + R[1] * b[0] + R[0] * b[1]
        D, E2 = brute(exc)
        assert np.allclose([D[0] / tab[0]['D0'], D[1] / tab[1]['D0']], R, rtol=1e-10)
        assert abs(R[0] * R[1] * E2 - got) < 1e-10 * max(1.0, abs(got)), (exc, R[0] * R[1] * E2, got)
