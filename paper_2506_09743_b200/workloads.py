"""Seeded synthetic inputs: the five BASELINE.json configs as plain arrays.

This module is the ONLY thing the CUDA path and the CPU oracle have in common.
It holds none of the method's arithmetic (no orbital, determinant, Jastrow,
energy or sampler code): it only draws numbers and lays out index lists.  The
recipe is SURVEY.md section 8(d) and DESIGN.md "Input recipe":

    rng = np.random.default_rng([config_index, 0]); draw order
    (1) zeta per shell, (2) MO matrix by QR of a normal matrix,
    (3) determinant selection, (4) CI coefficients, (5) walkers.

The molecules are *shaped* like the paper's H2 / LiH / Li2 / CO (PAPER.md:97,
178, 190-193: two atoms, 2/4/6/14 electrons, DZP-like STO shells, SD-type CI
expansions); the paper's ADF/DZP data is not available and is not recreated.
"""
from __future__ import annotations

import itertools
import math
from dataclasses import dataclass, field

import numpy as np

# shell kinds: (label, n, l, number of real harmonics)
_SHELL = {"1s": (1, 0, 1), "2s": (2, 0, 1), "2p": (2, 1, 3), "3d": (3, 2, 5)}


@dataclass
class SystemDesc:
    """Everything `qmc_setup` takes (include/qmc.h), as numpy arrays."""

    name: str
    atom_xyz: np.ndarray  # [n_atoms,3] bohr
    atom_Z: np.ndarray  # [n_atoms]
    n_up: int
    n_dn: int
    ao_atom: np.ndarray  # [n_ao] int32
    ao_n: np.ndarray  # [n_ao] int32 principal quantum number 1..3
    ao_l: np.ndarray  # [n_ao] int32 0..2
    ao_m: np.ndarray  # [n_ao] int32 index into the real solid harmonics of l
    ao_zeta: np.ndarray  # [n_ao]
    ao_norm: np.ndarray | None  # [n_ao] or None = standard normalisation
    mo_coeff: np.ndarray  # [n_ao, n_mo] row-major
    det_up: np.ndarray  # [n_det, n_up] int32 ordered MO column lists
    det_dn: np.ndarray  # [n_det, n_dn] int32
    ci_coeff: np.ndarray  # [n_det]
    jastrow_a_par: float = 0.25
    jastrow_a_anti: float = 0.5
    jastrow_b: float = 1.0
    jastrow_en_w0: float = 0.0  # electron-nucleus kernel (D.2), all zero = absent
    jastrow_en_w1: float = 0.0
    jastrow_en_w2: float = 0.0
    jastrow_een: np.ndarray | None = None  # electron-electron-nucleus kernel (D.3): [n_terms, 7] = (c, a1, b1, a2, b2, a3, b3)
    backflow_w: float = 0.0  # inverse backflow kernel K_BF(r) = w / r; 0 = none
    extra: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.atom_xyz.shape[0])

    @property
    def n_e(self) -> int:
        return self.n_up + self.n_dn

    @property
    def n_ao(self) -> int:
        return int(self.ao_atom.shape[0])

    @property
    def n_mo(self) -> int:
        return int(self.mo_coeff.shape[1])

    @property
    def n_det(self) -> int:
        return int(self.ci_coeff.shape[0])


def expand_shells(shells_per_atom, zeta_per_shell):
    """shells_per_atom: list (per atom) of shell labels; zeta_per_shell: flat
    list in the same atom-major order.  Returns per-AO arrays."""
    ao_atom, ao_n, ao_l, ao_m, ao_zeta = [], [], [], [], []
    k = 0
    for a, shells in enumerate(shells_per_atom):
        for lab in shells:
            n, l, nm = _SHELL[lab]
            for m in range(nm):
                ao_atom.append(a)
                ao_n.append(n)
                ao_l.append(l)
                ao_m.append(m)
                ao_zeta.append(zeta_per_shell[k])
            k += 1
    assert k == len(zeta_per_shell)
    return (np.array(ao_atom, np.int32), np.array(ao_n, np.int32), np.array(ao_l, np.int32),
            np.array(ao_m, np.int32), np.array(ao_zeta, np.float64))


# --------------------------------------------------------------------------
# SD(n_el, n_orb) excitation pools
# --------------------------------------------------------------------------

def excitation_pool(n_occ: int, virt: list[int]):
    """All single and double substitutions of the reference (0..n_occ-1 in both
    spins) into the virtual window `virt`, as ordered column lists obtained by
    in-place substitution.  Classes in the order
    [alpha-single, beta-single, alpha-beta, alpha-alpha, beta-beta], each
    enumerated lexicographically (occupied positions, then virtuals).
    Returns a list of 5 lists of (up_list, dn_list) tuples."""
    ref = tuple(range(n_occ))

    def singles():
        out = []
        for p in range(n_occ):
            for q in virt:
                lst = list(ref)
                lst[p] = q
                out.append(tuple(lst))
        return out

    def doubles():
        out = []
        for p1, p2 in itertools.combinations(range(n_occ), 2):
            for q1, q2 in itertools.combinations(virt, 2):
                lst = list(ref)
                lst[p1] = q1
                lst[p2] = q2
                out.append(tuple(lst))
        return out

    s, d = singles(), doubles()
    return [
        [(u, ref) for u in s],
        [(ref, v) for v in s],
        [(u, v) for u in s for v in s],
        [(u, ref) for u in d],
        [(ref, v) for v in d],
    ]


def sd_count(n_el: int, n_orb: int) -> int:
    """Number of determinants of the paper's SD(n_el, n_orb) active space:
    ground + singles + doubles, n_el/2 occupied of n_orb orbitals per spin."""
    o = n_el // 2
    virt = list(range(o, n_orb))
    return 1 + sum(len(c) for c in excitation_pool(o, virt))


def select_determinants(rng, n_occ: int, virt: list[int], n_det: int):
    """Reading Q12: shuffle each class with the config RNG, deal round-robin
    until n_det-1 excited determinants are chosen; determinant 0 = reference."""
    classes = excitation_pool(n_occ, virt)
    for c in classes:
        perm = rng.permutation(len(c))
        c[:] = [c[i] for i in perm]
    ref = tuple(range(n_occ))
    chosen = [(ref, ref)]
    ptr = [0] * len(classes)
    ci = 0
    while len(chosen) < n_det:
        if all(ptr[k] >= len(classes[k]) for k in range(len(classes))):
            raise ValueError("excitation pool exhausted")
        k = ci % len(classes)
        ci += 1
        if ptr[k] < len(classes[k]):
            chosen.append(classes[k][ptr[k]])
            ptr[k] += 1
    up = np.array([c[0] for c in chosen], np.int32).reshape(len(chosen), n_occ)
    dn = np.array([c[1] for c in chosen], np.int32).reshape(len(chosen), n_occ)
    return up, dn


# --------------------------------------------------------------------------
# walkers
# --------------------------------------------------------------------------

def make_walkers(rng, atom_xyz: np.ndarray, n_e: int, M: int) -> np.ndarray:
    """Electron coordinates N(nucleus picked uniformly, sigma = 1 bohr), in the
    SoA layout the library uses: float64 [n_e][3][M] (walker index fastest)."""
    nuc = rng.integers(0, atom_xyz.shape[0], (M, n_e))
    r = atom_xyz[nuc] + rng.standard_normal((M, n_e, 3))
    return np.ascontiguousarray(r.transpose(1, 2, 0))


# --------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------

_HEAVY = ["1s", "1s", "2s", "2s", "2p", "2p", "3d"]  # 15 AOs per atom


def _orthonormal(rng, n):
    g = rng.standard_normal((n, n))
    q, _ = np.linalg.qr(g)
    return np.ascontiguousarray(q)


def h2(M: int = 1024):
    """BASELINE.json configs[0]."""
    rng = np.random.default_rng([0, 0])
    R, zeta = 1.4, 1.24
    atom_xyz = np.array([[0, 0, -R / 2], [0, 0, R / 2]], np.float64)
    ao = expand_shells([["1s"], ["1s"]], [zeta, zeta])
    # overlap of two normalised 1s STOs, the config's stated closed form for c
    x = zeta * R
    S = math.exp(-x) * (1 + x + x * x / 3)
    c = 1.0 / math.sqrt(2 * (1 + S))
    sysd = SystemDesc("H2", atom_xyz, np.array([1.0, 1.0]), 1, 1, *ao, None,
                      np.array([[c], [c]], np.float64),
                      np.zeros((1, 1), np.int32), np.zeros((1, 1), np.int32), np.array([1.0]),
                      extra=dict(sweeps=10, step=0.5, overlap=S))
    return sysd, make_walkers(rng, atom_xyz, 2, M)


def lih(M: int = 8192):
    """BASELINE.json configs[1]."""
    rng = np.random.default_rng([1, 0])
    atom_xyz = np.array([[0, 0, 0], [0, 0, 3.015]], np.float64)
    shells = [["1s", "1s", "2s", "2s", "2p"], ["1s", "1s", "2p"]]
    zeta = rng.uniform(0.5, 3.5, sum(len(s) for s in shells))
    ao = expand_shells(shells, zeta)
    C = _orthonormal(rng, 12)[:, :2].copy()
    ref = np.arange(2, dtype=np.int32)[None, :]
    sysd = SystemDesc("LiH", atom_xyz, np.array([3.0, 1.0]), 2, 2, *ao, None, C,
                      ref.copy(), ref.copy(), np.array([1.0]),
                      extra=dict(sweeps=10, step=0.3))
    return sysd, make_walkers(rng, atom_xyz, 4, M)


def _heavy_diatomic(idx, name, Z, R, origin_centered, n_occ, n_mo, n_det, c0, s, zlo, zhi, M,
                    shells=None, extra=None, with_walkers=True):
    rng = np.random.default_rng([idx, 0])
    if origin_centered:
        atom_xyz = np.array([[0, 0, -R / 2], [0, 0, R / 2]], np.float64)
    else:
        atom_xyz = np.array([[0, 0, 0], [0, 0, R]], np.float64)
    shells = shells or [list(_HEAVY), list(_HEAVY)]
    zeta = rng.uniform(zlo, zhi, sum(len(x) for x in shells))
    ao = expand_shells(shells, zeta)
    n_ao = len(ao[0])
    C = _orthonormal(rng, n_ao)[:, :n_mo].copy()
    up, dn = select_determinants(rng, n_occ, list(range(n_occ, n_mo)), n_det)
    ci = np.concatenate([[c0], rng.normal(0.0, s, n_det - 1)])
    sysd = SystemDesc(name, atom_xyz, np.array(Z, np.float64), n_occ, n_occ, *ao, None, C, up, dn, ci,
                      extra=extra or {})
    walkers = make_walkers(rng, atom_xyz, 2 * n_occ, M) if with_walkers else None
    return sysd, walkers


def li2(M: int = 32768, variant: str = "30"):
    """BASELINE.json configs[2].  variant "30" = the listed composition
    (15 AOs/atom); "28" = reading Q1's alternative (second 2s dropped)."""
    shells = None
    if variant == "28":
        sh = ["1s", "1s", "2s", "2p", "2p", "3d"]
        shells = [list(sh), list(sh)]
    return _heavy_diatomic(2, "Li2" if variant == "30" else "Li2-28", [3, 3], 5.051, True, 3, 8, 20,
                           0.95, 0.05, 0.3, 4.0, M, shells=shells, extra=dict(sweeps=10, step=0.3))


def co(M: int = 131072, n_det: int = 100):
    """BASELINE.json configs[3] (the headline workload)."""
    return _heavy_diatomic(3, "CO", [6, 8], 2.132, False, 7, 14, n_det, 0.9, 0.03, 0.5, 9.0, M,
                           extra=dict(sweeps=20, step=0.2))


def co_scan(M: int = 262144, n_geom: int = 16, n_det: int = 500):
    """BASELINE.json configs[4]: 16 bond lengths 1.6 + 0.16 k; zeta, C, the
    determinant list and the CI coefficients are the same at every geometry
    (reading Q14); walkers are drawn per geometry around that geometry's
    nuclei.  Returns a list of (SystemDesc, walkers)."""
    out = []
    base, _ = _heavy_diatomic(4, "CO-scan", [6, 8], 1.6, False, 7, 14, n_det, 0.85, 0.02, 0.5, 9.0, 1,
                              extra=dict(sweeps=50, step=0.2), with_walkers=False)
    for k in range(n_geom):
        R = 1.6 + 0.16 * k
        xyz = np.array([[0, 0, 0], [0, 0, R]], np.float64)
        s = SystemDesc(f"CO-scan[{k}] R={R:.2f}", xyz, base.atom_Z, 7, 7, base.ao_atom, base.ao_n,
                       base.ao_l, base.ao_m, base.ao_zeta, None, base.mo_coeff, base.det_up,
                       base.det_dn, base.ci_coeff, extra=dict(sweeps=50, step=0.2, R=R))
        wr = np.random.default_rng([4, 1 + k])
        out.append((s, make_walkers(wr, xyz, 14, M)))
    return out


CONFIGS = {"H2": h2, "LiH": lih, "Li2": li2, "CO": co}
