"""ctypes binding of the CPU oracle (oracle/qmc_oracle.c).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from
the CUDA package; it takes any object with the attribute names of
`workloads.SystemDesc` (plain numpy arrays).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libqmc_oracle.so")
_SO_LD = os.path.join(_HERE, "libqmc_oracle_ld.so")  # the same source with real = long double (the adjudicator)
_SRC = os.path.join(_HERE, "qmc_oracle.c")
_lock = threading.Lock()
_libs = {}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math, no contraction): the float64 build and, from the same
    source, the extended-precision build (-DORACLE_REAL="long double", x87 80-bit) that adjudicates walkers on
    which two float64 evaluations cannot agree to the parity bound (reading Q24)."""
    hdr = os.path.join(_HERE, "qmc_oracle.h")
    for so, extra in ((_SO, []), (_SO_LD, ['-DORACLE_REAL=long double'])):
        stale = (not os.path.exists(so)) or any(os.path.getmtime(f) > os.path.getmtime(so) for f in (_SRC, hdr))
        if force or stale:
            subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared"] + extra +
                                  ["-o", so, _SRC, "-lm"])
    return _SO


class _Desc(C.Structure):
    _fields_ = [
        ("n_atoms", C.c_int32), ("atom_xyz", C.c_void_p), ("atom_Z", C.c_void_p),
        ("n_up", C.c_int32), ("n_dn", C.c_int32),
        ("n_ao", C.c_int32), ("ao_atom", C.c_void_p), ("ao_n", C.c_void_p), ("ao_l", C.c_void_p),
        ("ao_m", C.c_void_p), ("ao_zeta", C.c_void_p), ("ao_norm", C.c_void_p),
        ("n_mo", C.c_int32), ("mo_coeff", C.c_void_p),
        ("n_det", C.c_int32), ("det_up", C.c_void_p), ("det_dn", C.c_void_p), ("ci_coeff", C.c_void_p),
        ("jastrow_a_par", C.c_double), ("jastrow_a_anti", C.c_double), ("jastrow_b", C.c_double),
        ("jastrow_en_w0", C.c_double), ("jastrow_en_w1", C.c_double), ("jastrow_en_w2", C.c_double),
        ("n_een", C.c_int32), ("een_params", C.c_void_p), ("backflow_w", C.c_double),
    ]


def lib(extended: bool = False):
    """The float64 oracle, or with extended=True the long-double build of the same source."""
    with _lock:
        if extended not in _libs:
            build()
            L = C.CDLL(_SO_LD if extended else _SO)
            L.oracle_sto_norm.restype = C.c_double
            L.oracle_sto_norm.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double]
            L.oracle_det_inv.restype = C.c_double
            L.oracle_det_inv.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
            L.oracle_psi_plain.restype = C.c_double
            L.oracle_psi_plain.argtypes = [C.c_void_p, C.c_void_p]
            L.oracle_ao_eval.restype = None
            L.oracle_ao_eval.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
            L.oracle_local_energy.restype = C.c_int
            L.oracle_local_energy.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64,
                                              C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
            L.oracle_philox4x32_10.restype = None
            L.oracle_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
            L.oracle_walker_draws.restype = None
            L.oracle_walker_draws.argtypes = [C.c_uint64, C.c_int64, C.c_uint64, C.c_int, C.c_void_p, C.c_void_p]
            L.oracle_metropolis.restype = C.c_int
            L.oracle_metropolis.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64,
                                            C.c_double, C.c_int32, C.c_uint64, C.c_uint64,
                                            C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
            L.oracle_batch_stats.restype = None
            L.oracle_batch_stats.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
            L.oracle_log_derivatives.restype = C.c_int
            L.oracle_log_derivatives.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p]
            L.oracle_orbital_derivatives.restype = C.c_int
            L.oracle_orbital_derivatives.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p,
                                                     C.c_void_p]
            L.oracle_nuclear_log_gradient.restype = C.c_int
            L.oracle_nuclear_log_gradient.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p]
            L.oracle_energy_gradient.restype = None
            L.oracle_energy_gradient.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
            L.oracle_backflow_coords.restype = None
            L.oracle_backflow_coords.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
            L.oracle_ao_eval2.restype = None
            L.oracle_ao_eval2.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
            L.oracle_nuclear_energy_gradient.restype = C.c_int
            L.oracle_nuclear_energy_gradient.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p]
            L.oracle_force.restype = None
            L.oracle_force.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
            _libs[extended] = L
    return _libs[extended]


def _p(a):
    return None if a is None else a.ctypes.data


class OracleSystem:
    """Holds contiguous copies of the description arrays + the C struct."""

    def __init__(self, d, extended: bool = False):
        self.L = lib(extended)
        f64 = lambda a: np.ascontiguousarray(a, np.float64)
        i32 = lambda a: np.ascontiguousarray(a, np.int32)
        self.n_up, self.n_dn = int(d.n_up), int(d.n_dn)
        self.n_e = self.n_up + self.n_dn
        self._keep = dict(
            atom_xyz=f64(d.atom_xyz), atom_Z=f64(d.atom_Z), ao_atom=i32(d.ao_atom), ao_n=i32(d.ao_n),
            ao_l=i32(d.ao_l), ao_m=i32(d.ao_m), ao_zeta=f64(d.ao_zeta),
            ao_norm=None if d.ao_norm is None else f64(d.ao_norm), mo_coeff=f64(d.mo_coeff),
            det_up=i32(d.det_up), det_dn=i32(d.det_dn), ci_coeff=f64(d.ci_coeff))
        k = self._keep
        self.n_ao = int(k["ao_atom"].shape[0])
        self.c = _Desc(int(k["atom_xyz"].shape[0]), _p(k["atom_xyz"]), _p(k["atom_Z"]), self.n_up, self.n_dn,
                       self.n_ao, _p(k["ao_atom"]), _p(k["ao_n"]), _p(k["ao_l"]), _p(k["ao_m"]),
                       _p(k["ao_zeta"]), _p(k["ao_norm"]), int(k["mo_coeff"].shape[1]), _p(k["mo_coeff"]),
                       int(k["ci_coeff"].shape[0]), _p(k["det_up"]), _p(k["det_dn"]), _p(k["ci_coeff"]),
                       float(d.jastrow_a_par), float(d.jastrow_a_anti), float(d.jastrow_b),
                 float(getattr(d, "jastrow_en_w0", 0.0)), float(getattr(d, "jastrow_en_w1", 0.0)),
                 float(getattr(d, "jastrow_en_w2", 0.0)), 0, None, float(getattr(d, "backflow_w", 0.0)))
        een = getattr(d, "jastrow_een", None)
        if een is not None and len(een):
            k["een"] = np.ascontiguousarray(een, np.float64).reshape(-1, 7)
            self.c.n_een, self.c.een_params = int(k["een"].shape[0]), _p(k["een"])
        self.ref = C.addressof(self.c)


def _ranges(M, n):
    n = max(1, min(n, M))
    edges = np.linspace(0, M, n + 1).astype(np.int64)
    return [(int(edges[i]), int(edges[i + 1])) for i in range(n) if edges[i + 1] > edges[i]]


def sto_norm(n, l, m, zeta):
    return lib().oracle_sto_norm(n, l, m, zeta)


def det_inv(A):
    A = np.ascontiguousarray(A, np.float64)
    n = A.shape[0]
    inv = np.empty_like(A)
    d = lib().oracle_det_inv(n, _p(A), _p(inv))
    return d, inv


def ao_eval(sysd: OracleSystem, ao: int, xyz):
    xyz = np.ascontiguousarray(xyz, np.float64)
    out = np.empty(5)
    sysd.L.oracle_ao_eval(sysd.ref, ao, _p(xyz), _p(out))
    return out


def psi_plain(sysd: OracleSystem, r_aos):
    """r_aos: [n_e,3] one walker."""
    r = np.ascontiguousarray(r_aos, np.float64)
    return sysd.L.oracle_psi_plain(sysd.ref, _p(r))


def local_energy(sysd: OracleSystem, r_soa, threads: int = 1, parts: bool = False):
    """r_soa: float64 [n_e,3,M].  Returns logpsi, sign, eloc[, parts[M,4]]."""
    r = np.ascontiguousarray(r_soa, np.float64)
    M = r.shape[2]
    lp, sg, el = np.empty(M), np.empty(M), np.empty(M)
    pt = np.empty((M, 4)) if parts else None
    L = sysd.L

    def run(rng):
        rc = L.oracle_local_energy(sysd.ref, _p(r), M, rng[0], rng[1], _p(lp), _p(sg), _p(el), _p(pt))
        assert rc == 0

    rs = _ranges(M, threads)
    if len(rs) == 1:
        run(rs[0])
    else:
        with ThreadPoolExecutor(len(rs)) as ex:
            list(ex.map(run, rs))
    return (lp, sg, el, pt) if parts else (lp, sg, el)


def philox(ctr, key):
    c = np.ascontiguousarray(ctr, np.uint32)
    k = np.ascontiguousarray(key, np.uint32)
    out = np.empty(4, np.uint32)
    lib().oracle_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def walker_draws(seed, w, sweep, n_coord):
    z = np.empty(n_coord + 1)
    u = C.c_double()
    lib().oracle_walker_draws(seed, w, sweep, n_coord, _p(z), C.addressof(u))
    return z[:n_coord].copy(), u.value


def metropolis(sysd: OracleSystem, r_soa, step, n_sweeps, seed, sweep_offset=0, threads: int = 1,
               want_eloc_acc: bool = False):
    """Returns dict(r, logpsi, sign, accept[n_sweeps,M], margin[n_sweeps,M], eloc_acc)."""
    r = np.array(r_soa, np.float64, order="C", copy=True)
    M = r.shape[2]
    lp, sg = np.empty(M), np.empty(M)
    acc = np.zeros((n_sweeps, M), np.uint8)
    mg = np.zeros((n_sweeps, M))
    ea = np.zeros(M) if want_eloc_acc else None
    L = sysd.L

    def run(rng):
        rc = L.oracle_metropolis(sysd.ref, _p(r), M, rng[0], rng[1], step, n_sweeps, seed, sweep_offset,
                                 _p(lp), _p(sg), _p(acc), _p(mg), _p(ea))
        assert rc == 0

    rs = _ranges(M, threads)
    if len(rs) == 1:
        run(rs[0])
    else:
        with ThreadPoolExecutor(len(rs)) as ex:
            list(ex.map(run, rs))
    return dict(r=r, logpsi=lp, sign=sg, accept=acc, margin=mg, eloc_acc=ea)


def batch_stats(x):
    x = np.ascontiguousarray(x, np.float64)
    m, s = C.c_double(), C.c_double()
    lib().oracle_batch_stats(_p(x), x.shape[0], C.addressof(m), C.addressof(s))
    return m.value, s.value


def log_derivatives(sysd: OracleSystem, r_soa, threads: int = 1):
    """O[M, 6 + 7 n_een + n_det (+ 1)] = (dPsi/dtheta)/Psi for theta = (a_par, a_anti, b, en_w0, en_w1, en_w2,
    the seven parameters of every e-e-n term in een_params order, d_0 .. d_{n_det-1}, and -- with backflow on -- the
    backflow weight w)  (eq. 6)."""
    r = np.ascontiguousarray(r_soa, np.float64)
    M = r.shape[2]
    O = np.empty((M, 6 + 7 * int(sysd.c.n_een) + int(sysd.c.n_det) + (1 if float(sysd.c.backflow_w) != 0.0 else 0)))
    L = sysd.L

    def run(rng):
        rc = L.oracle_log_derivatives(sysd.ref, _p(r), M, rng[0], rng[1], _p(O))
        assert rc == 0

    rs = _ranges(M, threads)
    if len(rs) == 1:
        run(rs[0])
    else:
        with ThreadPoolExecutor(len(rs)) as ex:
            list(ex.map(run, rs))
    return O


def energy_gradient(eloc, O):
    """eq. 6: (E_v, grad[n_param]) with grad_p = (2/M) sum_m O[m,p] (E_L[m] - E_v)."""
    e = np.ascontiguousarray(eloc, np.float64)
    Oc = np.ascontiguousarray(O, np.float64)
    ev = C.c_double()
    g = np.empty(Oc.shape[1])
    lib().oracle_energy_gradient(_p(e), _p(Oc), e.shape[0], Oc.shape[1], C.addressof(ev), _p(g))
    return ev.value, g


def orbital_derivatives(sysd: OracleSystem, r_soa, threads: int = 1):
    """(dC[M, n_ao, n_mo], dzeta[M, n_ao]) = d ln Psi / d C[beta][alpha], d ln Psi / d zeta_beta."""
    r = np.ascontiguousarray(r_soa, np.float64)
    M = r.shape[2]
    dC = np.empty((M, sysd.n_ao, int(sysd.c.n_mo)))
    dz = np.empty((M, sysd.n_ao))
    L = sysd.L

    def run(rng):
        rc = L.oracle_orbital_derivatives(sysd.ref, _p(r), M, rng[0], rng[1], _p(dC), _p(dz))
        assert rc == 0

    rs = _ranges(M, threads)
    if len(rs) == 1:
        run(rs[0])
    else:
        with ThreadPoolExecutor(len(rs)) as ex:
            list(ex.map(run, rs))
    return dC, dz


def nuclear_log_gradient(sysd: OracleSystem, r_soa, threads: int = 1):
    """dR[M, n_atoms, 3] = grad_alpha ln|Psi| (eq. 7's grad_alpha ln rho / 2)."""
    r = np.ascontiguousarray(r_soa, np.float64)
    M = r.shape[2]
    dR = np.empty((M, int(sysd.c.n_atoms), 3))
    L = sysd.L

    def run(rng):
        rc = L.oracle_nuclear_log_gradient(sysd.ref, _p(r), M, rng[0], rng[1], _p(dR))
        assert rc == 0

    rs = _ranges(M, threads)
    if len(rs) == 1:
        run(rs[0])
    else:
        with ThreadPoolExecutor(len(rs)) as ex:
            list(ex.map(run, rs))
    return dR


def ao_eval2(sysd: OracleSystem, ao: int, xyz):
    """{phi, grad[3], lap, Hessian xx yy zz xy yz zx, grad lap[3]} of one AO at one point."""
    xyz = np.ascontiguousarray(xyz, np.float64)
    out = np.empty(14)
    sysd.L.oracle_ao_eval2(sysd.ref, ao, _p(xyz), _p(out))
    return out


def nuclear_energy_gradient(sysd: OracleSystem, r_soa, threads: int = 1):
    """dE[M, n_atoms, 3] = grad_alpha E_L (first term of eq. 7); Pade e-e Jastrow only."""
    r = np.ascontiguousarray(r_soa, np.float64)
    M = r.shape[2]
    dE = np.empty((M, int(sysd.c.n_atoms), 3))
    L = sysd.L

    def run(rng):
        rc = L.oracle_nuclear_energy_gradient(sysd.ref, _p(r), M, rng[0], rng[1], _p(dE))
        assert rc == 0, rc

    rs = _ranges(M, threads)
    if len(rs) == 1:
        run(rs[0])
    else:
        with ThreadPoolExecutor(len(rs)) as ex:
            list(ex.map(run, rs))
    return dE


def force(eloc, dE, dlnpsi):
    """eq. 7: (F[n_atoms, 3], terms[2, n_atoms, 3]) from E_L [M], grad_alpha E_L and grad_alpha ln|Psi| [M, n_atoms, 3]."""
    e = np.ascontiguousarray(eloc, np.float64)
    a = np.ascontiguousarray(dE, np.float64)
    b = np.ascontiguousarray(dlnpsi, np.float64)
    na = a.shape[1]
    F = np.empty((na, 3))
    T = np.empty((2, na, 3))
    lib().oracle_force(_p(e), _p(a), _p(b), e.shape[0], na, _p(F), _p(T))
    return F, T


def backflow_coords(sysd: OracleSystem, r_aos):
    """rt [n_e, 3] of one walker r [n_e, 3]."""
    r = np.ascontiguousarray(r_aos, np.float64)
    rt = np.empty_like(r)
    sysd.L.oracle_backflow_coords(sysd.ref, _p(r), _p(rt))
    return rt
