"""Small builders for hand-made systems used by the pins and parity tests."""
import numpy as np

from paper_2506_09743_b200.workloads import SystemDesc


def atom_system(Z, aos, C, n_up, n_dn, det_up=None, det_dn=None, ci=None, norm=None,
                a_par=0.0, a_anti=0.0, b=1.0, xyz=(0.0, 0.0, 0.0)):
    """One nucleus at xyz.  aos: list of (n, l, m, zeta)."""
    n_ao = len(aos)
    C = np.asarray(C, np.float64).reshape(n_ao, -1)
    if det_up is None:
        det_up = np.arange(n_up, dtype=np.int32)[None, :]
    if det_dn is None:
        det_dn = np.arange(n_dn, dtype=np.int32)[None, :]
    det_up = np.asarray(det_up, np.int32)
    det_dn = np.asarray(det_dn, np.int32)
    nd = det_up.shape[0] if n_up else det_dn.shape[0]
    det_up = det_up.reshape(nd, n_up)
    det_dn = det_dn.reshape(nd, n_dn)
    if ci is None:
        ci = np.ones(det_up.shape[0])
    return SystemDesc(
        "atom", np.array([xyz], np.float64), np.array([float(Z)]), n_up, n_dn,
        np.zeros(n_ao, np.int32), np.array([a[0] for a in aos], np.int32),
        np.array([a[1] for a in aos], np.int32), np.array([a[2] for a in aos], np.int32),
        np.array([a[3] for a in aos], np.float64), None if norm is None else np.asarray(norm, np.float64),
        C, det_up, det_dn, np.asarray(ci, np.float64), a_par, a_anti, b)


def soa(r_aos):
    """[M,n_e,3] -> [n_e,3,M]"""
    return np.ascontiguousarray(np.asarray(r_aos, np.float64).transpose(1, 2, 0))


def hydrogenic_set(Z):
    """Seven exact hydrogenic orbitals of nuclear charge Z as (AO list, C, energies).
    AOs (unnormalised via norm=1): 0: 1s zeta=Z; 1: 1s-type zeta=Z/2; 2: 2s-type (r e^{-Z r/2});
    3..5: 2p x,y,z zeta=Z/2; 6..10: 3d (5 harmonics) zeta=Z/3.
    MOs: 1s; 2s = 2*[1] - Z*[2]; 2px, 2py, 2pz; 3d_xy; 3d_z2; remaining d as extra columns."""
    aos = [(1, 0, 0, Z), (1, 0, 0, Z / 2), (2, 0, 0, Z / 2), (2, 1, 0, Z / 2), (2, 1, 1, Z / 2),
           (2, 1, 2, Z / 2)] + [(3, 2, m, Z / 3) for m in range(5)]
    n_ao = len(aos)
    cols = []
    e = []

    def col(**kw):
        v = np.zeros(n_ao)
        for k, x in kw.items():
            v[int(k[1:])] = x
        return v

    cols.append(col(a0=1.0)); e.append(-Z * Z / 2)
    cols.append(col(a1=2.0, a2=-float(Z))); e.append(-Z * Z / 8)
    for k in (3, 4, 5):
        cols.append(col(**{f"a{k}": 1.0})); e.append(-Z * Z / 8)
    for k in (6, 10, 7, 8, 9):
        cols.append(col(**{f"a{k}": 1.0})); e.append(-Z * Z / 18)
    return aos, np.stack(cols, axis=1), np.array(e)


def adjudicate(gpu, o64, ox, tol, scale=None, mask=None, what=""):
    """Parity with adjudication by the extended-precision oracle (reading Q24).

    gpu / o64 / ox: the CUDA result, the float64 oracle's and the long-double build's of the same oracle source,
    arrays whose first axis is the walker.  Per walker (max over the other axes), with e = |.|/scale:
      * where the float64 oracle is itself pinned by the extended run to a tenth of the bound, e(o64, ox) <= tol/10,
        the contract is asserted literally:  e(gpu, o64) <= tol;
      * elsewhere (counted and returned: walkers on which float64 arithmetic of this kind cannot deliver the bound --
        a nearly singular Slater matrix, a CI sum that cancels) the CUDA result must be as good as the float64
        oracle's: e(gpu, ox) <= max(tol, 4 e(o64, ox)).
    Returns the number of such exceptions inside `mask`."""
    import numpy as np
    gpu, o64, ox = (np.asarray(a, np.float64) for a in (gpu, o64, ox))
    sc = 1.0 if scale is None else np.asarray(scale, np.float64)

    def per_walker(a):
        a = np.abs(a) / sc
        return a.reshape(a.shape[0], -1).max(axis=1) if a.ndim > 1 else a

    with np.errstate(invalid="ignore"):
        e_g64, e_gx, e_64x = per_walker(gpu - o64), per_walker(gpu - ox), per_walker(o64 - ox)
    m = np.ones(e_g64.shape[0], bool) if mask is None else np.asarray(mask, bool)
    pinned = m & (e_64x <= tol / 10)
    exc = m & ~(e_64x <= tol / 10)
    bad = pinned & ~(e_g64 <= tol)
    assert not bad.any(), (what, "pinned walkers beyond the bound", [(int(i), float(e_g64[i])) for i in np.flatnonzero(bad)[:8]])
    bad = exc & ~(e_gx <= np.maximum(tol, 4 * e_64x))
    assert not bad.any(), (what, "exceptions worse than the float64 oracle",
                           [(int(i), float(e_gx[i]), float(e_64x[i])) for i in np.flatnonzero(bad)[:8]])
    return int(exc.sum())


def golden_values(name):
    """name -> float from a two-column text fixture under tests/golden (lines starting with # are citations)."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out
