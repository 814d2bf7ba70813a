"""Parity of the CUDA path (through the C ABI) against the CPU oracle, on a B200.

Tolerances are BASELINE.json north_star's: sign exact; log|Psi| 1e-10 absolute; per-walker
E_L 1e-8*max(1,|E_L|) for walkers with |Psi|/max|Psi| > 1e-6; batch mean E_L 1e-10 relative;
Metropolis accept masks bit-exact except inside the 1e-12 tie window."""
import math
import os

import numpy as np
import pytest

from paper_2506_09743_b200 import workloads as wl
from tests.helpers import adjudicate, atom_system, hydrogenic_set, soa

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import binding as ob
    from paper_2506_09743_b200 import binding as qb
    assert torch.cuda.is_available()
    qb.lib()
    return torch, ob, qb


def _to_gpu(torch, r):
    return torch.from_numpy(np.ascontiguousarray(r)).cuda()


def check_local_energy(env, d, r, threads=8, mean_rtol=1e-10):
    torch, ob, qb = env
    o = ob.OracleSystem(d)
    lp0, sg0, el0 = ob.local_energy(o, r, threads=threads)
    s = qb.QmcSystem(d)
    lp, sg, el = s.local_energy(_to_gpu(torch, r))
    lp2, sg2 = s.log_psi(_to_gpu(torch, r))
    torch.cuda.synchronize()
    lp, sg, el, lp2, sg2 = (t.cpu().numpy() for t in (lp, sg, el, lp2, sg2))
    s.close()
    assert np.array_equal(sg, sg0), f"sign mismatches: {(sg != sg0).sum()}"
    assert np.array_equal(sg2, sg0)
    assert np.max(np.abs(lp - lp0)) < 1e-10, np.max(np.abs(lp - lp0))
    assert np.max(np.abs(lp2 - lp0)) < 1e-10
    keep = lp0 - lp0.max() > math.log(1e-6)
    err = np.abs(el - el0) / np.maximum(1.0, np.abs(el0))
    assert keep.sum() > 0
    assert np.max(err[keep]) < 1e-8, (np.max(err[keep]), int(np.argmax(err * keep)))
    m0, _ = ob.batch_stats(el0)
    m1, _ = ob.batch_stats(el)
    assert abs(m1 - m0) <= mean_rtol * abs(m0), (m0, m1)
    return el0, el


@pytest.mark.parametrize("name,M", [("H2", 1024), ("LiH", 1531), ("Li2", 1027), ("CO", 1025)])
def test_local_energy_configs(env, name, M):
    d, r = wl.CONFIGS[name](M=M)
    check_local_energy(env, d, r)


def test_local_energy_li2_28(env):
    d, r = wl.li2(M=515, variant="28")
    check_local_energy(env, d, r)


def test_local_energy_co_500_determinants(env):
    d, r = wl.co_scan(M=300, n_geom=3)[2]
    check_local_energy(env, d, r)


@pytest.mark.parametrize("M", [1, 2, 3, 31, 33])
def test_ragged_and_tiny_batches(env, M):
    d, r = wl.co(M=M)
    check_local_energy(env, d, r, threads=1, mean_rtol=1e-9)
    d, r = wl.li2(M=M)
    check_local_energy(env, d, r, threads=1, mean_rtol=1e-9)


def test_hydrogenic_closed_forms_on_gpu(env):
    torch, ob, qb = env
    rng = np.random.default_rng(0)
    # P1: hydrogen atom, exact 1s
    d = atom_system(1, [(1, 0, 0, 1.0)], [[1.0]], 1, 0)
    r = soa(rng.standard_normal((257, 1, 3)) * 2)
    s = qb.QmcSystem(d)
    lp, sg, el = s.local_energy(_to_gpu(torch, r))
    assert float((el + 0.5).abs().max()) < 1e-12
    s.close()
    # P5: 7 same-spin electrons in hydrogenic orbitals + 3 opposite-spin ones
    Z = 2.0
    aos, C, e = hydrogenic_set(Z)
    d = atom_system(Z, aos, C[:, :7], 7, 3, norm=np.ones(len(aos)), det_up=[list(range(7))], det_dn=[[0, 2, 5]])
    r = rng.standard_normal((64, 10, 3)) * 2.0
    s = qb.QmcSystem(d)
    lp, sg, el = (t.cpu().numpy() for t in s.local_energy(_to_gpu(torch, soa(r))))
    s.close()
    vee = sum(1 / np.linalg.norm(r[:, i] - r[:, j], axis=1) for i in range(10) for j in range(i))
    ref = e[:7].sum() + e[[0, 2, 5]].sum() + vee
    ok = lp > lp.max() - 20
    assert np.max(np.abs(el[ok] - ref[ok]) / np.maximum(1, np.abs(ref[ok]))) < 1e-8


def test_incomplete_shells_custom_norm_and_unequal_spins(env):
    rng = np.random.default_rng(3)
    # single p / d functions out of shell order, user normalisation, n_up != n_dn, permuted reference columns
    aos = [(2, 1, 2, 1.1), (1, 0, 0, 2.0), (3, 2, 3, 0.9), (2, 1, 0, 1.3), (3, 2, 1, 0.7), (2, 0, 0, 1.5),
           (3, 0, 0, 1.2), (3, 1, 1, 0.8), (2, 1, 1, 1.3)]
    C = rng.standard_normal((len(aos), 6))
    det_up = [[4, 0, 2], [4, 5, 2], [1, 0, 2], [4, 3, 5]]
    det_dn = [[1, 3], [1, 3], [0, 3], [1, 2]]
    d = atom_system(3.0, aos, C, 3, 2, det_up=det_up, det_dn=det_dn, ci=[0.9, 0.2, -0.3, 0.15],
                    norm=rng.uniform(0.5, 2, len(aos)), a_par=0.25, a_anti=0.5, b=0.8, xyz=(0.1, -0.2, 0.3))
    r = soa(rng.standard_normal((200, 5, 3)) * 1.5)
    check_local_energy(env, d, r, threads=2)


def test_three_atoms_many_shell_kinds(env):
    rng = np.random.default_rng(4)
    from paper_2506_09743_b200.workloads import SystemDesc, expand_shells
    xyz = np.array([[0, 0, 0], [1.8, 0.2, 0], [-0.5, 1.6, 0.4]], float)
    shells = [["1s", "2s", "2p", "3d"], ["1s", "2p"], ["1s", "1s", "2s"]]
    ao = expand_shells(shells, rng.uniform(0.6, 3.0, 9))
    n_ao = len(ao[0])
    Cm = np.linalg.qr(rng.standard_normal((n_ao, n_ao)))[0][:, :7]
    up, dn = wl.select_determinants(rng, 4, [4, 5, 6], 12)
    d = SystemDesc("tri", xyz, np.array([6.0, 1.0, 1.0]), 4, 4, *ao, None, Cm, up, dn,
                   np.concatenate([[0.9], rng.normal(0, 0.1, 11)]))
    r = wl.make_walkers(rng, xyz, 8, 333)
    check_local_energy(env, d, r, threads=4)


def test_centre_without_basis_functions_and_many_shells(env):
    # a bare point charge (no AOs on it) still enters V_en and V_nn; 40 s shells on the other centre cross
    # several 16-row AO chunks
    rng = np.random.default_rng(9)
    from paper_2506_09743_b200.workloads import SystemDesc
    xyz = np.array([[0.0, 0.0, 0.0], [0.0, 1.1, 1.7]])
    n = 40
    zeta = rng.uniform(0.4, 3.0, n)
    z = np.zeros(n, np.int32)
    Cm = np.linalg.qr(rng.standard_normal((n, n)))[0][:, :4]
    d = SystemDesc("bare", xyz, np.array([3.0, 2.0]), 2, 1, z, np.ones(n, np.int32), z, z, zeta, None, Cm,
                   np.array([[0, 1], [0, 2], [3, 1]], np.int32), np.array([[0], [0], [1]], np.int32),
                   np.array([0.9, 0.2, -0.1]))
    r = wl.make_walkers(rng, xyz, 3, 129)
    el0, el = check_local_energy(env, d, r, threads=2)
    torch, ob, qb = env
    parts = ob.local_energy(ob.OracleSystem(d), r, parts=True)[3]
    assert abs(parts[0, 3] - 3.0 * 2.0 / np.linalg.norm(xyz[1])) < 1e-13  # V_nn counts the bare charge


# ----------------------------------------------------------------------------- Metropolis
def check_metropolis(env, d, r, step, n_sweeps, seed, threads=8, eloc_acc=False):
    torch, ob, qb = env
    o = ob.OracleSystem(d)
    ref = ob.metropolis(o, r, step, n_sweeps, seed, threads=threads, want_eloc_acc=eloc_acc)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    out = s.metropolis(rg, step, n_sweeps, seed, want_accept=True, want_eloc_acc=eloc_acc, count=True)
    torch.cuda.synchronize()
    acc = out["accept"].cpu().numpy()
    M = r.shape[2]
    alive = np.ones(M, bool)   # walkers whose trajectory has not legitimately forked
    excused = 0
    for sw in range(n_sweeps):
        diff = (acc[sw] != ref["accept"][sw]) & alive
        if diff.any():
            inside = np.abs(ref["margin"][sw]) < 1e-12
            assert np.all(inside[diff]), f"sweep {sw}: {int((diff & ~inside).sum())} decisions differ outside the tie window"
            excused += int(diff.sum())
            alive &= ~diff
    assert excused <= 1
    assert out["n_accepted"] == int(acc.sum())
    rf = rg.cpu().numpy()
    assert np.max(np.abs(rf[:, :, alive] - ref["r"][:, :, alive])) < 1e-12
    assert np.max(np.abs(out["logpsi"].cpu().numpy()[alive] - ref["logpsi"][alive])) < 1e-10
    assert np.array_equal(out["sign"].cpu().numpy()[alive], ref["sign"][alive])
    if eloc_acc:
        # per-walker sweep-summed E_L, element-wise at the contract's 1e-8 max(1, |.|); a walker that passed near a node
        # during the sweeps is adjudicated by the long-double run of the same oracle (reading Q24) and counted
        refx = ob.metropolis(ob.OracleSystem(d, extended=True), r, step, n_sweeps, seed, threads=threads, want_eloc_acc=True)
        same = alive & (refx["accept"] == ref["accept"]).all(axis=0)
        ea, ea0, eax = out["eloc_acc"].cpu().numpy(), ref["eloc_acc"], refx["eloc_acc"]
        n_exc = adjudicate(ea, ea0, eax, 1e-8, scale=np.maximum(1.0, np.abs(eax)), mask=same, what="sum of E_L over the sweeps")
        assert same.sum() >= 0.99 * M and n_exc <= max(2, M // 50), (int(same.sum()), n_exc)
    rate = acc.mean()
    assert 0.02 < rate < 0.99
    s.close()
    return rate


@pytest.mark.parametrize("name,M,step,sweeps", [("H2", 1024, 0.5, 10), ("LiH", 700, 0.3, 10), ("Li2", 301, 0.3, 10),
                                                ("CO", 259, 0.2, 20)])
def test_metropolis_configs(env, name, M, step, sweeps):
    d, r = wl.CONFIGS[name](M=M)
    check_metropolis(env, d, r, step, sweeps, seed=2024)


def test_metropolis_eloc_every_sweep(env):
    d, r = wl.co_scan(M=64, n_geom=2)[1]
    check_metropolis(env, d, r, 0.2, 5, seed=7, threads=8, eloc_acc=True)


def test_metropolis_resume_and_offsets(env):
    torch, ob, qb = env
    d, r = wl.li2(M=200)
    s = qb.QmcSystem(d)
    a = _to_gpu(torch, r)
    oa = s.metropolis(a, 0.3, 6, seed=99, want_accept=True)
    b = _to_gpu(torch, r)
    s.metropolis(b, 0.3, 2, seed=99)
    ob2 = s.metropolis(b, 0.3, 4, seed=99, sweep_offset=2, want_accept=True)
    assert torch.equal(a, b) and torch.equal(oa["accept"][2:], ob2["accept"])
    # shard: walkers 120.. evaluated alone with walker_offset reproduce the same trajectories
    c = _to_gpu(torch, r[:, :, 120:])
    s.metropolis(c, 0.3, 6, seed=99, walker_offset=120)
    assert torch.equal(c, a[:, :, 120:])
    s.close()


def test_batch_stats(env):
    torch, ob, qb = env
    x = np.random.default_rng(1).standard_normal(100003) * 3 - 40.0
    m0, s0 = ob.batch_stats(x)
    m, s = qb.batch_stats(torch.from_numpy(x).cuda())
    assert abs(m - m0) < 1e-12 * abs(m0) and abs(s - s0) < 1e-10 * s0


def test_error_codes(env):
    torch, ob, qb = env
    import copy
    d, r = wl.lih(M=4)
    bad = copy.copy(d); bad.ao_l = d.ao_l.copy(); bad.ao_l[0] = 1  # l >= n for a 1s
    with pytest.raises(qb.QmcError) as ei:
        qb.QmcSystem(bad)
    assert ei.value.status == qb.QMC_EINVAL
    bad = copy.copy(d); bad.det_up = np.array([[0, 0]], np.int32)
    with pytest.raises(qb.QmcError) as ei:
        qb.QmcSystem(bad)
    assert ei.value.status == qb.QMC_EINVAL
    big = atom_system(10.0, [(1, 0, 0, 1.0 + 0.1 * i) for i in range(12)], np.eye(12)[:, :9], 9, 0)
    with pytest.raises(qb.QmcError) as ei:
        qb.QmcSystem(big)
    assert ei.value.status == qb.QMC_EUNSUPPORTED
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    with pytest.raises(qb.QmcError):
        s.metropolis(rg, -1.0, 2, seed=1)
    s.close()


def test_fp64_peak_and_model_flops(env):
    torch, ob, qb = env
    t = qb.fp64_peak(0, reps=2)
    assert 5.0 < t < 80.0
    d, _ = wl.co(M=2)
    s = qb.QmcSystem(d)
    assert 5.5e4 < s.model_flops(0) < 6.5e4 and 2.5e4 < s.model_flops(1) < 4e4
    s.close()


# ----------------------------------------------------------------------------- full BASELINE sizes
@pytest.mark.parametrize("name", ["H2", "LiH", "Li2"])
def test_full_size_small_configs(env, name):
    """BASELINE configs[0..2] at their stated walker counts, every walker compared."""
    d, r = wl.CONFIGS[name]()
    check_local_energy(env, d, r, threads=os.cpu_count() or 8)


def test_full_size_co_every_walker(env):
    """BASELINE configs[3] at its stated size, in the launch configuration bench.py times: ALL 131072 walkers against
    the oracle -- sign exact, log|Psi| 1e-10, E_L 1e-8 max(1, |E_L|) on walkers with |Psi|/max|Psi| > 1e-6, batch mean
    1e-10.  Walkers on which the float64 oracle is itself more than a tenth of the bound away from the long-double run
    of the same source are adjudicated by that run (tests.helpers.adjudicate, reading Q24) and counted."""
    torch, ob, qb = env
    d, r = wl.co()
    M = r.shape[2]
    nt = os.cpu_count() or 8
    s = qb.QmcSystem(d)
    lp, sg, el = (t.cpu().numpy() for t in s.local_energy(_to_gpu(torch, r)))
    lp2, sg2 = (t.cpu().numpy() for t in s.log_psi(_to_gpu(torch, r)))
    lp0, sg0, el0 = ob.local_energy(ob.OracleSystem(d), r, threads=nt)
    lpx, sgx, elx = ob.local_energy(ob.OracleSystem(d, extended=True), r, threads=nt)
    assert np.array_equal(sg0, sgx)
    assert np.array_equal(sg, sg0) and np.array_equal(sg2, sg0), int((sg != sg0).sum())
    n_lp = adjudicate(lp, lp0, lpx, 1e-10, what="log|Psi| (E_L kernel)")
    n_lp2 = adjudicate(lp2, lp0, lpx, 1e-10, what="log|Psi| (values-only kernel)")
    keep = lp0 - lp0.max() > math.log(1e-6)
    n_el = adjudicate(el, el0, elx, 1e-8, scale=np.maximum(1.0, np.abs(elx)), mask=keep, what="E_L")
    # measured on this batch: 26 walkers of 131072 for log|Psi| (near-singular Slater matrices or a cancelling CI sum,
    # the float64 oracle itself up to 6.8e-10 from the long-double value), none for E_L
    assert n_lp <= 64 and n_lp2 <= 64 and n_el <= 4, (n_lp, n_lp2, n_el)
    # batch mean, 1e-10 relative (reading Q15): over the walkers of the per-walker criterion, and over ALL walkers.  The
    # latter is dominated by a handful of walkers next to a node of Psi (|E_L| up to 4.5e6 on this batch), where one part
    # in 1e9 of a single E_L is the whole bound: the float64 oracle's own all-walker mean is 2.7e-10 from its long-double
    # build's.  Same adjudication as per walker (Q24): literal against the float64 oracle where that is pinned to a tenth
    # of the bound by the long-double mean, else as good as the float64 oracle against the long-double mean.
    for sel, what in ((keep, "criterion set"), (np.ones(M, bool), "all walkers")):
        m0, m1, mx = (ob.batch_stats(a[sel])[0] for a in (el0, el, elx))
        if abs(m0 - mx) <= 1e-11 * abs(mx):
            assert abs(m1 - m0) <= 1e-10 * abs(m0), (what, m0, m1)
        else:
            assert abs(m1 - mx) <= max(1e-10 * abs(mx), 4 * abs(m0 - mx)), (what, m0, m1, mx)
    m, e = qb.batch_stats(torch.from_numpy(el).cuda())
    mo, eo = ob.batch_stats(el)
    assert abs(m - mo) < 1e-12 * abs(mo) and abs(e - eo) < 1e-10 * eo
    # Metropolis at full size: contiguous sample ranges, global walker indices
    rg = _to_gpu(torch, r)
    out = s.metropolis(rg, 0.2, 5, seed=4242, want_accept=True)
    acc = out["accept"].cpu().numpy()
    rf = rg.cpu().numpy()
    o = ob.OracleSystem(d)
    for w0 in (0, 40001, M - 96):
        w1 = w0 + 96
        rr = np.array(r, order="C", copy=True)
        a0 = np.zeros((5, M), np.uint8); mg = np.zeros((5, M)); l0 = np.zeros(M); s0 = np.zeros(M)
        assert o.L.oracle_metropolis(o.ref, rr.ctypes.data, M, w0, w1, 0.2, 5, 4242, 0, l0.ctypes.data, s0.ctypes.data,
                                     a0.ctypes.data, mg.ctypes.data, None) == 0
        bad = (acc[:, w0:w1] != a0[:, w0:w1]) & (np.abs(mg[:, w0:w1]) >= 1e-12)
        assert not bad.any()
        same = (acc[:, w0:w1] == a0[:, w0:w1]).all(axis=0)
        assert np.max(np.abs(rf[:, :, w0:w1][:, :, same] - rr[:, :, w0:w1][:, :, same])) < 1e-12
    s.close()


def test_full_size_co_scan_geometry(env):
    """BASELINE configs[4] at its stated size for one geometry: 262144 walkers, 500 determinants, 50 sweeps with E_L
    after every sweep.  The oracle follows the first 1024 walkers (Philox is keyed by the global walker index, so a
    prefix reproduces exactly those trajectories): accept masks bit-exact outside the tie window, final positions,
    per-walker sweep-averaged E_L element-wise at 1e-8 max(1, |.|) with adjudication (walkers that pass near a node
    are counted, not hidden), and the reported quantity of reading Q16: mean and standard error over walkers."""
    torch, ob, qb = env
    d, r = wl.co_scan(M=262144, n_geom=6)[5]      # R = 2.40 bohr
    M, P, n_sweeps, step, seed = r.shape[2], 1024, 50, 0.2, 777
    nt = os.cpu_count() or 8
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    out = s.metropolis(rg, step, n_sweeps, seed, want_accept=True, want_eloc_acc=True, count=True)
    torch.cuda.synchronize()
    acc = out["accept"].cpu().numpy()
    assert out["n_accepted"] == int(acc.sum())
    ea = out["eloc_acc"].cpu().numpy()
    assert np.isfinite(ea).all()
    rp = np.ascontiguousarray(r[:, :, :P])
    ref = ob.metropolis(ob.OracleSystem(d), rp, step, n_sweeps, seed, threads=nt, want_eloc_acc=True)
    refx = ob.metropolis(ob.OracleSystem(d, extended=True), rp, step, n_sweeps, seed, threads=nt, want_eloc_acc=True)
    alive = np.ones(P, bool)
    excused = 0
    for sw in range(n_sweeps):
        diff = (acc[sw, :P] != ref["accept"][sw]) & alive
        if diff.any():
            assert np.all(np.abs(ref["margin"][sw])[diff] < 1e-12), f"sweep {sw}: decisions differ outside the tie window"
            excused += int(diff.sum())
            alive &= ~diff
    assert excused <= 1
    rf = rg[:, :, :P].cpu().numpy()
    assert np.max(np.abs(rf[:, :, alive] - ref["r"][:, :, alive])) < 1e-12
    lp = out["logpsi"].cpu().numpy()[:P]
    same = alive & (refx["accept"] == ref["accept"]).all(axis=0)
    adjudicate(lp, ref["logpsi"], refx["logpsi"], 1e-10, mask=same, what="final log|Psi|")
    assert np.array_equal(out["sign"].cpu().numpy()[:P][alive], ref["sign"][alive])
    eb, eb0, ebx = ea[:P] / n_sweeps, ref["eloc_acc"] / n_sweeps, refx["eloc_acc"] / n_sweeps
    n_exc = adjudicate(eb, eb0, ebx, 1e-8, scale=np.maximum(1.0, np.abs(ebx)), mask=same, what="sweep-averaged E_L per walker")
    assert same.sum() >= P - 8 and n_exc <= P // 50, (int(same.sum()), n_exc)
    # reading Q16: mean and standard error over walkers of the per-walker sweep averages -- on the prefix against the
    # oracle (device reduction on the GPU's own values), and the full-size device reduction against the oracle's
    # reduction of the same array
    sel = torch.from_numpy(np.flatnonzero(same)).cuda()
    mg_, eg_ = qb.batch_stats((out["eloc_acc"][:P] / n_sweeps)[sel].contiguous())
    m0, e0 = ob.batch_stats(eb0[same])
    assert abs(mg_ - m0) <= 1e-10 * abs(m0) and abs(eg_ - e0) <= 1e-8 * e0, (mg_, m0, eg_, e0)
    mf, ef = qb.batch_stats((out["eloc_acc"] / n_sweeps).contiguous())
    mo, eo = ob.batch_stats(ea / n_sweeps)
    assert abs(mf - mo) <= 1e-12 * abs(mo) and abs(ef - eo) <= 1e-10 * eo
    rate = acc.mean()
    assert 0.05 < rate < 0.95
    s.close()


def test_full_size_co_derivatives_sampled(env):
    """The NEXT-1 calls in the sizes bench.py times them at: O_p on 131072 CO walkers, the orbital-parameter derivatives
    on the first 32768; the oracle evaluates a sample of walkers, and the eq. 6 reduction is checked on the full arrays
    by properties (sum rule per walker, Euler's identity for the MO coefficients)."""
    torch, ob, qb = env
    d, r = wl.co()
    M = r.shape[2]
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    lp, sg, el, O = s.log_derivatives(rg)
    idx = np.unique(np.concatenate([np.arange(0, 32), np.arange(M - 33, M), np.random.default_rng(1).integers(0, M, 512)]))
    o = ob.OracleSystem(d)
    rs = np.ascontiguousarray(r[:, :, idx])
    lp0 = ob.local_energy(o, rs, threads=os.cpu_count() or 8)[0]
    O0 = ob.log_derivatives(o, rs, threads=os.cpu_count() or 8)
    keep = lp0 - float(lp.max()) > math.log(1e-6)
    On = O[torch.from_numpy(idx).cuda()].cpu().numpy()
    assert np.max((np.abs(On - O0) / np.maximum(1.0, np.abs(O0)))[keep]) < 1e-8
    ci = torch.from_numpy(np.asarray(d.ci_coeff)).cuda()
    lpn = lp.cpu().numpy()
    good = torch.from_numpy(lpn - lpn.max() > math.log(1e-6)).cuda()
    assert float(((O[:, 6:] @ ci - 1.0).abs() * good).max()) < 1e-8           # Sigma is linear in the CI coefficients
    ev, g = qb.energy_gradient(el, O)
    assert np.isfinite(g).all() and abs(ev - float(el.mean())) < 1e-9 * abs(ev)
    # orbital parameters
    Mo = 32768
    ro = rg[:, :, :Mo].contiguous()
    dC, dz = s.orbital_derivatives(ro, d.n_ao, d.n_mo)
    io = idx[idx < Mo]
    ko = keep[idx < Mo]
    dC0, dz0 = ob.orbital_derivatives(o, np.ascontiguousarray(r[:, :, io]), threads=os.cpu_count() or 8)
    sel = torch.from_numpy(io).cuda()
    eC = np.abs(dC[sel].cpu().numpy() - dC0) / np.maximum(1.0, np.abs(dC0))
    ez = np.abs(dz[sel].cpu().numpy() - dz0) / np.maximum(1.0, np.abs(dz0))
    assert np.max(eC[ko]) < 1e-8 and np.max(ez[ko]) < 1e-8
    # Euler: Psi is homogeneous of degree N_e in the MO coefficients -> sum C dlnPsi/dC = N_e for every walker
    Cm = torch.from_numpy(np.asarray(d.mo_coeff, np.float64)).cuda()
    euler = (dC * Cm[None]).sum(dim=(1, 2))
    assert float(((euler - d.n_e).abs() * good[:Mo]).max()) < 1e-7
    s.close()


def test_co_scan_geometries_sampled(env):
    """BASELINE configs[4] shape: 500 determinants, several bond lengths, E_L accumulated every sweep."""
    torch, ob, qb = env
    for k, (d, r) in enumerate(wl.co_scan(M=96, n_geom=16)):
        if k not in (0, 7, 15):
            continue
        check_local_energy(env, d, r, threads=os.cpu_count() or 8, mean_rtol=1e-9)


def test_triple_and_quadruple_substitutions(env):
    """Determinants with more than two substitutions in a spin (general k x k path)."""
    rng = np.random.default_rng(11)
    d, r = wl.li2(M=130)
    import copy
    d = copy.copy(d)
    # reference (0,1,2); virtuals 3..7
    d.det_up = np.array([[0, 1, 2], [3, 4, 5], [0, 6, 2], [7, 3, 6], [3, 1, 4], [5, 7, 4]], np.int32)
    d.det_dn = np.array([[0, 1, 2], [0, 1, 2], [4, 5, 6], [0, 1, 7], [5, 3, 6], [7, 6, 3]], np.int32)
    d.ci_coeff = np.array([0.9, 0.2, -0.15, 0.1, 0.25, -0.12])
    check_local_energy(env, d, r, threads=4)
    check_metropolis(env, d, r, 0.3, 4, seed=3)
    # CO-sized: quadruple in one spin, triple in the other
    d, r = wl.co(M=66)
    d = copy.copy(d)
    up = d.det_up.copy(); dn = d.det_dn.copy()
    up[5] = [7, 8, 9, 10, 4, 5, 6]; dn[5] = [0, 11, 2, 12, 4, 13, 6]
    up[9] = [0, 1, 2, 13, 12, 11, 6]
    d.det_up, d.det_dn = up, dn
    check_local_energy(env, d, r, threads=8)


# ----------------------------------------------------------------------------- parameter derivatives (eq. 6)
def check_log_derivatives(env, d, r, threads=8):
    """O_p = (dPsi/dtheta_p)/Psi and the gradient estimator of eq. 6 against the oracle.
    Tolerance: 1e-8 * max(1, |O|) per element for walkers with |Psi|/max|Psi| > 1e-6,
    E_L as in check_local_energy, gradient 1e-8 of its absolute-sum scale."""
    torch, ob, qb = env
    o = ob.OracleSystem(d)
    lp0, sg0, el0 = ob.local_energy(o, r, threads=threads)
    O0 = ob.log_derivatives(o, r, threads=threads)
    s = qb.QmcSystem(d)
    assert s.n_param() == O0.shape[1]
    rg = _to_gpu(torch, r)
    lp, sg, el, O = s.log_derivatives(rg)
    el_plain = s.local_energy(rg)[2]
    torch.cuda.synchronize()
    assert torch.equal(el, el_plain), "E_L of the derivative kernel differs from qmc_local_energy"
    ev, g = qb.energy_gradient(el, O)
    # the fused call (qmc_local_energy_gradient): same E_L bit for bit, the estimator without O in HBM, bit-repeatable
    lpf, sgf, elf, evf, gf = s.local_energy_gradient(rg)
    assert torch.equal(elf, el) and torch.equal(lpf, lp) and torch.equal(sgf, sg)
    evf2, gf2 = s.local_energy_gradient(rg)[3:]
    assert evf2 == evf and np.array_equal(gf2, gf)
    lpn, sgn, eln, On = (t.cpu().numpy() for t in (lp, sg, el, O))
    s.close()
    assert np.array_equal(sgn, sg0) and np.max(np.abs(lpn - lp0)) < 1e-10
    keep = lp0 - lp0.max() > math.log(1e-6)
    err = np.abs(On - O0) / np.maximum(1.0, np.abs(O0))
    assert np.max(err[keep]) < 1e-8, (np.max(err[keep]), np.unravel_index(np.argmax(err * keep[:, None]), err.shape))
    # sum rule on the GPU result itself
    assert np.max(np.abs(On[keep, On.shape[1] - len(d.ci_coeff):] @ np.asarray(d.ci_coeff) - 1.0)) < 1e-9
    # estimator: the oracle's reduction applied to the oracle's E_L and O
    ev0, g0 = ob.energy_gradient(el0, O0)
    scale = 2.0 * np.mean(np.abs(O0) * np.abs(el0 - ev0)[:, None], axis=0)
    assert abs(ev - ev0) <= 1e-10 * abs(ev0)
    assert np.max(np.abs(g - g0) / np.maximum(scale, 1e-300)) < 1e-8, np.max(np.abs(g - g0) / np.maximum(scale, 1e-300))
    assert abs(evf - ev0) <= 1e-10 * abs(ev0)
    assert np.max(np.abs(gf - g0) / np.maximum(scale, 1e-300)) < 1e-8, np.max(np.abs(gf - g0) / np.maximum(scale, 1e-300))
    # and the GPU reduction applied to identical inputs agrees with the oracle's to rounding
    ev1, g1 = qb.energy_gradient(torch.from_numpy(el0).cuda(), torch.from_numpy(O0).cuda())
    assert abs(ev1 - ev0) <= 1e-13 * abs(ev0) and np.max(np.abs(g1 - g0) / np.maximum(scale, 1e-300)) < 1e-12


@pytest.mark.parametrize("name,M", [("H2", 1024), ("LiH", 700), ("Li2", 1027), ("CO", 1025)])
def test_log_derivatives_configs(env, name, M):
    d, r = wl.CONFIGS[name](M=M)
    check_log_derivatives(env, d, r)


def test_log_derivatives_co_500_determinants_and_ragged(env):
    d, r = wl.co_scan(M=301, n_geom=2)[1]
    check_log_derivatives(env, d, r)
    d, r = wl.co(M=3)
    check_log_derivatives(env, d, r, threads=1)


def test_log_derivatives_general_substitutions_and_unequal_spins(env):
    rng = np.random.default_rng(11)
    aos = [(1, 0, 0, 2.0), (2, 0, 0, 1.5), (2, 1, 0, 1.3), (2, 1, 1, 1.3), (2, 1, 2, 1.3), (3, 2, 3, 0.9), (3, 0, 0, 1.2),
           (1, 0, 0, 0.8)]
    C = rng.standard_normal((len(aos), 8))
    # reference, a repeated reference, singles, a same-spin double, a triple (general path) and mixed ones
    det_up = [[0, 1, 2, 3], [0, 1, 2, 3], [0, 4, 2, 3], [5, 1, 6, 3], [4, 5, 6, 3], [0, 1, 2, 7], [4, 1, 5, 3]]
    det_dn = [[0, 1], [0, 1], [0, 1], [0, 1], [2, 1], [0, 3], [4, 5]]
    d = atom_system(4.0, aos, C, 4, 2, det_up=det_up, det_dn=det_dn, ci=[0.8, 0.1, -0.3, 0.15, 0.05, 0.2, -0.1],
                    a_par=0.25, a_anti=0.5, b=0.8, xyz=(0.1, -0.2, 0.3))
    r = soa(rng.standard_normal((257, 6, 3)) * 1.3)
    check_log_derivatives(env, d, r, threads=2)


# ----------------------------------------------------------------------------- electron-nucleus Jastrow (D.2)
def _with_en(d, w0, w1, w2):
    import copy
    d2 = copy.copy(d)
    d2.jastrow_en_w0, d2.jastrow_en_w1, d2.jastrow_en_w2 = w0, w1, w2
    return d2


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 700), ("Li2", 1027), ("CO", 1025)])
def test_en_jastrow_local_energy_and_metropolis(env, name, M):
    d, r = wl.CONFIGS[name](M=M)
    d = _with_en(d, 0.35, -0.04, 0.9)
    el0, el = check_local_energy(env, d, r)
    # the term is really there: E_L differs from the e-e-only wavefunction's
    torch, ob, qb = env
    el_plain = ob.local_energy(ob.OracleSystem(_with_en(d, 0.0, 0.0, 0.9)), r[:, :, :8])[2]
    assert np.max(np.abs(el_plain - el0[:8])) > 1e-3
    check_metropolis(env, d, r[:, :, :257], 0.25, 6, seed=11)
    check_log_derivatives(env, d, r[:, :, :129])


def test_en_jastrow_three_atoms_unequal_spins(env):
    rng = np.random.default_rng(21)
    from paper_2506_09743_b200.workloads import SystemDesc, expand_shells
    xyz = np.array([[0, 0, 0], [1.8, 0.2, 0], [-0.5, 1.6, 0.4]], float)
    ao = expand_shells([["1s", "2s", "2p"], ["1s", "2p"], ["1s", "1s"]], rng.uniform(0.6, 3.0, 7))
    n_ao = len(ao[0])
    Cm = np.linalg.qr(rng.standard_normal((n_ao, n_ao)))[0][:, :6]
    d = SystemDesc("tri-en", xyz, np.array([4.0, 1.0, 1.0]), 3, 2, *ao, None, Cm,
                   np.array([[0, 1, 2], [0, 3, 2], [4, 1, 5]], np.int32), np.array([[0, 1], [0, 1], [2, 1]], np.int32),
                   np.array([0.9, 0.2, -0.15]), 0.25, 0.5, 0.8, -0.3, 0.06, 1.1)
    r = wl.make_walkers(rng, xyz, 5, 333)
    check_local_energy(env, d, r, threads=4)
    check_metropolis(env, d, r[:, :, :200], 0.3, 5, seed=3)


# ----------------------------------------------------------------------------- host-buffer entry point
@pytest.mark.parametrize("M,chunks,pinned", [(1027, 4, True), (1027, 1, True), (33, 8, True), (515, 3, False)])
def test_local_energy_host_matches_device_call(env, M, chunks, pinned):
    torch, ob, qb = env
    d, r = wl.co(M=M)
    s = qb.QmcSystem(d)
    ref = torch.stack(s.local_energy(_to_gpu(torch, r))).cpu()
    rh = torch.from_numpy(np.ascontiguousarray(r))
    out = torch.empty((3, M), dtype=torch.float64)
    if pinned:
        rh, out = rh.pin_memory(), out.pin_memory()
    got = s.local_energy_host(rh, out, n_chunks=chunks)
    assert torch.equal(got, ref)  # walkers are independent: chunking changes nothing, bit for bit
    got2 = s.local_energy_host(rh, None, n_chunks=2)  # reuses / regrows the handle's scratch
    assert torch.equal(got2, ref)
    s.close()


# ----------------------------------------------------------------------------- CUDA graphs
def _with_bf_early(d, w):
    import copy
    d2 = copy.copy(d)
    d2.backflow_w = w
    return d2


@pytest.mark.parametrize("name,bf", [("H2", False), ("Li2", False), ("Li2", True), ("CO", True)])
def test_calls_can_be_captured_in_a_cuda_graph(env, name, bf):
    # after one warm-up call (which sizes the handle's per-stream fallback scratch) qmc_metropolis and
    # qmc_local_energy contain nothing that breaks stream capture; a replay reproduces the eager run bit for bit
    # (bf: the backflow kernels, table route + listed walkers on the explicit kernel)
    torch, ob, qb = env
    d, r = wl.CONFIGS[name](M=777)
    if bf:
        d = _with_bf_early(d, 0.07)
    s = qb.QmcSystem(d)
    r0 = _to_gpu(torch, r)
    rg = r0.clone()
    M = r.shape[2]
    lp = torch.empty(M, dtype=torch.float64, device="cuda")
    sg, el, acc = torch.empty_like(lp), torch.empty_like(lp), torch.zeros_like(lp)
    st = torch.cuda.Stream()

    def body(k):
        s.metropolis(rg, 0.3, 1, seed=7, sweep_offset=k, logpsi=lp, sign=sg, stream=st)
        s.local_energy(rg, lp, sg, el, stream=st)
        acc.add_(el)

    with torch.cuda.stream(st):
        for k in range(4):
            body(k)
        ref_acc, ref_r = acc.clone(), rg.clone()
        rg.copy_(r0)
        acc.zero_()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            for k in range(4):
                body(k)
        rg.copy_(r0)
        acc.zero_()
        g.replay()
        torch.cuda.synchronize()
    assert torch.equal(acc, ref_acc) and torch.equal(rg, ref_r)
    s.close()


# ----------------------------------------------------------------------------- electron-electron-nucleus Jastrow (D.3)
EEN = np.array([[0.30, 0.8, 0.9, 0.5, 1.4, 0.7, 0.6],
                [-0.12, 1.1, 0.4, 0.9, 0.8, 0.35, 1.2],
                [0.05, 0.6, 1.7, 1.3, 0.5, 1.0, 0.9],
                [0.02, 1.0, 1.0, 1.0, 1.0, 0.5, 2.0],
                [-0.04, 0.4, 0.3, 0.7, 2.2, 1.5, 0.4]])


def _with_een(d, een=EEN):
    import copy
    d2 = copy.copy(d)
    d2.jastrow_een = np.asarray(een, np.float64)
    return d2


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 700), ("Li2", 517), ("CO", 513)])
def test_een_jastrow_local_energy_and_metropolis(env, name, M):
    d, r = wl.CONFIGS[name](M=M)
    d = _with_een(_with_en(d, 0.2, -0.03, 0.8))  # the many-body Jastrow of PAPER.md:245-253: e-e + e-n + e-e-n (5 terms)
    el0, el = check_local_energy(env, d, r)
    torch, ob, qb = env
    el_plain = ob.local_energy(ob.OracleSystem(_with_een(d, np.zeros((0, 7)))), r[:, :, :8])[2]
    assert np.max(np.abs(el_plain - el0[:8])) > 1e-3
    check_metropolis(env, d, r[:, :, :257], 0.25, 6, seed=13)


def test_een_jastrow_three_atoms_unequal_spins_and_limits(env):
    torch, ob, qb = env
    rng = np.random.default_rng(23)
    from paper_2506_09743_b200.workloads import SystemDesc, expand_shells
    xyz = np.array([[0, 0, 0], [1.8, 0.2, 0], [-0.5, 1.6, 0.4]], float)
    ao = expand_shells([["1s", "2s", "2p"], ["1s", "2p"], ["1s", "1s"]], rng.uniform(0.6, 3.0, 7))
    n_ao = len(ao[0])
    Cm = np.linalg.qr(rng.standard_normal((n_ao, n_ao)))[0][:, :6]
    d = SystemDesc("tri-een", xyz, np.array([4.0, 1.0, 1.0]), 3, 2, *ao, None, Cm,
                   np.array([[0, 1, 2], [0, 3, 2], [4, 1, 5]], np.int32), np.array([[0, 1], [0, 1], [2, 1]], np.int32),
                   np.array([0.9, 0.2, -0.15]), 0.25, 0.5, 0.8, -0.3, 0.06, 1.1, EEN[:2])
    r = wl.make_walkers(rng, xyz, 5, 333)
    check_local_energy(env, d, r, threads=4)
    check_metropolis(env, d, r[:, :, :200], 0.3, 5, seed=3)
    # more terms than compiled for: reported, not mis-evaluated
    import ctypes as C
    desc, keep = qb.make_desc(_with_een(d, np.tile(EEN, (2, 1))[:7]))
    h = C.c_void_p()
    assert qb.lib().qmc_setup(C.addressof(desc), 0, C.byref(h)) == qb.QMC_EUNSUPPORTED


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 300), ("Li2", 259), ("CO", 130)])
def test_log_derivatives_with_een_terms(env, name, M):
    """O_p in the seven parameters of every e-e-n term (D.3), between the D.1/D.2 block and the CI block."""
    d, r = wl.CONFIGS[name](M=M)
    d = _with_een(_with_en(d, 0.2, -0.03, 0.8))
    check_log_derivatives(env, d, r)


def test_log_derivatives_with_one_and_six_een_terms(env):
    d, r = wl.lih(M=64)
    d1 = _with_een(_with_en(d, 0.1, 0.02, 1.1), EEN[:1])
    check_log_derivatives(env, d1, r, threads=2)
    d6 = _with_een(d1, np.concatenate([EEN, 0.5 * EEN[:1]]))   # the maximum of six terms
    check_log_derivatives(env, d6, r, threads=2)


def test_vmc_example_gradient_descent_lowers_the_h2_energy(env):
    # eq. 6 end to end on the GPU path (sampler -> E_L + O_p -> estimator -> parameter step -> new handle): for the H2
    # configuration, switching on the electron-nucleus kernel by gradient descent lowers the variational energy by
    # several standard errors in the first step and the gradient norm collapses; seeded, hence reproducible
    import copy
    from paper_2506_09743_b200 import vmc_example as vx
    d, r = wl.h2(M=65536)
    d = copy.copy(d)
    d.jastrow_en_w2 = 1.0
    hist, d_opt = vx.optimise(d, r, iterations=4, lr=0.2, step=0.5, verbose=False)
    e = [h[0] for h in hist]
    err = max(h[1] for h in hist)
    assert err < 2e-3
    assert min(e[1:]) < e[0] - 4 * err, (e, err)
    assert hist[1][2] < 0.5 * hist[0][2]
    assert d_opt.jastrow_en_w1 != 0.0 and -1.20 < e[-1] < -1.10   # exact H2: -1.1745 Ha; HF-like orbital + Jastrow ~ -1.15


def test_vmc_example_optimises_the_backflow_weight(env):
    # eq. 6 for a backflow wavefunction (qmc_log_derivatives with the backflow weight as its last parameter): H2 with a
    # far too strong inverse backflow, w = 0.3 and w = -0.2; descending along the gradient takes both to the same small
    # weight and the energy down to the Jastrow-only level (seeded, hence reproducible)
    import copy
    from paper_2506_09743_b200 import vmc_example as vx
    d, r = wl.h2(M=65536)
    finals = []
    for w0 in (0.3, -0.2):
        d1 = copy.copy(d)
        d1.backflow_w = w0
        hist, d_opt = vx.optimise(d1, r, iterations=6, lr=0.2, step=0.5, verbose=False)
        e = [h[0] for h in hist]
        assert e[-1] < e[0] - 4 * max(hist[0][1], hist[-1][1]), (w0, hist)
        assert hist[-1][2] < 0.1 * hist[0][2]                      # the gradient norm collapses
        assert -1.17 < e[-1] < -1.13 and abs(d_opt.backflow_w) < 0.06, (w0, e, d_opt.backflow_w)
        finals.append(d_opt.backflow_w)
    assert abs(finals[0] - finals[1]) < 0.03, finals


def test_vmc_example_recovers_detuned_exponents_through_the_orbital_derivatives(env):
    # eq. 6 with O = d ln Psi / d zeta, d ln Psi / d C (qmc_orbital_derivatives): H2 with both AO exponents scaled by 1.35;
    # descending along the orbital gradient brings zeta back towards its value and the energy down by ten standard
    # errors relative to optimising the Jastrow parameters alone (seeded, hence reproducible)
    import copy
    from paper_2506_09743_b200 import vmc_example as vx
    d, r = wl.h2(M=65536)
    d = copy.copy(d)
    z0 = np.asarray(d.ao_zeta, np.float64)
    d.ao_zeta = 1.35 * z0
    d.jastrow_en_w2 = 1.0
    h_j, _ = vx.optimise(d, r, iterations=8, lr=0.2, step=0.5, verbose=False)
    h_o, d_o = vx.optimise(d, r, iterations=8, lr=0.2, step=0.5, verbose=False, optimise_orbitals=True, lr_orbitals=0.3)
    err = max(h[1] for h in h_j + h_o)
    assert err < 5e-3                                            # detuned exponents break the cusp: larger variance
    assert h_o[-1][0] < h_j[-1][0] - 6 * err, (h_o[-1], h_j[-1])
    assert h_o[-1][0] < h_o[1][0] - 3 * err                      # iteration 0 still carries the initial walkers
    assert np.all(d_o.ao_zeta < 1.35 * z0 - 0.15) and np.all(d_o.ao_zeta > z0)


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 300), ("Li2", 1027), ("CO", 1025)])
def test_explicit_route_for_every_walker(env, name, M):
    """qmc_local_energy_explicit (every determinant eliminated on its own, Fig. 11's "explicit") against the oracle,
    which is built the same way, and against the table path."""
    torch, ob, qb = env
    d, r = wl.CONFIGS[name](M=M)
    o = ob.OracleSystem(d)
    lp0, sg0, el0 = ob.local_energy(o, r, threads=8)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    lp, sg, el = (t.cpu().numpy() for t in s.local_energy_explicit(rg))
    lpt, sgt, elt = (t.cpu().numpy() for t in s.local_energy(rg))
    s.close()
    keep = lp0 - lp0.max() > math.log(1e-6)
    assert np.array_equal(sg, sg0) and np.max(np.abs(lp - lp0)) < 1e-10
    assert np.max((np.abs(el - el0) / np.maximum(1, np.abs(el0)))[keep]) < 1e-8
    assert np.array_equal(sg, sgt) and np.max(np.abs(lp - lpt)) < 1e-10
    assert np.max((np.abs(el - elt) / np.maximum(1, np.abs(el0)))[keep]) < 1e-8


def test_kernel_timing_events(env):
    """qmc_set_kernel_timing / qmc_kernel_times (bench.py's roofline): the two kernel durations of an E_L call are
    positive, add up to no more than the events around the call, and the outputs do not change."""
    torch, ob, qb = env
    d, r = wl.co(M=8192)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    ref = [t.clone() for t in s.local_energy(rg)]
    with pytest.raises(qb.QmcError):
        s.kernel_times()                      # never enabled
    s.set_kernel_timing(True)
    for _ in range(2):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        out = s.local_energy(rg)
        b.record()
        torch.cuda.synchronize()
        k_main, k_fb = s.kernel_times()
        assert k_main > 0.0 and k_fb > 0.0 and k_main + k_fb <= a.elapsed_time(b) * 1.001 + 1e-3
        assert all(torch.equal(x, y) for x, y in zip(out, ref))
    s.set_kernel_timing(False)
    s.close()
    d1, r1 = wl.lih(M=256)                     # single determinant: no fallback kernel
    s = qb.QmcSystem(d1)
    s.set_kernel_timing(True)
    s.local_energy(_to_gpu(torch, r1))
    k_main, k_fb = s.kernel_times()
    assert k_main > 0.0 and k_fb == 0.0
    s.close()


def test_results_are_repeatable_bit_for_bit(env):
    # the fallback work list fills in a nondeterministic order, the results must not depend on it (slice-ordered sums)
    torch, ob, qb = env
    d, r = wl.li2(M=16384)   # initial Li2 walkers: a few dozen groups take the explicit fallback
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    ref = [t.clone() for t in s.local_energy(rg)]
    for _ in range(4):
        assert all(torch.equal(a, b) for a, b in zip(s.local_energy(rg), ref))
    r1, r2 = rg.clone(), rg.clone()
    a = s.metropolis(r1, 0.3, 3, seed=9, want_accept=True, want_eloc_acc=True)
    b = s.metropolis(r2, 0.3, 3, seed=9, want_accept=True, want_eloc_acc=True)
    assert torch.equal(r1, r2) and torch.equal(a["accept"], b["accept"]) and torch.equal(a["eloc_acc"], b["eloc_acc"])
    s.close()


def test_metropolis_zero_sweeps_only_evaluates(env):
    torch, ob, qb = env
    d, r = wl.li2(M=333)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    r0 = rg.clone()
    out = s.metropolis(rg, 0.3, 0, seed=1, want_accept=True, count=True)
    lp, sg = s.log_psi(r0)
    assert torch.equal(rg, r0) and torch.equal(out["logpsi"], lp) and torch.equal(out["sign"], sg)
    assert out["n_accepted"] == 0 and tuple(out["accept"].shape) == (0, 333)
    out = s.metropolis(rg, 0.3, 0, seed=1, want_eloc_acc=True)
    assert float(out["eloc_acc"].abs().max()) == 0.0 and torch.equal(out["logpsi"], lp)
    s.close()


# ----------------------------------------------------------------------------- orbital-parameter derivatives
def check_orbital_derivatives(env, d, r, threads=8):
    torch, ob, qb = env
    o = ob.OracleSystem(d)
    lp0 = ob.local_energy(o, r, threads=threads)[0]
    dC0, dz0 = ob.orbital_derivatives(o, r, threads=threads)
    s = qb.QmcSystem(d)
    dC, dz = (t.cpu().numpy() for t in s.orbital_derivatives(_to_gpu(torch, r), d.n_ao, d.n_mo))
    s.close()
    keep = lp0 - lp0.max() > math.log(1e-6)
    eC = np.abs(dC - dC0) / np.maximum(1.0, np.abs(dC0))
    ez = np.abs(dz - dz0) / np.maximum(1.0, np.abs(dz0))
    assert np.max(eC[keep]) < 1e-8, np.max(eC[keep])
    assert np.max(ez[keep]) < 1e-8, np.max(ez[keep])


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 300), ("Li2", 257), ("CO", 129)])
def test_orbital_derivatives_configs(env, name, M):
    d, r = wl.CONFIGS[name](M=M)
    check_orbital_derivatives(env, d, r)


def test_orbital_derivatives_odd_system(env):
    rng = np.random.default_rng(31)
    aos = [(2, 1, 2, 1.1), (1, 0, 0, 2.0), (3, 2, 3, 0.9), (2, 1, 0, 1.3), (3, 2, 1, 0.7), (2, 0, 0, 1.5),
           (3, 0, 0, 1.2), (3, 1, 1, 0.8), (2, 1, 1, 1.3)]
    C = rng.standard_normal((len(aos), 7))
    det_up = [[4, 0, 2], [4, 5, 2], [1, 0, 2], [4, 3, 5]]
    det_dn = [[1, 3], [1, 3], [0, 3], [1, 2]]
    for norm in (None, rng.uniform(0.5, 2, len(aos))):
        d = atom_system(3.0, aos, C, 3, 2, det_up=det_up, det_dn=det_dn, ci=[0.9, 0.2, -0.3, 0.15], norm=norm,
                        a_par=0.25, a_anti=0.5, b=0.8, xyz=(0.1, -0.2, 0.3))
        r = soa(rng.standard_normal((131, 5, 3)) * 1.5)
        check_orbital_derivatives(env, d, r, threads=2)


def _classes_system(rng, with_general):
    """4 up / 3 down electrons in 9 random MOs with every determinant class of the table path: one substitution in
    one spin, one in each, two in one spin, two in both, and (optionally) a triple, which sends the call down the
    explicit per-determinant route."""
    aos = [(1, 0, 0, 2.4), (2, 0, 0, 1.1), (2, 1, 0, 1.3), (2, 1, 1, 1.3), (2, 1, 2, 1.3), (3, 0, 0, 0.8),
           (3, 1, 1, 0.9), (3, 2, 0, 1.0), (3, 2, 4, 1.0), (3, 2, 2, 0.7), (2, 0, 0, 2.0)]
    C = rng.standard_normal((len(aos), 9))
    det_up = [[0, 1, 2, 3], [0, 1, 2, 5], [0, 1, 2, 3], [0, 4, 2, 3], [0, 1, 6, 7], [0, 1, 2, 3], [5, 1, 6, 3],
              [4, 5, 2, 3], [0, 8, 2, 3]]
    det_dn = [[0, 1, 2], [0, 1, 2], [0, 1, 6], [0, 5, 2], [0, 1, 2], [4, 1, 8], [0, 4, 7], [3, 1, 5], [7, 1, 2]]
    ci = [0.8, 0.3, -0.25, 0.2, 0.15, -0.1, 0.12, 0.22, -0.18]
    if with_general:
        det_up.append([4, 5, 6, 3]); det_dn.append([0, 1, 3]); ci.append(0.14)
    return atom_system(4.0, aos, C, 4, 3, det_up=det_up, det_dn=det_dn, ci=ci, a_par=0.25, a_anti=0.5, b=0.9,
                       xyz=(0.2, 0.1, -0.3))


@pytest.mark.parametrize("with_general", [False, True])
def test_orbital_derivatives_every_determinant_class(env, with_general):
    rng = np.random.default_rng(77)
    d = _classes_system(rng, with_general)
    r = soa(rng.standard_normal((203, 7, 3)) * 1.2 + np.array([0.2, 0.1, -0.3]))
    check_orbital_derivatives(env, d, r, threads=4)


def test_orbital_derivatives_near_singular_reference(env):
    """Walkers on which the reference determinant all but vanishes (two same-spin electrons at almost the same
    radius in a reference of s orbitals only) while the excited determinants do not: Sigma/D_0 ~ 1e5, the group
    is flagged and takes the explicit route; the neighbouring groups stay on the tables."""
    rng = np.random.default_rng(78)
    aos = [(1, 0, 0, 2.5), (2, 0, 0, 1.0), (3, 0, 0, 0.7), (2, 1, 0, 1.2), (2, 1, 1, 1.2), (2, 1, 2, 1.2)]
    C = np.zeros((6, 6))
    C[:3, :2] = rng.standard_normal((3, 2))          # MOs 0, 1: s only
    C[:, 2:] = rng.standard_normal((6, 4))
    d = atom_system(3.0, aos, C, 2, 1, det_up=[[0, 1], [0, 2], [3, 1], [2, 4], [5, 3]], det_dn=[[0], [0], [1], [0], [2]],
                    ci=[0.7, 0.3, -0.2, 0.25, 0.1], a_par=0.25, a_anti=0.5, b=1.0)
    r = rng.standard_normal((160, 3, 3)) * 1.3
    for w in range(0, 160, 3):                        # every third walker: |r_1| = |r_0| (1 + 1e-5 u)
        u = rng.standard_normal(3)
        r[w, 1] = u / np.linalg.norm(u) * np.linalg.norm(r[w, 0]) * (1.0 + 1e-5 * rng.uniform(0.5, 1.0))
    r = soa(r)
    check_orbital_derivatives(env, d, r, threads=2)


def test_orbital_derivatives_are_repeatable_bit_for_bit(env):
    torch, ob, qb = env
    d, r = wl.co(M=1031)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    a = [t.clone() for t in s.orbital_derivatives(rg, d.n_ao, d.n_mo)]
    for _ in range(3):
        b = s.orbital_derivatives(rg, d.n_ao, d.n_mo)
        assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    s.close()


def test_orbital_derivatives_full_size_sampled_euler_identity_and_repeatability(env):
    """32768 CO walkers (the size bench.py times the call on), the seeded batch and the same walkers after 60 sweeps of this
    library's sampler (where nearly all walkers sit in the criterion set and the groups with a nearly singular reference go
    through orbital_explicit_kernel in determinant slices): a sample of the seeded batch against the oracle (dC and dzeta),
    Euler's identity sum C d ln Psi / d C = N_e on every walker of both batches, bit-repeatability at this size."""
    torch, ob, qb = env
    from tests.helpers import adjudicate
    d, r = wl.co(M=32768)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    Ct = torch.from_numpy(np.asarray(d.mo_coeff, np.float64)).cuda()
    for stage in range(2):
        if stage == 1:
            s.metropolis(rg, 0.2, 60, seed=77)
        dC, dz = s.orbital_derivatives(rg, d.n_ao, d.n_mo)
        dC2, dz2 = s.orbital_derivatives(rg, d.n_ao, d.n_mo)
        assert torch.equal(dC, dC2) and torch.equal(dz, dz2)
        lp = s.log_psi(rg)[0]
        keep = lp - lp.max() > math.log(1e-6)
        euler = (dC * Ct[None]).sum(dim=(1, 2))
        scale = (dC * Ct[None]).abs().amax(dim=(1, 2)).clamp(min=1.0)
        assert float(((euler - d.n_e).abs() / scale)[keep].max()) < 1e-8, stage
        if stage == 0:
            idx = np.random.default_rng(9).choice(np.flatnonzero(keep.cpu().numpy()), 192, replace=False)
            rs = np.ascontiguousarray(r[:, :, idx])
            o, ox = ob.OracleSystem(d), ob.OracleSystem(d, extended=True)
            dC0, dz0 = ob.orbital_derivatives(o, rs, threads=8)
            dCx, dzx = ob.orbital_derivatives(ox, rs, threads=8)
            it = torch.from_numpy(idx).cuda()
            adjudicate(dC[it].cpu().numpy(), dC0, dCx, 1e-8, scale=np.maximum(1.0, np.abs(dCx)), what="dC at full size")
            adjudicate(dz[it].cpu().numpy(), dz0, dzx, 1e-8, scale=np.maximum(1.0, np.abs(dzx)), what="dzeta at full size")
    s.close()


# ----------------------------------------------------------------------------- nuclear log-gradient (eq. 7)
def check_nuclear_log_gradient(env, d, r, threads=8):
    torch, ob, qb = env
    o = ob.OracleSystem(d)
    lp0 = ob.local_energy(o, r, threads=threads)[0]
    g0 = ob.nuclear_log_gradient(o, r, threads=threads)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    g = s.nuclear_log_gradient(rg, d.n_atoms)
    g2 = s.nuclear_log_gradient(rg, d.n_atoms)
    assert torch.equal(g, g2)                         # deterministic
    g = g.cpu().numpy()
    s.close()
    assert g.shape == g0.shape
    keep = lp0 - lp0.max() > math.log(1e-6)
    err = np.abs(g - g0) / np.maximum(1.0, np.abs(g0))
    assert np.max(err[keep]) < 1e-8, np.max(err[keep])
    return g


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 300), ("Li2", 257), ("CO", 129)])
@pytest.mark.parametrize("many_body", [False, True])
def test_nuclear_log_gradient_configs(env, name, M, many_body):
    d, r = wl.CONFIGS[name](M=M)
    if many_body:
        d = _with_een(_with_en(d, 0.3, -0.05, 0.7))
    check_nuclear_log_gradient(env, d, r)


def test_nuclear_log_gradient_odd_system_and_determinant_classes(env):
    rng = np.random.default_rng(31)
    aos = [(2, 1, 2, 1.1), (1, 0, 0, 2.0), (3, 2, 3, 0.9), (2, 1, 0, 1.3), (3, 2, 1, 0.7), (2, 0, 0, 1.5),
           (3, 0, 0, 1.2), (3, 1, 1, 0.8), (2, 1, 1, 1.3)]
    C = rng.standard_normal((len(aos), 7))
    for norm in (None, rng.uniform(0.5, 2, len(aos))):
        d = atom_system(3.0, aos, C, 3, 2, det_up=[[4, 0, 2], [4, 5, 2], [1, 0, 2], [4, 3, 5]],
                        det_dn=[[1, 3], [1, 3], [0, 3], [1, 2]], ci=[0.9, 0.2, -0.3, 0.15], norm=norm,
                        a_par=0.25, a_anti=0.5, b=0.8, xyz=(0.1, -0.2, 0.3))
        r = soa(rng.standard_normal((131, 5, 3)) * 1.5)
        check_nuclear_log_gradient(env, _with_en(d, -0.4, 0.1, 1.3), r, threads=2)
    for with_general in (False, True):
        rng = np.random.default_rng(77)
        d = _classes_system(rng, with_general)
        r = soa(rng.standard_normal((203, 7, 3)) * 1.2 + np.array([0.2, 0.1, -0.3]))
        check_nuclear_log_gradient(env, d, r, threads=4)


def test_nuclear_log_gradient_full_size_sampled_and_translation_invariance(env):
    """CO at the size bench.py times the derivative calls (32768 walkers), D.2 and D.3 on: sampled walkers against
    the oracle; on every walker sum_a grad_a ln|Psi| = -sum_i grad_i ln|Psi|, the right side by central differences
    of the GPU's own log|Psi| under a rigid shift of all electrons."""
    torch, ob, qb = env
    M = 32768
    d, r = wl.co(M=M)
    d = _with_een(_with_en(d, 0.3, -0.05, 0.7))
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    g = s.nuclear_log_gradient(rg, d.n_atoms)
    lp = s.log_psi(rg)[0]
    idx = np.unique(np.concatenate([np.arange(0, 32), np.arange(M - 33, M), np.random.default_rng(2).integers(0, M, 256)]))
    o = ob.OracleSystem(d)
    rs = np.ascontiguousarray(r[:, :, idx])
    lp0 = ob.local_energy(o, rs, threads=os.cpu_count() or 8)[0]
    g0 = ob.nuclear_log_gradient(o, rs, threads=os.cpu_count() or 8)
    keep = lp0 - float(lp.max()) > math.log(1e-6)
    gn = g[torch.from_numpy(idx).cuda()].cpu().numpy()
    assert np.max((np.abs(gn - g0) / np.maximum(1.0, np.abs(g0)))[keep]) < 1e-8
    good = lp - lp.max() > math.log(1e-6)
    h = 1e-4
    for c in range(3):
        def shifted(t):
            r2 = rg.clone()
            r2[:, c, :] += t
            return s.log_psi(r2)[0]
        cd = lambda hh: (shifted(hh) - shifted(-hh)) / (2 * hh)
        c1, c2 = cd(h), cd(2 * h)
        ref = (4 * c1 - c2) / 3
        # the differences are only trusted where the two step sizes agree (not next to a nucleus' cusp or a node)
        smooth = good & ((c1 - c2).abs() < 1e-4 * torch.clamp(ref.abs(), min=1.0))
        assert float(smooth.sum()) > 0.98 * float(good.sum())
        tot = g[:, :, c].sum(dim=1)
        rel = (tot + ref).abs() / torch.clamp(ref.abs(), min=1.0)
        assert float(rel[smooth].max()) < 1e-5, float(rel[smooth].max())
    s.close()


def test_nuclear_log_gradient_near_singular_reference(env):
    rng = np.random.default_rng(78)
    aos = [(1, 0, 0, 2.5), (2, 0, 0, 1.0), (3, 0, 0, 0.7), (2, 1, 0, 1.2), (2, 1, 1, 1.2), (2, 1, 2, 1.2)]
    C = np.zeros((6, 6))
    C[:3, :2] = rng.standard_normal((3, 2))
    C[:, 2:] = rng.standard_normal((6, 4))
    d = atom_system(3.0, aos, C, 2, 1, det_up=[[0, 1], [0, 2], [3, 1], [2, 4], [5, 3]], det_dn=[[0], [0], [1], [0], [2]],
                    ci=[0.7, 0.3, -0.2, 0.25, 0.1], a_par=0.25, a_anti=0.5, b=1.0)
    r = rng.standard_normal((160, 3, 3)) * 1.3
    for w in range(0, 160, 3):
        u = rng.standard_normal(3)
        r[w, 1] = u / np.linalg.norm(u) * np.linalg.norm(r[w, 0]) * (1.0 + 1e-5 * rng.uniform(0.5, 1.0))
    check_nuclear_log_gradient(env, d, soa(r), threads=2)


def test_nuclear_log_gradient_edge_sizes_and_a_centre_without_basis_functions(env):
    import copy
    torch, ob, qb = env
    # H2 with both AOs moved to the first nucleus: the second centre is seen by V_en and D.2 only
    d, r = wl.h2(M=33)
    d = copy.copy(d)
    d.ao_atom = np.zeros_like(np.asarray(d.ao_atom))
    g = check_nuclear_log_gradient(env, _with_en(d, 0.3, -0.05, 0.7), r, threads=1)
    assert np.abs(g[:, 1]).max() > 1e-3
    d0 = copy.copy(d)                                   # without D.2 that centre's gradient is exactly zero
    g = check_nuclear_log_gradient(env, d0, r, threads=1)
    assert np.all(g[:, 1] == 0.0)
    for name, M in (("H2", 1), ("LiH", 1), ("Li2", 3), ("CO", 1), ("CO", 2)):
        dd, rr = wl.CONFIGS[name](M=M)
        check_nuclear_log_gradient(env, dd, rr, threads=1)
    s = qb.QmcSystem(d)
    with pytest.raises(qb.QmcError):
        s.nuclear_log_gradient(torch.empty((2, 3, 0), dtype=torch.float64, device="cuda"), d.n_atoms)
    s.close()


def test_force_estimator_second_term_through_the_eq6_reduction(env):
    """Eq. 7 (DESIGN.md section 12 reading): F_alpha = -<grad_alpha E_L> - <(E_L - E_v) grad_alpha ln rho>.
    The second (Pulay) term is eq. 6's reduction with O = grad_alpha ln|Psi|: -(2/M) sum (E_L - E_v) grad_alpha ln|Psi|,
    so qmc_energy_gradient serves it; against the oracle's E_L, gradient and reduction on the same walkers."""
    torch, ob, qb = env
    d, r = wl.li2(M=2048)
    o = ob.OracleSystem(d)
    el0 = ob.local_energy(o, r, threads=os.cpu_count() or 8)[2]
    g0 = ob.nuclear_log_gradient(o, r, threads=os.cpu_count() or 8)
    ev0, f0 = ob.energy_gradient(el0, g0.reshape(len(el0), -1))
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    el = s.local_energy(rg)[2]
    g = s.nuclear_log_gradient(rg, d.n_atoms)
    ev, f = qb.energy_gradient(el, g.reshape(g.shape[0], -1))
    s.close()
    assert abs(ev - ev0) < 1e-10 * abs(ev0)
    assert np.max(np.abs(f - f0) / np.maximum(1.0, np.abs(f0))) < 1e-8
    assert np.isfinite(f).all() and np.abs(f).max() > 0


@pytest.mark.parametrize("name,M", [("H2", 70), ("LiH", 37), ("Li2", 23), ("CO", 9)])
def test_nuclear_log_gradient_writes_exactly_its_output(env, name, M):
    """Guard words around dR stay untouched and every entry inside is written (NaN-filled before the call); the
    walker coordinates are not modified.  Raw C-ABI call with a pointer into the middle of a larger buffer."""
    torch, ob, qb = env
    d, r = wl.CONFIGS[name](M=M)
    d = _with_een(_with_en(d, 0.3, -0.05, 0.7))
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    r_before = rg.clone()
    n, pad = M * d.n_atoms * 3, 4096
    buf = torch.full((n + 2 * pad,), float("nan"), dtype=torch.float64, device="cuda")
    buf[:pad] = 12345.0
    buf[pad + n:] = 12345.0
    rc = qb.lib().qmc_nuclear_log_gradient(s._h, rg.data_ptr(), M, buf.data_ptr() + 8 * pad,
                                           torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == 0
    assert bool((buf[:pad] == 12345.0).all()) and bool((buf[pad + n:] == 12345.0).all())
    assert bool(torch.isfinite(buf[pad:pad + n]).all())
    assert torch.equal(rg, r_before)
    assert torch.equal(buf[pad:pad + n].view(M, d.n_atoms, 3), s.nuclear_log_gradient(rg, d.n_atoms))
    s.close()


# ----------------------------------------------------------------------------- output bounds (no memory checker on this pool)
class _Guarded:
    """A device buffer of n elements carved from the middle of a larger allocation: guard words on both sides, the
    payload pre-filled with a sentinel (NaN for doubles, 0xAB for bytes) that a complete write must replace."""

    PAD = 2048

    def __init__(self, torch, n, dtype=None):
        self.torch, self.n = torch, n
        self.dtype = dtype or torch.float64
        if self.dtype == torch.float64:
            self.buf = torch.full((n + 2 * self.PAD,), float("nan"), dtype=self.dtype, device="cuda")
            self.guard = 12345.0
        else:
            self.buf = torch.full((n + 2 * self.PAD,), 0xAB, dtype=self.dtype, device="cuda")
            self.guard = 0x5C
        self.buf[:self.PAD] = self.guard
        self.buf[self.PAD + n:] = self.guard

    @property
    def ptr(self):
        return self.buf.data_ptr() + self.buf.element_size() * self.PAD

    @property
    def view(self):
        return self.buf[self.PAD:self.PAD + self.n]

    def check(self, what):
        assert bool((self.buf[:self.PAD] == self.guard).all()) and bool((self.buf[self.PAD + self.n:] == self.guard).all()), \
            f"{what}: guard words overwritten"
        if self.dtype == self.torch.float64:
            assert bool(self.torch.isfinite(self.view).all()), f"{what}: entries left unwritten"
        else:
            assert bool((self.view <= 1).all()), f"{what}: entries left unwritten"


@pytest.mark.parametrize("name,M", [("H2", 1), ("LiH", 37), ("Li2", 131), ("CO", 67), ("CO", 2049)])
def test_every_call_writes_exactly_its_outputs(env, name, M):
    """Raw C-ABI calls with every output pointing into the middle of a larger buffer, at ragged batch sizes (walkers
    that do not fill the last warp pass): guard words stay untouched, every entry is written, inputs are not
    modified.  Covers qmc_local_energy, qmc_log_psi, qmc_local_energy_explicit, qmc_log_derivatives,
    qmc_orbital_derivatives and qmc_metropolis (accept mask, summed E_L, in-place walkers)."""
    torch, ob, qb = env
    d, r = wl.CONFIGS[name](M=M)
    s = qb.QmcSystem(d)
    L, st = qb.lib(), torch.cuda.current_stream().cuda_stream
    rg = _to_gpu(torch, r)
    r_before = rg.clone()
    G = lambda n, dt=None: _Guarded(torch, n, dt)
    for call in ("qmc_local_energy", "qmc_local_energy_explicit"):
        a, b, c = G(M), G(M), G(M)
        assert getattr(L, call)(s._h, rg.data_ptr(), M, a.ptr, b.ptr, c.ptr, st) == 0
        torch.cuda.synchronize()
        for g, nm in ((a, "logpsi"), (b, "sign"), (c, "eloc")):
            g.check(f"{call} {nm}")
    a, b = G(M), G(M)
    assert L.qmc_log_psi(s._h, rg.data_ptr(), M, a.ptr, b.ptr, st) == 0
    torch.cuda.synchronize()
    a.check("qmc_log_psi logpsi"); b.check("qmc_log_psi sign")
    npar = s.n_param()
    a, b, c, O = G(M), G(M), G(M), G(M * npar)
    assert L.qmc_log_derivatives(s._h, rg.data_ptr(), M, a.ptr, b.ptr, c.ptr, O.ptr, st) == 0
    torch.cuda.synchronize()
    for g, nm in ((a, "logpsi"), (b, "sign"), (c, "eloc"), (O, "O")):
        g.check(f"qmc_log_derivatives {nm}")
    dC, dz = G(M * d.n_ao * d.n_mo), G(M * d.n_ao)
    assert L.qmc_orbital_derivatives(s._h, rg.data_ptr(), M, dC.ptr, dz.ptr, st) == 0
    torch.cuda.synchronize()
    dC.check("qmc_orbital_derivatives dC"); dz.check("qmc_orbital_derivatives dzeta")
    assert torch.equal(rg, r_before)
    # sampler: walkers in place inside a guarded buffer, accept mask, summed E_L
    n_sweeps = 3
    for with_acc in (False, True):
        rw = G(r.size)
        rw.view.copy_(rg.reshape(-1))
        a, b, acc, ea = G(M), G(M), G(n_sweeps * M, torch.uint8), G(M)
        assert L.qmc_metropolis(s._h, rw.ptr, M, 0.3, n_sweeps, 5, 0, 0, a.ptr, b.ptr, acc.ptr, ea.ptr if with_acc else None,
                                None, st) == 0
        torch.cuda.synchronize()
        for g, nm in ((rw, "walkers"), (a, "logpsi"), (b, "sign"), (acc, "accept")) + (((ea, "eloc_acc"),) if with_acc else ()):
            g.check(f"qmc_metropolis {nm}")
    s.close()


# ----------------------------------------------------------------------------- forces: grad_alpha E_L and eq. 7
def check_nuclear_energy_gradient(env, d, r, threads=8):
    """qmc_nuclear_energy_gradient against the oracle at 1e-8 max(1, |.|) on walkers with |Psi|/max|Psi| > 1e-6, with
    long-double adjudication (tests.helpers.adjudicate); deterministic; returns (GPU array, exceptions)."""
    torch, ob, qb = env
    o, ox = ob.OracleSystem(d), ob.OracleSystem(d, extended=True)
    lp0 = ob.local_energy(o, r, threads=threads)[0]
    g0 = ob.nuclear_energy_gradient(o, r, threads=threads)
    gx = ob.nuclear_energy_gradient(ox, r, threads=threads)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    g = s.nuclear_energy_gradient(rg, d.n_atoms)
    g2 = s.nuclear_energy_gradient(rg, d.n_atoms)
    assert torch.equal(g, g2)
    g = g.cpu().numpy()
    s.close()
    assert g.shape == g0.shape
    keep = (lp0 - lp0.max() > math.log(1e-6)) & np.isfinite(gx).all(axis=(1, 2))
    assert keep.sum() > 0
    n_exc = adjudicate(g, g0, gx, 1e-8, scale=np.maximum(1.0, np.abs(gx)), mask=keep, what="grad_alpha E_L")
    return g, n_exc


@pytest.mark.parametrize("name,M", [("H2", 515), ("LiH", 300), ("Li2", 257), ("CO", 129)])
def test_nuclear_energy_gradient_configs(env, name, M):
    d, r = wl.CONFIGS[name](M=M)
    g, n_exc = check_nuclear_energy_gradient(env, d, r)
    assert n_exc <= max(2, M // 50)


def test_nuclear_energy_gradient_odd_systems_determinant_classes_and_500_determinants(env):
    rng = np.random.default_rng(31)
    aos = [(2, 1, 2, 1.1), (1, 0, 0, 2.0), (3, 2, 3, 0.9), (2, 1, 0, 1.3), (3, 2, 1, 0.7), (2, 0, 0, 1.5),
           (3, 0, 0, 1.2), (3, 1, 1, 0.8), (2, 1, 1, 1.3), (4, 2, 4, 1.1), (4, 1, 0, 0.9)]
    C = rng.standard_normal((len(aos), 7))
    for norm in (None, rng.uniform(0.5, 2, len(aos))):   # lone p / d functions, radial powers, custom normalisation, 3 up 2 down
        d = atom_system(3.0, aos, C, 3, 2, det_up=[[4, 0, 2], [4, 5, 2], [1, 0, 2], [4, 3, 5]],
                        det_dn=[[1, 3], [1, 3], [0, 3], [1, 2]], ci=[0.9, 0.2, -0.3, 0.15], norm=norm,
                        a_par=0.25, a_anti=0.5, b=0.8, xyz=(0.1, -0.2, 0.3))
        check_nuclear_energy_gradient(env, d, soa(rng.standard_normal((131, 5, 3)) * 1.5), threads=2)
    for with_general in (False, True):                   # every determinant class, with and without a triple substitution
        rng = np.random.default_rng(77)
        d = _classes_system(rng, with_general)
        check_nuclear_energy_gradient(env, d, soa(rng.standard_normal((203, 7, 3)) * 1.2 + np.array([0.2, 0.1, -0.3])), threads=4)
    d, r = wl.co_scan(M=40, n_geom=2)[1]                 # 500 determinants
    check_nuclear_energy_gradient(env, d, r)


def test_nuclear_energy_gradient_three_centres_bare_charge_edge_sizes_and_unsupported(env):
    torch, ob, qb = env
    rng = np.random.default_rng(4)
    from paper_2506_09743_b200.workloads import SystemDesc, expand_shells
    xyz = np.array([[0, 0, 0], [1.8, 0.2, 0], [-0.5, 1.6, 0.4], [0.3, -1.5, 1.1]], float)
    shells = [["1s", "2s", "2p", "3d"], ["1s", "2p"], ["1s", "1s", "2s"], []]      # the last centre is a bare charge
    ao = expand_shells(shells, rng.uniform(0.6, 3.0, 9))
    n_ao = len(ao[0])
    Cm = np.linalg.qr(rng.standard_normal((n_ao, n_ao)))[0][:, :7]
    up, dn = wl.select_determinants(rng, 4, [4, 5, 6], 12)
    d = SystemDesc("tri+q", xyz, np.array([6.0, 1.0, 1.0, 0.5]), 4, 4, *ao, None, Cm, up, dn,
                   np.concatenate([[0.9], rng.normal(0, 0.1, 11)]))
    for M in (1, 2, 3, 333):
        check_nuclear_energy_gradient(env, d, wl.make_walkers(rng, xyz, 8, M), threads=4)
    # hydrogen-like closed form on the GPU: grad_R E_L = (zeta - Z)(r - R)/|r - R|^3
    Z, zeta, R = 2.0, 1.6, np.array([0.3, -0.2, 0.5])
    da = atom_system(Z, [(1, 0, 0, zeta)], [[1.0]], 1, 0, xyz=tuple(R))
    rr = rng.standard_normal((257, 1, 3)) * 1.5 + R
    s = qb.QmcSystem(da)
    g = s.nuclear_energy_gradient(_to_gpu(torch, soa(rr)), 1).cpu().numpy()
    v = rr[:, 0] - R
    want = (zeta - Z) * v / np.linalg.norm(v, axis=1, keepdims=True) ** 3
    assert np.max(np.abs(g[:, 0] - want) / np.maximum(1, np.abs(want))) < 1e-10
    with pytest.raises(qb.QmcError) as ei:                          # empty batch
        s.nuclear_energy_gradient(torch.empty((1, 3, 0), dtype=torch.float64, device="cuda"), 1)
    assert ei.value.status == qb.QMC_EINVAL
    s.close()
    dl, rl = wl.lih(M=8)                                            # the e-n kernel is not covered: the call says so
    s = qb.QmcSystem(_with_en(dl, 0.3, -0.05, 0.7))
    with pytest.raises(qb.QmcError) as ei:
        s.nuclear_energy_gradient(_to_gpu(torch, rl), 2)
    assert ei.value.status == qb.QMC_EUNSUPPORTED
    s.close()


def test_nuclear_energy_gradient_near_singular_reference(env):
    rng = np.random.default_rng(78)
    aos = [(1, 0, 0, 2.5), (2, 0, 0, 1.0), (3, 0, 0, 0.7), (2, 1, 0, 1.2), (2, 1, 1, 1.2), (2, 1, 2, 1.2)]
    C = np.zeros((6, 6))
    C[:3, :2] = rng.standard_normal((3, 2))
    C[:, 2:] = rng.standard_normal((6, 4))
    d = atom_system(3.0, aos, C, 2, 1, det_up=[[0, 1], [0, 2], [3, 1], [2, 4], [5, 3]], det_dn=[[0], [0], [1], [0], [2]],
                    ci=[0.7, 0.3, -0.2, 0.25, 0.1], a_par=0.25, a_anti=0.5, b=1.0)
    r = rng.standard_normal((160, 3, 3)) * 1.3
    for w in range(0, 160, 3):   # the two up electrons at (nearly) the same distance: the s-only reference all but vanishes
        u = rng.standard_normal(3)
        r[w, 1] = u / np.linalg.norm(u) * np.linalg.norm(r[w, 0]) * (1.0 + 1e-5 * rng.uniform(0.5, 1.0))
    check_nuclear_energy_gradient(env, d, soa(r), threads=2)


@pytest.mark.parametrize("name,M", [("H2", 1), ("Li2", 131), ("CO", 67)])
def test_nuclear_energy_gradient_writes_exactly_its_output(env, name, M):
    torch, ob, qb = env
    d, r = wl.CONFIGS[name](M=M)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    r_before = rg.clone()
    out = _Guarded(torch, M * d.n_atoms * 3)
    assert qb.lib().qmc_nuclear_energy_gradient(s._h, rg.data_ptr(), M, out.ptr, torch.cuda.current_stream().cuda_stream) == 0
    torch.cuda.synchronize()
    out.check("qmc_nuclear_energy_gradient dE")
    assert torch.equal(rg, r_before)
    assert torch.equal(out.view.view(M, d.n_atoms, 3), s.nuclear_energy_gradient(rg, d.n_atoms))
    s.close()


def test_force_estimator_end_to_end(env):
    """eq. 7 through the C ABI on Li2 (20 determinants, 2048 equilibrated walkers): E_L, grad_alpha E_L and
    grad_alpha ln|Psi| from the GPU, reduced by qmc_force, against the oracle's arrays reduced by the oracle; the GPU
    reduction applied to the oracle's own arrays; and the symmetry of the molecule: the force is along z."""
    torch, ob, qb = env
    d, r = wl.li2(M=2048)
    nt = os.cpu_count() or 8
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    s.metropolis(rg, 0.3, 30, seed=5)
    rr = rg.cpu().numpy()
    lp, sg, el = s.local_energy(rg)
    dE = s.nuclear_energy_gradient(rg, d.n_atoms)
    dl = s.nuclear_log_gradient(rg, d.n_atoms)
    F, T = qb.force(el, dE, dl)
    o = ob.OracleSystem(d)
    el0 = ob.local_energy(o, rr, threads=nt)[2]
    dE0, dl0 = ob.nuclear_energy_gradient(o, rr, threads=nt), ob.nuclear_log_gradient(o, rr, threads=nt)
    F0, T0 = ob.force(el0, dE0, dl0)
    scale = np.abs(dE0).mean(axis=0) + 2 * (np.abs(el0 - el0.mean())[:, None, None] * np.abs(dl0)).mean(axis=0)
    assert np.max(np.abs(F - F0) / scale) < 1e-8 and np.max(np.abs(T - T0) / scale) < 1e-8, (F, F0)
    F1, T1 = qb.force(torch.from_numpy(el0).cuda(), torch.from_numpy(dE0).cuda(), torch.from_numpy(dl0).cuda())
    assert np.max(np.abs(F1 - F0)) < 1e-12 * np.max(scale) and np.max(np.abs(T1 - T0)) < 1e-12 * np.max(scale)
    s.close()


# ----------------------------------------------------------------------------- NEXT-3: inverse backflow
def _with_bf(d, w):
    import copy
    d2 = copy.copy(d)
    d2.backflow_w = w
    return d2


def check_backflow(env, d, r, threads=8):
    """log|Psi| / sign from the values-only kernel and from the E_L kernel, and E_L, against the oracle's general
    formulas (F.4 with its cross term, F.5 coordinate by coordinate), contract tolerances with adjudication Q24."""
    torch, ob, qb = env
    o, ox = ob.OracleSystem(d), ob.OracleSystem(d, extended=True)
    lp0, sg0, el0 = ob.local_energy(o, r, threads=threads)
    lpx, sgx, elx = ob.local_energy(ox, r, threads=threads)
    s = qb.QmcSystem(d)
    lp, sg, el = (t.cpu().numpy() for t in s.local_energy(_to_gpu(torch, r)))
    lp2, sg2 = (t.cpu().numpy() for t in s.log_psi(_to_gpu(torch, r)))
    el_b = s.local_energy(_to_gpu(torch, r))[2].cpu().numpy()
    s.close()
    assert np.array_equal(el, el_b)                               # deterministic
    keep = (lpx - lpx.max() > math.log(1e-6)) & np.isfinite(elx)
    assert np.array_equal(sg[keep], sg0[keep]) and np.array_equal(sg2[keep], sg0[keep])
    n1 = adjudicate(lp, lp0, lpx, 1e-10, mask=keep, what="backflow log|Psi| (E_L kernel)")
    n2 = adjudicate(lp2, lp0, lpx, 1e-10, mask=keep, what="backflow log|Psi| (values-only kernel)")
    n3 = adjudicate(el, el0, elx, 1e-8, scale=np.maximum(1.0, np.abs(elx)), mask=keep, what="backflow E_L")
    # eq. 6 factors of the backflow wavefunction (Jastrow entries, CI entries at the backflow coordinates, the backflow
    # weight last), with E_L / log|Psi| / sign of the same call bit-identical to qmc_local_energy's
    O0, Ox = ob.log_derivatives(o, r, threads=threads), ob.log_derivatives(ox, r, threads=threads)
    s = qb.QmcSystem(d)
    n_een = 0 if d.jastrow_een is None else len(d.jastrow_een)
    assert s.n_param() == O0.shape[1] == 6 + 7 * n_een + len(d.ci_coeff) + 1
    lpd_t, sgd_t, eld_t, O_t = s.log_derivatives(_to_gpu(torch, r))
    lpd, sgd, eld, O = (t.cpu().numpy() for t in (lpd_t, sgd_t, eld_t, O_t))
    # the estimator call (for backflow: the same two steps inside the library) against the two calls made here
    ev_u, g_u = qb.energy_gradient(eld_t, O_t)
    _, _, _, ev_f, g_f = s.local_energy_gradient(_to_gpu(torch, r))
    assert ev_f == ev_u and np.array_equal(g_f, g_u)
    s.close()
    assert np.array_equal(lpd, lp) and np.array_equal(sgd, sg) and np.array_equal(eld, el)
    n4 = adjudicate(O, O0, Ox, 1e-8, scale=np.maximum(1.0, np.abs(Ox)), mask=keep, what="backflow O_p")
    return n1, n2, max(n3, n4), int(keep.sum())


@pytest.mark.parametrize("name,M,w", [("H2", 515, 0.2), ("LiH", 300, 0.12), ("Li2", 257, 0.08), ("CO", 129, 0.05), ("CO", 3, 0.05)])
def test_backflow_configs(env, name, M, w):
    d, r = wl.CONFIGS[name](M=M)
    n1, n2, n3, nk = check_backflow(env, _with_bf(d, w), r)
    assert max(n1, n2, n3) <= max(2, nk // 20), (n1, n2, n3, nk)


def test_backflow_odd_systems_500_determinants_and_the_zero_limit(env):
    torch, ob, qb = env
    rng = np.random.default_rng(31)
    aos = [(2, 1, 2, 1.1), (1, 0, 0, 2.0), (3, 2, 3, 0.9), (2, 1, 0, 1.3), (3, 2, 1, 0.7), (2, 0, 0, 1.5),
           (3, 0, 0, 1.2), (3, 1, 1, 0.8), (2, 1, 1, 1.3), (4, 2, 4, 1.1), (4, 1, 0, 0.9)]
    C = rng.standard_normal((len(aos), 7))
    for norm in (None, rng.uniform(0.5, 2, len(aos))):   # lone p / d functions, radial powers, custom normalisation, 3 up 2 down
        d = atom_system(3.0, aos, C, 3, 2, det_up=[[4, 0, 2], [4, 5, 2], [1, 0, 2], [4, 3, 5]],
                        det_dn=[[1, 3], [1, 3], [0, 3], [1, 2]], ci=[0.9, 0.2, -0.3, 0.15], norm=norm,
                        a_par=0.25, a_anti=0.5, b=0.8, xyz=(0.1, -0.2, 0.3))
        check_backflow(env, _with_bf(d, 0.15), soa(rng.standard_normal((131, 5, 3)) * 1.5), threads=2)
    for with_general in (False, True):                   # every determinant class; spin-polarised 4 up / 3 down
        rng = np.random.default_rng(77)
        d = _classes_system(rng, with_general)
        check_backflow(env, _with_bf(d, -0.07), soa(rng.standard_normal((203, 7, 3)) * 1.2 + np.array([0.2, 0.1, -0.3])), threads=4)
    d, r = wl.co_scan(M=24, n_geom=2)[1]                 # 500 determinants
    check_backflow(env, _with_bf(d, 0.04), r)
    # one electron: the map is the identity, the hydrogen atom stays exact
    da = _with_bf(atom_system(1, [(1, 0, 0, 1.0)], [[1.0]], 1, 0), 0.3)
    s = qb.QmcSystem(da)
    el = s.local_energy(_to_gpu(torch, soa(rng.standard_normal((257, 1, 3)) * 2)))[2]
    assert float((el + 0.5).abs().max()) < 1e-12
    s.close()
    # w -> 0: the backflow kernel's general formulas against the plain path of the same library
    d, r = wl.li2(M=200)
    s0, s1 = qb.QmcSystem(d), qb.QmcSystem(_with_bf(d, 1e-200))
    lp0, sg0, el0 = (t.cpu().numpy() for t in s0.local_energy(_to_gpu(torch, r)))
    lp1, sg1, el1 = (t.cpu().numpy() for t in s1.local_energy(_to_gpu(torch, r)))
    keep = lp0 - lp0.max() > math.log(1e-6)
    assert np.array_equal(sg0, sg1) and np.max(np.abs(lp1 - lp0)) < 1e-10
    assert np.max((np.abs(el1 - el0) / np.maximum(1, np.abs(el0)))[keep]) < 1e-8
    s0.close(); s1.close()


def test_backflow_full_size_table_route_against_the_explicit_route_and_sampled_oracle(env):
    """32768 CO walkers (the size bench.py times the backflow E_L on): the table route (F.6-F.9, one elimination per
    spin) against the explicit route of the same library (every determinant eliminated on its own) on every walker, and
    against the oracle on a sample."""
    torch, ob, qb = env
    d, r = wl.co(M=32768)
    d = _with_bf(d, 0.05)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    lp, sg, el = (t.cpu().numpy() for t in s.local_energy(rg))
    lpe, sge, ele = (t.cpu().numpy() for t in s.local_energy_explicit(rg))
    s.close()
    keep = (lpe - lpe.max() > math.log(1e-6)) & np.isfinite(ele)
    assert keep.sum() > 4000                                       # the seeded batch is not equilibrated
    assert np.array_equal(sg[keep], sge[keep])
    assert np.max(np.abs(lp - lpe)[keep]) < 1e-10
    rel = np.abs(el - ele) / np.maximum(1.0, np.abs(ele))
    # the two routes share phases 1-2 and differ in the determinant algebra: 1e-8 is the contract, the bulk sits far below
    assert np.max(rel[keep]) < 1e-8, (int(np.argmax(np.where(keep, rel, 0))), float(np.max(rel[keep])))
    assert np.median(rel[keep]) < 1e-12
    idx = np.random.default_rng(5).choice(np.flatnonzero(keep), 192, replace=False)
    rs = np.ascontiguousarray(r[:, :, idx])
    o, ox = ob.OracleSystem(d), ob.OracleSystem(d, extended=True)
    lp0, sg0, el0 = ob.local_energy(o, rs, threads=8)
    lpx, sgx, elx = ob.local_energy(ox, rs, threads=8)
    assert np.array_equal(sg[idx], sg0)
    adjudicate(lp[idx], lp0, lpx, 1e-10, what="backflow log|Psi| at full size")
    adjudicate(el[idx], el0, elx, 1e-8, scale=np.maximum(1.0, np.abs(elx)), what="backflow E_L at full size")
    # the same property on equilibrated walkers (the bench's: 260 sweeps of the plain sampler of this library first), where
    # nearly all walkers sit in the criterion set and nearly singular references are typical rather than rare
    d0, r0 = wl.co(M=32768)
    s0 = qb.QmcSystem(d0)
    rg = _to_gpu(torch, r0)
    s0.metropolis(rg, 0.2, 260, seed=1234)
    s0.close()
    s = qb.QmcSystem(d)
    lp, sg, el = s.local_energy(rg)
    lpe, sge, ele = s.local_energy_explicit(rg)
    s.close()
    keep = (lpe - lpe.max() > math.log(1e-6)) & torch.isfinite(ele)
    assert int(keep.sum()) > 16000
    assert bool((sg == sge)[keep].all()) and float((lp - lpe).abs()[keep].max()) < 1e-10
    rel = ((el - ele).abs() / ele.abs().clamp(min=1.0))[keep]
    assert float(rel.max()) < 5e-9, float(rel.max())               # half the contract's bound between the two routes


@pytest.mark.parametrize("name,M,w", [("H2", 131, -0.15), ("LiH", 200, 0.1), ("Li2", 131, 0.08), ("CO", 67, 0.05)])
def test_backflow_with_the_many_body_jastrow(env, name, M, w):
    """Backflow combined with the electron-nucleus and electron-electron-nucleus Jastrow kernels (D.2, D.3,
    PAPER.md:245-253; the Jastrow factor and its derivatives sit at r, the orbitals at the backflow coordinates): E_L,
    log|Psi| from both kernels, the eq. 6 factors of all 6 + 7 n_een + n_det + 1 parameters, and the sampler."""
    d, r = wl.CONFIGS[name](M=M)
    d_en = _with_bf(_with_en(d, 0.3, -0.05, 0.7), w)
    n1, n2, n3, nk = check_backflow(env, d_en, r)
    assert max(n1, n2, n3) <= max(2, nk // 20), (n1, n2, n3, nk)
    d_all = _with_bf(_with_een(_with_en(d, 0.2, -0.03, 0.8)), w)
    n1, n2, n3, nk = check_backflow(env, d_all, r)
    assert max(n1, n2, n3) <= max(2, nk // 20), (n1, n2, n3, nk)
    check_metropolis(env, d_all, r[:, :, :64].copy(), 0.3, 3, seed=21, eloc_acc=True)


@pytest.mark.parametrize("name,M,w", [("H2", 131, -0.15), ("LiH", 200, 0.1), ("Li2", 257, 0.08), ("CO", 129, 0.05)])
def test_backflow_orbital_derivatives_and_nuclear_log_gradient(env, name, M, w):
    """d ln Psi / d C, d ln Psi / d zeta and grad_alpha ln|Psi| of a backflow wavefunction (AOs at the backflow
    coordinates; the nuclear gradient with the D.2 / D.3 Jastrow parts at r), both routes of the kernel."""
    d, r = wl.CONFIGS[name](M=M)
    check_orbital_derivatives(env, _with_bf(d, w), r)
    check_nuclear_log_gradient(env, _with_bf(_with_een(_with_en(d, 0.2, -0.03, 0.8)), w), r)


def test_backflow_sampler_unsupported_calls_and_output_bounds(env):
    torch, ob, qb = env
    d, r = wl.li2(M=301)
    d = _with_bf(d, 0.1)
    check_metropolis(env, d, r, 0.3, 8, seed=11)
    d5, r5 = wl.co(M=64)
    check_metropolis(env, _with_bf(d5, 0.05), r5, 0.2, 4, seed=12, eloc_acc=True)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    for call in (lambda: s.nuclear_energy_gradient(rg, d.n_atoms),):
        with pytest.raises(qb.QmcError) as ei:
            call()
        assert ei.value.status == qb.QMC_EUNSUPPORTED
    M = 131
    a, b, c = _Guarded(torch, M), _Guarded(torch, M), _Guarded(torch, M)
    rq = rg[:, :, :M].contiguous()
    assert qb.lib().qmc_local_energy(s._h, rq.data_ptr(), M, a.ptr, b.ptr, c.ptr, torch.cuda.current_stream().cuda_stream) == 0
    torch.cuda.synchronize()
    a.check("backflow logpsi"); b.check("backflow sign"); c.check("backflow eloc")
    a, b, c, o = _Guarded(torch, M), _Guarded(torch, M), _Guarded(torch, M), _Guarded(torch, M * s.n_param())
    assert qb.lib().qmc_log_derivatives(s._h, rq.data_ptr(), M, a.ptr, b.ptr, c.ptr, o.ptr, torch.cuda.current_stream().cuda_stream) == 0
    torch.cuda.synchronize()
    a.check("backflow logpsi (derivative call)"); b.check("backflow sign (derivative call)")
    c.check("backflow eloc (derivative call)"); o.check("backflow O")
    s.close()


def test_fused_energy_gradient_with_listed_groups_and_at_full_size(env):
    """qmc_local_energy_gradient where many groups take the explicit route (their rows are parked and added with the
    corrected energies): a system whose reference all but vanishes on a third of the walkers, against the unfused
    path of the same library and the oracle; then CO at 131072 walkers, fused against unfused."""
    torch, ob, qb = env
    rng = np.random.default_rng(78)
    aos = [(1, 0, 0, 2.5), (2, 0, 0, 1.0), (3, 0, 0, 0.7), (2, 1, 0, 1.2), (2, 1, 1, 1.2), (2, 1, 2, 1.2)]
    C = np.zeros((6, 6))
    C[:3, :2] = rng.standard_normal((3, 2))
    C[:, 2:] = rng.standard_normal((6, 4))
    d = atom_system(3.0, aos, C, 2, 1, det_up=[[0, 1], [0, 2], [3, 1], [2, 4], [5, 3]], det_dn=[[0], [0], [1], [0], [2]],
                    ci=[0.7, 0.3, -0.2, 0.25, 0.1], a_par=0.25, a_anti=0.5, b=1.0)
    r = rng.standard_normal((1601, 3, 3)) * 1.3
    for w in range(0, 1601, 3):
        u = rng.standard_normal(3)
        r[w, 1] = u / np.linalg.norm(u) * np.linalg.norm(r[w, 0]) * (1.0 + 1e-5 * rng.uniform(0.5, 1.0))
    check_log_derivatives(env, d, soa(r), threads=4)
    d, r = wl.co()
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    lp, sg, el, O = s.log_derivatives(rg)
    ev, g = qb.energy_gradient(el, O)
    del O
    lpf, sgf, elf, evf, gf = s.local_energy_gradient(rg)
    assert torch.equal(elf, el) and torch.equal(lpf, lp)
    scale = np.maximum(np.abs(g), 1e-3 * np.max(np.abs(g)))
    assert abs(evf - ev) <= 1e-12 * abs(ev) and np.max(np.abs(gf - g) / scale) < 1e-9, np.max(np.abs(gf - g) / scale)
    s.close()


def test_nuclear_energy_gradient_full_size_sampled_and_translation_invariance(env):
    """CO at the size bench.py times the call (32768 walkers, initial and after 30 sweeps): sampled walkers against the
    oracle with adjudication; on every walker translation invariance, sum_alpha grad_alpha E_L = -sum_i grad_i E_L, the
    right side by Richardson central differences of the GPU's own E_L under a rigid shift of all electrons."""
    torch, ob, qb = env
    M = 32768
    d, r = wl.co(M=M)
    s = qb.QmcSystem(d)
    o, ox = ob.OracleSystem(d), ob.OracleSystem(d, extended=True)
    nt = os.cpu_count() or 8
    rg = _to_gpu(torch, r)
    for stage in ("initial", "equilibrated"):
        if stage == "equilibrated":
            s.metropolis(rg, 0.2, 30, seed=9)
        g = s.nuclear_energy_gradient(rg, d.n_atoms)
        lp = s.log_psi(rg)[0].cpu().numpy()
        rr = rg.cpu().numpy()
        idx = np.unique(np.concatenate([np.arange(0, 32), np.arange(M - 33, M), np.random.default_rng(3).integers(0, M, 448)]))
        rs = np.ascontiguousarray(rr[:, :, idx])
        g0, gx = ob.nuclear_energy_gradient(o, rs, threads=nt), ob.nuclear_energy_gradient(ox, rs, threads=nt)
        keep = lp[idx] - lp.max() > math.log(1e-6)
        n_exc = adjudicate(g.cpu().numpy()[idx], g0, gx, 1e-8, scale=np.maximum(1.0, np.abs(gx)), mask=keep, what=f"grad_alpha E_L ({stage})")
        assert n_exc <= 8, n_exc
        # translation invariance on every walker
        def el_shift(c, t):
            r2 = rg.clone()
            r2[:, c, :] += t
            return s.local_energy(r2)[2]
        tot = g.sum(dim=1)
        good = torch.from_numpy(lp - lp.max() > math.log(1e-6)).cuda()
        for c in range(3):
            cd = lambda h: (el_shift(c, h) - el_shift(c, -h)) / (2 * h)
            a, b = cd(1e-4), cd(2e-4)
            ref = -(4 * a - b) / 3
            ok = good & ((a - b).abs() <= 1e-5 * torch.clamp(ref.abs(), min=1.0))   # where the two step sizes agree
            err = ((tot[:, c] - ref).abs() / torch.clamp(ref.abs(), min=1.0))[ok]
            assert float(ok.float().mean()) > 0.15 and float(err.max()) < 1e-5, (stage, c, float(ok.float().mean()), float(err.max()))
    s.close()


def test_h2_force_is_along_the_axis_and_antisymmetric(env):
    """eq. 7 on the H2 config (the force component along the molecular axis): 131072 walkers equilibrated
    on the GPU; by the symmetry of the molecule the force has no x, y component and F_z(A) = -F_z(B), both within the
    statistical error of the estimator (per-walker terms from the GPU, standard error over walkers)."""
    torch, ob, qb = env
    d, r = wl.h2(M=131072)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    s.metropolis(rg, 0.5, 60, seed=21)
    lp, sg, el = s.local_energy(rg)
    dE = s.nuclear_energy_gradient(rg, 2)
    dl = s.nuclear_log_gradient(rg, 2)
    F, T = qb.force(el, dE, dl)
    per = -(dE + 2.0 * (el - el.mean())[:, None, None] * dl)
    sig = (per.std(dim=0) / math.sqrt(per.shape[0])).cpu().numpy()
    assert np.all(np.abs(F[:, :2]) < 5 * sig[:, :2] + 1e-12), (F, sig)
    both = per[:, 0, 2] + per[:, 1, 2]
    assert abs(F[0, 2] + F[1, 2]) < 5 * float(both.std() / math.sqrt(both.numel())), (F, sig)
    assert np.all(np.isfinite(F)) and abs(F[0, 2]) < 1.0
    s.close()


def test_vmc_step_host_equals_the_device_calls(env):
    """qmc_vmc_step_host (host buffers, chunked over two streams) against qmc_metropolis + qmc_local_energy +
    qmc_batch_stats on device buffers: same trajectories bit for bit (Philox is keyed by the global walker index), same
    E_L and statistics up to rounding order; ragged size, 1 and 3 chunks."""
    torch, ob, qb = env
    d, r = wl.li2(M=4099)
    s = qb.QmcSystem(d)
    rg = _to_gpu(torch, r)
    s.metropolis(rg, 0.3, 7, seed=33, sweep_offset=5, walker_offset=11)
    el = s.local_energy(rg)[2]
    m0, e0 = qb.batch_stats(el)
    for n_chunks in (1, 3):
        rh = torch.from_numpy(r.copy()).pin_memory()
        eh = torch.empty(4099, dtype=torch.float64).pin_memory()
        m, e = s.vmc_step_host(rh, 0.3, 7, 33, sweep_offset=5, walker_offset=11, eloc_host=eh, n_chunks=n_chunks)
        assert torch.equal(rh, rg.cpu())
        # E_L: bit for bit except on the few walkers the explicit route re-evaluates, whose determinant slices are dealt
        # over the grid according to the size of the launch (rounding order of the slice sums)
        elc = el.cpu()
        diff = (eh - elc).abs() / elc.abs().clamp(min=1.0)
        assert float(diff.max()) < 1e-11 and int((diff > 0).sum()) <= 4099 // 50, (float(diff.max()), int((diff > 0).sum()))
        assert abs(m - m0) <= 1e-11 * abs(m0) and abs(e - e0) <= 1e-10 * e0
    s.close()
