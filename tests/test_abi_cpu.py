"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every
symbol include/qmc.h declares; setup validation that needs no GPU."""
import ctypes as C
import os
import re

import numpy as np

from paper_2506_09743_b200 import binding as qb
from paper_2506_09743_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "qmc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(qmc_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(qb.EXPORTS), declared ^ set(qb.EXPORTS)
    L = qb.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_status_strings_and_null_arguments():
    L = qb.lib()
    assert L.qmc_status_string(0) == b"ok"
    assert b"invalid" in L.qmc_status_string(qb.QMC_EINVAL)
    h = C.c_void_p()
    assert L.qmc_setup(None, 0, C.byref(h)) == qb.QMC_EINVAL
    assert L.qmc_local_energy(None, None, 4, None, None, None, None) == qb.QMC_EINVAL
    assert L.qmc_metropolis(None, None, 4, 0.1, 1, 0, 0, 0, None, None, None, None, None, None) == qb.QMC_EINVAL
    L.qmc_destroy(None)
    assert L.qmc_model_flops(None, 0) == 0.0
    assert L.qmc_n_param(None) == qb.QMC_EINVAL
    assert L.qmc_local_energy_explicit(None, None, 4, None, None, None, None) == qb.QMC_EINVAL
    assert L.qmc_set_kernel_timing(None, 1) == qb.QMC_EINVAL
    assert L.qmc_kernel_times(None, None, None) == qb.QMC_EINVAL
    assert L.qmc_log_derivatives(None, None, 4, None, None, None, None, None) == qb.QMC_EINVAL
    g = np.zeros(3)
    assert L.qmc_energy_gradient(None, None, 4, 3, None, g.ctypes.data, None) == qb.QMC_EINVAL


def test_record_stream_limit_is_reported_before_any_cuda_call():
    # more shell + atom records than the kernel parameter block holds: QMC_EUNSUPPORTED, not a crash
    from tests.helpers import atom_system
    n = 230
    d = atom_system(1.0, [(1, 0, 0, 0.5 + 0.01 * i) for i in range(n)], np.ones((n, 1)), 1, 0)
    desc, keep = qb.make_desc(d)
    h = C.c_void_p()
    assert qb.lib().qmc_setup(C.addressof(desc), 0, C.byref(h)) == qb.QMC_EUNSUPPORTED


def test_setup_validation_happens_before_any_cuda_call():
    d, _ = wl.lih(M=2)
    desc, keep = qb.make_desc(d)
    L = qb.lib()
    h = C.c_void_p()
    # bad quantum numbers
    keep["ao_l"][0] = 3
    assert L.qmc_setup(C.addressof(desc), 0, C.byref(h)) == qb.QMC_EINVAL
    keep["ao_l"][0] = 0
    keep["ao_zeta"][1] = -1.0
    assert L.qmc_setup(C.addressof(desc), 0, C.byref(h)) == qb.QMC_EINVAL


def test_no_oracle_import_in_product():
    pkg = os.path.join(ROOT, "paper_2506_09743_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle", "").replace("CPU oracle", "") or f == "workloads.py", f


def test_workload_shapes():
    for name, (ne, nao, nmo, ndet) in {"H2": (2, 2, 1, 1), "LiH": (4, 12, 2, 1), "Li2": (6, 30, 8, 20),
                                        "CO": (14, 30, 14, 100)}.items():
        d, r = wl.CONFIGS[name](M=16)
        assert (d.n_e, d.n_ao, d.n_mo, d.n_det) == (ne, nao, nmo, ndet)
        assert r.shape == (ne, 3, 16) and r.dtype == np.float64
    d, r = wl.li2(M=4, variant="28")
    assert d.n_ao == 28
    scan = wl.co_scan(M=4, n_geom=16)
    assert len(scan) == 16 and scan[0][0].n_det == 500
    assert abs(scan[15][0].atom_xyz[1, 2] - 4.0) < 1e-12 and abs(scan[0][0].atom_xyz[1, 2] - 1.6) < 1e-12
    assert np.array_equal(scan[0][0].mo_coeff, scan[7][0].mo_coeff)
    # determinism
    d2, r2 = wl.co(M=16)
    d3, r3 = wl.co(M=16)
    assert np.array_equal(r2, r3) and np.array_equal(d2.ci_coeff, d3.ci_coeff)


def test_bench_reference_arm_contract():
    # bench.py --impl reference runs on the host cores (no GPU) and prints ONE JSON line with the contract's keys
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
              "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert k in d, k
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["vs_baseline"] is None and d["dtype"] == "f64"
