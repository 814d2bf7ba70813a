"""Thin ctypes binding of libqmcb200 (include/qmc.h).  Argument marshalling only:
every step of the path runs in the CUDA kernels.  PyTorch supplies device memory and
streams.  There is no CPU fallback: a missing library raises."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

QMC_OK, QMC_EINVAL, QMC_EUNSUPPORTED, QMC_ECUDA, QMC_ENOMEM, QMC_ETOOLARGE = 0, -1, -2, -3, -4, -5
_lib = None

EXPORTS = ["qmc_setup", "qmc_destroy", "qmc_local_energy", "qmc_log_psi", "qmc_metropolis", "qmc_batch_stats",
           "qmc_fp64_peak", "qmc_model_flops", "qmc_launch_count", "qmc_status_string", "qmc_n_param", "qmc_local_energy_explicit", "qmc_set_kernel_timing", "qmc_kernel_times",
           "qmc_log_derivatives", "qmc_energy_gradient", "qmc_local_energy_host", "qmc_orbital_derivatives",
           "qmc_nuclear_log_gradient", "qmc_nuclear_energy_gradient", "qmc_force", "qmc_local_energy_gradient",
           "qmc_static_scratch_init", "qmc_batch_stats_static", "qmc_vmc_step_host"]


class QmcError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"libqmcb200 status {status}: {msg}")
        self.status = status


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


def lib():
    """Load libqmcb200.so (building it with nvcc if the sources are newer)."""
    global _lib
    if _lib is None:
        so = _build.SO
        if _build.needs_build():
            so = _build.build()
        if not os.path.exists(so):
            raise ImportError("libqmcb200.so is missing and could not be built; there is no CPU fallback")
        L = C.CDLL(so)
        vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
        L.qmc_setup.restype = C.c_int
        L.qmc_setup.argtypes = [vp, C.c_int, C.POINTER(vp)]
        L.qmc_destroy.restype = None
        L.qmc_destroy.argtypes = [vp]
        L.qmc_local_energy.restype = C.c_int
        L.qmc_local_energy.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.qmc_local_energy_explicit.restype = C.c_int
        L.qmc_local_energy_explicit.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.qmc_set_kernel_timing.restype = C.c_int
        L.qmc_set_kernel_timing.argtypes = [vp, C.c_int]
        L.qmc_kernel_times.restype = C.c_int
        L.qmc_kernel_times.argtypes = [vp, vp, vp]
        L.qmc_orbital_derivatives.restype = C.c_int
        L.qmc_orbital_derivatives.argtypes = [vp, vp, i64, vp, vp, vp]
        L.qmc_nuclear_log_gradient.restype = C.c_int
        L.qmc_nuclear_log_gradient.argtypes = [vp, vp, i64, vp, vp]
        L.qmc_local_energy_gradient.restype = C.c_int
        L.qmc_local_energy_gradient.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp]
        L.qmc_nuclear_energy_gradient.restype = C.c_int
        L.qmc_nuclear_energy_gradient.argtypes = [vp, vp, i64, vp, vp]
        L.qmc_force.restype = C.c_int
        L.qmc_force.argtypes = [vp, vp, vp, i64, C.c_int32, vp, vp, vp]
        L.qmc_local_energy_host.restype = C.c_int
        L.qmc_local_energy_host.argtypes = [vp, vp, i64, vp, vp, vp, C.c_int32]
        L.qmc_vmc_step_host.restype = C.c_int
        L.qmc_vmc_step_host.argtypes = [vp, vp, i64, dbl, C.c_int32, C.c_uint64, C.c_uint64, i64, vp, vp, vp, C.c_int32]
        L.qmc_log_psi.restype = C.c_int
        L.qmc_log_psi.argtypes = [vp, vp, i64, vp, vp, vp]
        L.qmc_metropolis.restype = C.c_int
        L.qmc_metropolis.argtypes = [vp, vp, i64, dbl, C.c_int32, C.c_uint64, C.c_uint64, i64, vp, vp, vp, vp, vp, vp]
        L.qmc_batch_stats.restype = C.c_int
        L.qmc_batch_stats.argtypes = [vp, i64, vp, vp, vp]
        L.qmc_static_scratch_init.restype = C.c_int
        L.qmc_static_scratch_init.argtypes = [C.c_int]
        L.qmc_batch_stats_static.restype = C.c_int
        L.qmc_batch_stats_static.argtypes = [vp, i64, vp, vp]
        L.qmc_fp64_peak.restype = C.c_int
        L.qmc_fp64_peak.argtypes = [C.c_int, C.c_int, C.c_int, vp]
        L.qmc_model_flops.restype = dbl
        L.qmc_model_flops.argtypes = [vp, C.c_int]
        L.qmc_launch_count.restype = i64
        L.qmc_launch_count.argtypes = [C.c_int]
        L.qmc_n_param.restype = C.c_int
        L.qmc_n_param.argtypes = [vp]
        L.qmc_log_derivatives.restype = C.c_int
        L.qmc_log_derivatives.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp]
        L.qmc_energy_gradient.restype = C.c_int
        L.qmc_energy_gradient.argtypes = [vp, vp, i64, C.c_int32, vp, vp, vp]
        L.qmc_status_string.restype = C.c_char_p
        L.qmc_status_string.argtypes = [C.c_int]
        _lib = L
    return _lib


def _check(rc):
    if rc != QMC_OK:
        raise QmcError(rc, lib().qmc_status_string(rc).decode())


def _np(a):
    return None if a is None else a.ctypes.data


def _dp(t):
    return None if t is None else t.data_ptr()


def _stream(stream=None):
    st = stream if stream is not None else torch.cuda.current_stream()
    return st.cuda_stream


def make_desc(d):
    """SystemDesc-like object -> (ctypes struct, keep-alive dict of contiguous arrays)."""
    f64 = lambda a: np.ascontiguousarray(a, np.float64)
    i32 = lambda a: np.ascontiguousarray(a, np.int32)
    k = dict(atom_xyz=f64(d.atom_xyz), atom_Z=f64(d.atom_Z), ao_atom=i32(d.ao_atom), ao_n=i32(d.ao_n),
             ao_l=i32(d.ao_l), ao_m=i32(d.ao_m), ao_zeta=f64(d.ao_zeta),
             ao_norm=None if d.ao_norm is None else f64(d.ao_norm), mo_coeff=f64(d.mo_coeff),
             det_up=i32(d.det_up), det_dn=i32(d.det_dn), ci_coeff=f64(d.ci_coeff))
    desc = _Desc(int(k["atom_xyz"].shape[0]), _np(k["atom_xyz"]), _np(k["atom_Z"]), int(d.n_up), int(d.n_dn),
                 int(k["ao_atom"].shape[0]), _np(k["ao_atom"]), _np(k["ao_n"]), _np(k["ao_l"]), _np(k["ao_m"]),
                 _np(k["ao_zeta"]), _np(k["ao_norm"]), int(k["mo_coeff"].shape[1]), _np(k["mo_coeff"]),
                 int(k["ci_coeff"].shape[0]), _np(k["det_up"]), _np(k["det_dn"]), _np(k["ci_coeff"]),
                 float(d.jastrow_a_par), float(d.jastrow_a_anti), float(d.jastrow_b),
                 float(getattr(d, "jastrow_en_w0", 0.0)), float(getattr(d, "jastrow_en_w1", 0.0)),
                 float(getattr(d, "jastrow_en_w2", 0.0)), 0, None, float(getattr(d, "backflow_w", 0.0)))
    een = getattr(d, "jastrow_een", None)
    if een is not None and len(een):
        k["een"] = np.ascontiguousarray(een, np.float64).reshape(-1, 7)
        desc.n_een, desc.een_params = int(k["een"].shape[0]), _np(k["een"])
    return desc, k


class QmcSystem:
    """Handle returned by qmc_setup; methods mirror the C calls."""

    def __init__(self, d, device: int = 0):
        self.n_up, self.n_dn = int(d.n_up), int(d.n_dn)
        self.n_e = self.n_up + self.n_dn
        self.device = device
        desc, keep = make_desc(d)
        h = C.c_void_p()
        _check(lib().qmc_setup(C.addressof(desc), device, C.byref(h)))
        del keep
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            lib().qmc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk_r(self, r):
        assert r.is_cuda and r.dtype == torch.float64 and r.is_contiguous()
        assert r.dim() == 3 and r.shape[0] == self.n_e and r.shape[1] == 3, "walkers must be [n_e,3,M]"
        return int(r.shape[2])

    def local_energy(self, r, logpsi=None, sign=None, eloc=None, stream=None):
        """qmc_local_energy: r float64 cuda [n_e,3,M] -> (logpsi, sign, eloc) each [M]."""
        M = self._chk_r(r)
        new = lambda: torch.empty(M, dtype=torch.float64, device=r.device)
        logpsi = new() if logpsi is None else logpsi
        sign = new() if sign is None else sign
        eloc = new() if eloc is None else eloc
        _check(lib().qmc_local_energy(self._h, _dp(r), M, _dp(logpsi), _dp(sign), _dp(eloc), _stream(stream)))
        return logpsi, sign, eloc

    def set_kernel_timing(self, enabled: bool = True):
        """qmc_set_kernel_timing: events around the two kernels of every E_L call (bench.py's roofline)."""
        _check(lib().qmc_set_kernel_timing(self._h, int(bool(enabled))))

    def kernel_times(self):
        """qmc_kernel_times: (table-path kernel ms, explicit fallback kernel ms) of the most recent timed call."""
        a, b = C.c_double(), C.c_double()
        _check(lib().qmc_kernel_times(self._h, C.addressof(a), C.addressof(b)))
        return a.value, b.value

    def local_energy_explicit(self, r, logpsi=None, sign=None, eloc=None, stream=None):
        """qmc_local_energy_explicit: the same outputs with every determinant eliminated on its own (Fig. 11's
        "explicit" route) for every walker."""
        M = self._chk_r(r)
        new = lambda: torch.empty(M, dtype=torch.float64, device=r.device)
        logpsi = new() if logpsi is None else logpsi
        sign = new() if sign is None else sign
        eloc = new() if eloc is None else eloc
        _check(lib().qmc_local_energy_explicit(self._h, _dp(r), M, _dp(logpsi), _dp(sign), _dp(eloc), _stream(stream)))
        return logpsi, sign, eloc

    def local_energy_host(self, r_host, out_host=None, n_chunks: int = 2):
        """qmc_local_energy_host: r_host float64 CPU tensor [n_e,3,M] (pinned for copy/compute overlap) ->
        out_host float64 CPU tensor [3,M] = (logpsi, sign, eloc).  Synchronous."""
        assert (not r_host.is_cuda) and r_host.dtype == torch.float64 and r_host.is_contiguous()
        assert r_host.dim() == 3 and r_host.shape[0] == self.n_e and r_host.shape[1] == 3
        M = int(r_host.shape[2])
        if out_host is None:
            out_host = torch.empty((3, M), dtype=torch.float64).pin_memory()
        assert (not out_host.is_cuda) and out_host.dtype == torch.float64 and out_host.is_contiguous()
        assert tuple(out_host.shape) == (3, M)
        _check(lib().qmc_local_energy_host(self._h, r_host.data_ptr(), M, out_host[0].data_ptr(), out_host[1].data_ptr(),
                                           out_host[2].data_ptr(), int(n_chunks)))
        return out_host

    def vmc_step_host(self, r_host, step, n_sweeps, seed, sweep_offset=0, walker_offset=0, eloc_host=None, n_chunks: int = 2):
        """qmc_vmc_step_host: r_host float64 CPU tensor [n_e,3,M] is sampled in place (n_sweeps sweeps) and its E_L
        evaluated; returns (mean, stderr); eloc_host (CPU tensor [M]) receives the per-walker energies.  Synchronous."""
        assert (not r_host.is_cuda) and r_host.dtype == torch.float64 and r_host.is_contiguous()
        assert r_host.dim() == 3 and r_host.shape[0] == self.n_e and r_host.shape[1] == 3
        M = int(r_host.shape[2])
        if eloc_host is not None:
            assert (not eloc_host.is_cuda) and eloc_host.dtype == torch.float64 and eloc_host.is_contiguous() and eloc_host.numel() == M
        m, e = C.c_double(), C.c_double()
        _check(lib().qmc_vmc_step_host(self._h, r_host.data_ptr(), M, float(step), int(n_sweeps), int(seed), int(sweep_offset),
                                       int(walker_offset), None if eloc_host is None else eloc_host.data_ptr(),
                                       C.addressof(m), C.addressof(e), int(n_chunks)))
        return m.value, e.value

    def log_psi(self, r, logpsi=None, sign=None, stream=None):
        M = self._chk_r(r)
        new = lambda: torch.empty(M, dtype=torch.float64, device=r.device)
        logpsi = new() if logpsi is None else logpsi
        sign = new() if sign is None else sign
        _check(lib().qmc_log_psi(self._h, _dp(r), M, _dp(logpsi), _dp(sign), _stream(stream)))
        return logpsi, sign

    def metropolis(self, r, step, n_sweeps, seed, sweep_offset=0, walker_offset=0, logpsi=None, sign=None,
                   accept=None, eloc_acc=None, want_accept=False, want_eloc_acc=False, count=False, stream=None):
        """qmc_metropolis: r is updated in place.  Returns dict(logpsi, sign, accept, eloc_acc, n_accepted)."""
        M = self._chk_r(r)
        new = lambda: torch.empty(M, dtype=torch.float64, device=r.device)
        logpsi = new() if logpsi is None else logpsi
        sign = new() if sign is None else sign
        if want_accept and accept is None:
            accept = torch.empty((n_sweeps, M), dtype=torch.uint8, device=r.device)
        if want_eloc_acc and eloc_acc is None:
            eloc_acc = new()
        nacc = C.c_int64(-1)
        _check(lib().qmc_metropolis(self._h, _dp(r), M, float(step), int(n_sweeps), int(seed), int(sweep_offset),
                                    int(walker_offset), _dp(logpsi), _dp(sign), _dp(accept), _dp(eloc_acc),
                                    C.addressof(nacc) if count else None, _stream(stream)))
        return dict(logpsi=logpsi, sign=sign, accept=accept, eloc_acc=eloc_acc,
                    n_accepted=nacc.value if count else None)

    def orbital_derivatives(self, r, n_ao: int, n_mo: int, stream=None):
        """qmc_orbital_derivatives: (dC[M, n_ao, n_mo], dzeta[M, n_ao]) = d ln Psi / d C, d ln Psi / d zeta."""
        M = self._chk_r(r)
        dC = torch.empty((M, n_ao, n_mo), dtype=torch.float64, device=r.device)
        dz = torch.empty((M, n_ao), dtype=torch.float64, device=r.device)
        _check(lib().qmc_orbital_derivatives(self._h, _dp(r), M, _dp(dC), _dp(dz), _stream(stream)))
        return dC, dz

    def nuclear_log_gradient(self, r, n_atoms: int, stream=None):
        """qmc_nuclear_log_gradient: dR[M, n_atoms, 3] = grad_alpha ln|Psi| (eq. 7's grad_alpha ln rho / 2)."""
        M = self._chk_r(r)
        dR = torch.empty((M, n_atoms, 3), dtype=torch.float64, device=r.device)
        _check(lib().qmc_nuclear_log_gradient(self._h, _dp(r), M, _dp(dR), _stream(stream)))
        return dR

    def nuclear_energy_gradient(self, r, n_atoms: int, stream=None):
        """qmc_nuclear_energy_gradient: dE[M, n_atoms, 3] = grad_alpha E_L (first term of eq. 7)."""
        M = self._chk_r(r)
        dE = torch.empty((M, n_atoms, 3), dtype=torch.float64, device=r.device)
        _check(lib().qmc_nuclear_energy_gradient(self._h, _dp(r), M, _dp(dE), _stream(stream)))
        return dE

    def n_param(self) -> int:
        return int(lib().qmc_n_param(self._h))

    def log_derivatives(self, r, logpsi=None, sign=None, eloc=None, O=None, stream=None):
        """qmc_log_derivatives: (logpsi, sign, eloc, O[M, n_param]) with O_p = (dPsi/dtheta_p)/Psi (eq. 6),
        theta = (a_par, a_anti, b, en_w0, en_w1, en_w2, 7 parameters per e-e-n term, d_0 .. d_{n_det-1}, and -- for a
        backflow wavefunction -- the backflow weight w)."""
        M = self._chk_r(r)
        new = lambda: torch.empty(M, dtype=torch.float64, device=r.device)
        logpsi = new() if logpsi is None else logpsi
        sign = new() if sign is None else sign
        eloc = new() if eloc is None else eloc
        if O is None:
            O = torch.empty((M, self.n_param()), dtype=torch.float64, device=r.device)
        assert O.is_cuda and O.dtype == torch.float64 and O.is_contiguous() and tuple(O.shape) == (M, self.n_param())
        _check(lib().qmc_log_derivatives(self._h, _dp(r), M, _dp(logpsi), _dp(sign), _dp(eloc), _dp(O),
                                         _stream(stream)))
        return logpsi, sign, eloc, O

    def local_energy_gradient(self, r, logpsi=None, sign=None, eloc=None, stream=None):
        """qmc_local_energy_gradient: (logpsi, sign, eloc, E_v, grad[n_param]) -- E_L and the eq. 6 estimator in one pass,
        the per-walker derivatives never leave the SMs."""
        M = self._chk_r(r)
        new = lambda: torch.empty(M, dtype=torch.float64, device=r.device)
        logpsi = new() if logpsi is None else logpsi
        sign = new() if sign is None else sign
        eloc = new() if eloc is None else eloc
        ev = C.c_double()
        g = np.empty(self.n_param())
        _check(lib().qmc_local_energy_gradient(self._h, _dp(r), M, _dp(logpsi), _dp(sign), _dp(eloc), C.addressof(ev), _np(g),
                                               _stream(stream)))
        return logpsi, sign, eloc, ev.value, g

    def model_flops(self, which: int) -> float:
        return lib().qmc_model_flops(self._h, which)


def batch_stats(x, stream=None):
    """qmc_batch_stats: mean and standard error of a float64 cuda vector."""
    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
    m, s = C.c_double(), C.c_double()
    _check(lib().qmc_batch_stats(_dp(x), x.numel(), C.addressof(m), C.addressof(s), _stream(stream)))
    return m.value, s.value


def batch_stats_static(x, out, stream=None):
    """qmc_batch_stats_static: the allocation-free variant; out = float64 cuda tensor [2] supplied by the caller receives
    {mean, standard error}.  Asynchronous; at most 2^26 values; calls on one device must not overlap on the GPU."""
    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 2
    _check(lib().qmc_batch_stats_static(_dp(x), x.numel(), _dp(out), _stream(stream)))
    return out


def energy_gradient(eloc, O, stream=None):
    """qmc_energy_gradient: (E_v, grad[n_param]) of eq. 6 from device E_L [M] and O [M, n_param]."""
    assert eloc.is_cuda and O.is_cuda and eloc.dtype == O.dtype == torch.float64
    assert eloc.is_contiguous() and O.is_contiguous() and O.shape[0] == eloc.numel()
    ev = C.c_double()
    g = np.empty(int(O.shape[1]))
    _check(lib().qmc_energy_gradient(_dp(eloc), _dp(O), eloc.numel(), int(O.shape[1]), C.addressof(ev), _np(g),
                                     _stream(stream)))
    return ev.value, g


def force(eloc, dE, dlnpsi, stream=None):
    """qmc_force: (F[n_atoms, 3], terms[2, n_atoms, 3]) of eq. 7 from device E_L [M], grad_alpha E_L and
    grad_alpha ln|Psi| [M, n_atoms, 3]."""
    assert eloc.is_cuda and dE.is_cuda and dlnpsi.is_cuda and eloc.dtype == dE.dtype == dlnpsi.dtype == torch.float64
    assert eloc.is_contiguous() and dE.is_contiguous() and dlnpsi.is_contiguous()
    assert dE.shape == dlnpsi.shape and dE.shape[0] == eloc.numel() and dE.shape[2] == 3
    na = int(dE.shape[1])
    F, T = np.empty((na, 3)), np.empty((2, na, 3))
    _check(lib().qmc_force(_dp(eloc), _dp(dE), _dp(dlnpsi), eloc.numel(), na, _np(F), _np(T), _stream(stream)))
    return F, T


def fp64_peak(kind: int = 0, reps: int = 5, device: int = 0) -> float:
    """qmc_fp64_peak: measured TFLOP/s of the DFMA (0) / DMMA (1) / mixed (2) microbenchmark."""
    v = C.c_double()
    _check(lib().qmc_fp64_peak(device, kind, reps, C.addressof(v)))
    return v.value


def launch_count(reset: bool = False) -> int:
    return lib().qmc_launch_count(1 if reset else 0)
