"""ctypes access to oracle/sc_ivr_oracle.c.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

build() compiles the C file with gcc -O2 -fopenmp (no fast-math) into oracle/libsc_ivr_oracle.so.
All arrays are host numpy float64, C-contiguous, in the layouts of include/sc_ivr.h.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sc_ivr_oracle.c")
_LIB = os.path.join(_HERE, "libsc_ivr_oracle.so")
_lib = None

_dp = C.POINTER(C.c_double)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.sc_ivr_oracle_max_f.restype = C.c_int
        _lib.sc_ivr_oracle_num_threads.restype = C.c_int
        _lib.sc_ivr_oracle_eval_pes.restype = C.c_int
        _lib.sc_ivr_oracle_eval_pes.argtypes = [C.c_int, C.c_int, _dp, C.c_long, _dp, C.c_long, _dp, _dp, _dp]
        _lib.sc_ivr_oracle_propagate.restype = C.c_int
        _lib.sc_ivr_oracle_propagate.argtypes = [
            C.c_int, C.c_int, _dp, C.c_long, _dp, C.c_double, C.c_int, C.c_int, C.c_int, C.c_double,
            _dp, C.c_long, _dp, _dp, _dp, _dp, _dp, C.POINTER(C.c_ubyte), _dp]
        _lib.sc_ivr_oracle_fourier.restype = C.c_int
        _lib.sc_ivr_oracle_fourier.argtypes = [_dp, C.c_long, C.c_int, C.c_double, _dp, C.c_int, C.c_int, _dp]
        _lib.sc_ivr_oracle_run.restype = C.c_int
        _lib.sc_ivr_oracle_run.argtypes = [
            C.c_int, C.c_int, _dp, C.c_long, _dp, C.c_double, C.c_int, C.c_int, C.c_int, C.c_double,
            _dp, _dp, C.c_long, _dp, _dp, C.c_int, C.c_int, _dp, C.POINTER(C.c_longlong)]
        _lib.sc_ivr_oracle_run_combo.restype = C.c_int
        _lib.sc_ivr_oracle_run_combo.argtypes = [
            C.c_int, C.c_int, _dp, C.c_long, _dp, C.c_double, C.c_int, C.c_int, C.c_int, C.c_double,
            _dp, _dp, C.c_long, _dp, C.c_int, _dp, _dp, C.c_int, C.c_int, _dp, C.POINTER(C.c_longlong)]
    return _lib


def num_threads() -> int:
    return int(lib().sc_ivr_oracle_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def eval_pes(F, kind, coeffs, q):
    """q [F][n] -> V [n], g [F][n], H [F][F][n]."""
    coeffs = _f64(coeffs)
    q = _f64(q).reshape(F, -1)
    n = q.shape[1]
    V = np.empty(n)
    g = np.empty((F, n))
    H = np.empty((F, F, n))
    rc = lib().sc_ivr_oracle_eval_pes(F, kind, _p(coeffs), coeffs.size, _p(q), n, _p(V), _p(g), _p(H))
    if rc:
        raise ValueError(f"oracle eval_pes rc={rc}")
    return V, g, H


def propagate(F, kind, coeffs, gamma, dt, nsteps, p0q0, chi=None, integrator=0, det_stride=1,
              det_tol=1e-6, want_z=False, want_M=True):
    """Returns dict(pq [2F][n], S [n], M [4][F][F][n], theta [n], good [n] uint8, z [n][nsteps+1] complex)."""
    coeffs = _f64(coeffs)
    gamma = _f64(gamma)
    p0q0 = _f64(p0q0).reshape(2 * F, -1)
    n = p0q0.shape[1]
    chi_a = None if chi is None else _f64(chi)
    pq = np.empty((2 * F, n))
    S = np.empty(n)
    M = np.empty((4, F, F, n)) if want_M else None
    th = np.empty(n)
    good = np.empty(n, dtype=np.uint8)
    z = np.empty((n, nsteps + 1, 2)) if want_z else None
    rc = lib().sc_ivr_oracle_propagate(
        F, kind, _p(coeffs), coeffs.size, _p(gamma), float(dt), int(nsteps), int(integrator), int(det_stride),
        float(det_tol), _p(p0q0), n, _p(chi_a), _p(pq), _p(S), _p(M), _p(th),
        good.ctypes.data_as(C.POINTER(C.c_ubyte)), _p(z))
    if rc:
        raise ValueError(f"oracle propagate rc={rc}")
    out = dict(pq=pq, S=S, M=M, theta=th, good=good)
    if want_z:
        out["z"] = z[..., 0] + 1j * z[..., 1]
    return out


def fourier(z, dt, E, mode=0):
    """z [n][nsteps+1] complex -> A [n][k] complex, A_j(E_i) = sum_c z_jc e^{i E_i c dt}."""
    z = np.ascontiguousarray(np.asarray(z, dtype=np.complex128))
    if z.ndim == 1:
        z = z[None, :]
    n, ns1 = z.shape
    E = _f64(E)
    zz = np.ascontiguousarray(z.view(np.float64).reshape(n, ns1, 2))
    A = np.empty((n, E.size, 2))
    rc = lib().sc_ivr_oracle_fourier(_p(zz), n, ns1 - 1, float(dt), _p(E), E.size, int(mode), _p(A))
    if rc:
        raise ValueError(f"oracle fourier rc={rc}")
    return A[..., 0] + 1j * A[..., 1]


def run(F, kind, coeffs, gamma, dt, nsteps, p0q0, chi, E, weights=None, integrator=0, det_stride=1,
        det_tol=1e-6, fourier_mode=1):
    """The whole path.  Returns (I [k], n_good, rc)."""
    coeffs = _f64(coeffs)
    gamma = _f64(gamma)
    p0q0 = _f64(p0q0).reshape(2 * F, -1)
    n = p0q0.shape[1]
    chi = _f64(chi)
    E = _f64(E)
    w = None if weights is None else _f64(weights)
    I = np.empty(E.size)
    ng = C.c_longlong(0)
    rc = lib().sc_ivr_oracle_run(
        F, kind, _p(coeffs), coeffs.size, _p(gamma), float(dt), int(nsteps), int(integrator), int(det_stride),
        float(det_tol), _p(p0q0), _p(w), n, _p(chi), _p(E), E.size, int(fourier_mode), _p(I), C.byref(ng))
    if rc not in (0, 5):
        raise ValueError(f"oracle run rc={rc}")
    return I, int(ng.value), rc


def run_combo(F, kind, coeffs, gamma, dt, nsteps, p0q0, chis, eps, E, weights=None, integrator=0, det_stride=1,
              det_tol=1e-6, fourier_mode=1):
    """The whole path for the reference state |chi> = sum_m eps[m] |chis[m]>.
    chis [ncs][2F] (p_m then q_m), eps [ncs] complex.  Returns (I [k], n_good, rc)."""
    coeffs = _f64(coeffs)
    gamma = _f64(gamma)
    p0q0 = _f64(p0q0).reshape(2 * F, -1)
    n = p0q0.shape[1]
    chis = _f64(chis).reshape(-1, 2 * F)
    ncs = chis.shape[0]
    e = np.asarray(eps, dtype=np.complex128).reshape(ncs)
    ee = np.ascontiguousarray(np.stack([e.real, e.imag], axis=1))
    E = _f64(E)
    w = None if weights is None else _f64(weights)
    I = np.empty(E.size)
    ng = C.c_longlong(0)
    rc = lib().sc_ivr_oracle_run_combo(
        F, kind, _p(coeffs), coeffs.size, _p(gamma), float(dt), int(nsteps), int(integrator), int(det_stride),
        float(det_tol), _p(p0q0), _p(w), n, _p(chis), ncs, _p(ee), _p(E), E.size, int(fourier_mode), _p(I), C.byref(ng))
    if rc not in (0, 5):
        raise ValueError(f"oracle run_combo rc={rc}")
    return I, int(ng.value), rc


def run_workload(w, ntraj=None, fourier_mode=1, **kw):
    """Convenience: run a paper_1312_4698_b200.inputs.Workload (optionally its first ntraj trajectories)."""
    p0q0 = w.p0q0 if ntraj is None else np.ascontiguousarray(w.p0q0[:, :ntraj])
    return run(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, p0q0, w.chi, w.E,
               fourier_mode=fourier_mode, **kw)


def find_peaks(I, rel_height=1e-3):
    """R19: strict local maxima over both neighbours with height >= rel_height * max(I)."""
    I = np.asarray(I)
    thr = rel_height * I.max()
    idx = [i for i in range(1, I.size - 1) if I[i] > I[i - 1] and I[i] >= I[i + 1] and I[i] >= thr]
    return np.array(idx, dtype=np.int64)
