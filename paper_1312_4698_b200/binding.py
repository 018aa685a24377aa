"""Thin ctypes binding of libsc_ivr.so (include/sc_ivr.h).  Argument marshalling only.

PyTorch supplies device memory and the CUDA stream; every step of the path runs in the library's
kernels.  There is no CPU fallback: loading fails loudly when the library is missing, and
sc_ivr_create fails when there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsc_ivr.so")

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, ENOGOOD = 0, 1, 2, 3, 4, 5
PES_MORSE1D, PES_QFF, PES_MORSE_UNCOUPLED = 0, 1, 2

EXPORTS = [
    "sc_ivr_create", "sc_ivr_destroy", "sc_ivr_last_error", "sc_ivr_workspace_bytes", "sc_ivr_min_batch",
    "sc_ivr_run", "sc_ivr_host_staging_bytes", "sc_ivr_run_host", "sc_ivr_propagate_workspace_bytes",
    "sc_ivr_propagate", "sc_ivr_eval_pes", "sc_ivr_fourier_workspace_bytes", "sc_ivr_fourier",
    "sc_ivr_fourier_power_workspace_bytes", "sc_ivr_fourier_power", "sc_ivr_multi_workspace_bytes", "sc_ivr_run_multi",
    "sc_ivr_fp64_probe", "sc_ivr_set_timing", "sc_ivr_last_timings", "sc_ivr_last_fallbacks",
    "sc_ivr_fourier_static", "sc_ivr_fourier_static_scratch_bytes", "sc_ivr_fourier_static_last_error", "sc_ivr_assemble_z",
]
STATIC_SCRATCH_BYTES = 16 << 20  # SC_IVR_STATIC_SCRATCH_BYTES


class sc_ivr_options(C.Structure):
    _fields_ = [("det_stride", C.c_int), ("det_tol", C.c_double), ("integrator", C.c_int),
                ("lu_growth_max", C.c_double), ("fourier_mode", C.c_int)]


class ScIvrError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"sc_ivr status {status}: {msg}")
        self.status = status


_lib = None
_dp = C.POINTER(C.c_double)
_vp = C.c_void_p


def lib():
    """Load the C-ABI library (never builds it: run `python -m paper_1312_4698_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1312_4698_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.sc_ivr_create.restype = C.c_int
    L.sc_ivr_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, _dp, C.c_size_t, _dp, C.c_double, C.c_int,
                                C.POINTER(sc_ivr_options)]
    L.sc_ivr_destroy.restype = None
    L.sc_ivr_destroy.argtypes = [_vp]
    L.sc_ivr_last_error.restype = C.c_char_p
    L.sc_ivr_last_error.argtypes = [_vp]
    L.sc_ivr_workspace_bytes.restype = C.c_size_t
    L.sc_ivr_workspace_bytes.argtypes = [_vp, C.c_longlong, C.c_int, C.c_longlong]
    L.sc_ivr_min_batch.restype = C.c_longlong
    L.sc_ivr_min_batch.argtypes = [_vp]
    run_args = [_vp, _vp, _vp, C.c_longlong, _dp, _dp, C.c_int, _vp, C.POINTER(C.c_longlong), _vp, C.c_size_t, _vp]
    L.sc_ivr_run.restype = C.c_int
    L.sc_ivr_run.argtypes = run_args
    L.sc_ivr_run_host.restype = C.c_int
    L.sc_ivr_run_host.argtypes = run_args
    L.sc_ivr_host_staging_bytes.restype = C.c_size_t
    L.sc_ivr_host_staging_bytes.argtypes = [_vp, C.c_longlong, C.c_int]
    L.sc_ivr_propagate_workspace_bytes.restype = C.c_size_t
    L.sc_ivr_propagate_workspace_bytes.argtypes = [_vp, C.c_longlong, C.c_int]
    L.sc_ivr_propagate.restype = C.c_int
    L.sc_ivr_propagate.argtypes = [_vp, _vp, C.c_longlong, C.c_int, _dp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_size_t, _vp]
    L.sc_ivr_eval_pes.restype = C.c_int
    L.sc_ivr_eval_pes.argtypes = [_vp, _vp, C.c_longlong, _vp, _vp, _vp, _vp]
    L.sc_ivr_fourier_workspace_bytes.restype = C.c_size_t
    L.sc_ivr_fourier_workspace_bytes.argtypes = [_vp, C.c_longlong, C.c_int]
    L.sc_ivr_multi_workspace_bytes.restype = C.c_size_t
    L.sc_ivr_multi_workspace_bytes.argtypes = [_vp, C.c_longlong, C.c_int, C.c_int, C.c_longlong]
    L.sc_ivr_run_multi.restype = C.c_int
    L.sc_ivr_run_multi.argtypes = [_vp, _vp, _vp, C.c_longlong, _dp, C.c_int, _dp, C.c_int, _dp, C.c_int, _vp,
                                   C.POINTER(C.c_longlong), _vp, C.c_size_t, _vp]
    L.sc_ivr_fourier_power_workspace_bytes.restype = C.c_size_t
    L.sc_ivr_fourier_power_workspace_bytes.argtypes = [_vp, C.c_longlong, C.c_int]
    L.sc_ivr_fourier_power.restype = C.c_int
    L.sc_ivr_fourier_power.argtypes = [_vp, _vp, C.c_longlong, _dp, C.c_int, _vp, _vp, C.c_size_t, _vp]
    L.sc_ivr_fourier.restype = C.c_int
    L.sc_ivr_fourier.argtypes = [_vp, _vp, C.c_longlong, _dp, C.c_int, _vp, _vp, C.c_size_t, _vp]
    L.sc_ivr_assemble_z.restype = C.c_int
    L.sc_ivr_assemble_z.argtypes = [_vp, _vp, C.c_longlong, C.c_int, _vp, _vp, _vp]
    L.sc_ivr_fourier_static.restype = C.c_int
    L.sc_ivr_fourier_static.argtypes = [_vp, C.c_longlong, C.c_int, C.c_double, _vp, C.c_int, _vp, _vp]
    L.sc_ivr_fourier_static_scratch_bytes.restype = C.c_size_t
    L.sc_ivr_fourier_static_scratch_bytes.argtypes = [C.c_longlong, C.c_int, C.c_int]
    L.sc_ivr_fourier_static_last_error.restype = C.c_char_p
    L.sc_ivr_fourier_static_last_error.argtypes = []
    L.sc_ivr_fp64_probe.restype = C.c_int
    L.sc_ivr_fp64_probe.argtypes = [C.c_int, C.c_int, _dp, _dp]
    L.sc_ivr_set_timing.restype = None
    L.sc_ivr_set_timing.argtypes = [_vp, C.c_int]
    L.sc_ivr_last_timings.restype = C.c_int
    L.sc_ivr_last_timings.argtypes = [_vp, _dp]
    L.sc_ivr_last_fallbacks.restype = C.c_longlong
    L.sc_ivr_last_fallbacks.argtypes = [_vp]
    _lib = L
    return L


def _host(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _hp(a):
    return a.ctypes.data_as(_dp)


def _dev(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _workspace(nbytes, device):
    import torch
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def fp64_probe(mode=0, iters=20000):
    """Achieved FP64 FLOP/s of a register-only DFMA (mode 0) or DMMA m8n8k4 (mode 1) loop, and its ms."""
    fl, ms = C.c_double(0), C.c_double(0)
    rc = lib().sc_ivr_fp64_probe(mode, iters, C.byref(fl), C.byref(ms))
    if rc:
        raise ScIvrError(rc, lib().sc_ivr_last_error(None).decode())
    return fl.value, ms.value


def fourier_static_scratch_bytes(n, nsteps, k):
    """sc_ivr_fourier_static_scratch_bytes: what (n, nsteps, k) needs of the STATIC_SCRATCH_BYTES array (0 = out of range)."""
    return int(lib().sc_ivr_fourier_static_scratch_bytes(int(n), int(nsteps), int(k)))


def fourier_static(z, E, dt, A_out):
    """sc_ivr_fourier_static: A_out[j][i] = sum_c z[c][j] e^{i E_i c dt} for callers that cannot allocate device memory.

    Nothing is allocated, here or in the library: z DEVICE complex128 [nsteps+1, n], E DEVICE float64 [k] and the output
    A_out DEVICE complex128 [n, k] are all the caller's; the scratch is the library's static array (one per device, shared
    by every call: do not let two calls overlap on the GPU).  Sizes beyond the array raise ScIvrError(EINVAL)."""
    import torch
    assert z.is_cuda and z.dtype == torch.complex128 and z.is_contiguous() and z.dim() == 2
    assert E.is_cuda and E.dtype == torch.float64 and E.is_contiguous() and E.dim() == 1
    n, k = z.shape[1], E.shape[0]
    assert A_out.is_cuda and A_out.dtype == torch.complex128 and A_out.is_contiguous() and tuple(A_out.shape) == (n, k)
    rc = lib().sc_ivr_fourier_static(_dev(z), n, z.shape[0] - 1, float(dt), _dev(E), k, _dev(A_out), _stream())
    if rc:
        raise ScIvrError(rc, lib().sc_ivr_fourier_static_last_error().decode())
    return A_out


class ScIvr:
    """One context = one PES + (gamma, dt, nsteps, options).  Methods mirror the C entry points."""

    def __init__(self, F, pes_kind, pes_coeffs, gamma, dt, nsteps, det_stride=1, det_tol=1e-6, integrator=0,
                 lu_growth_max=0.0, fourier_mode=0):
        self._h = _vp(None)
        L = lib()
        co, ga = _host(pes_coeffs), _host(gamma)
        opt = sc_ivr_options(int(det_stride), float(det_tol), int(integrator), float(lu_growth_max), int(fourier_mode))
        rc = L.sc_ivr_create(C.byref(self._h), int(F), int(pes_kind), _hp(co), co.size, _hp(ga), float(dt), int(nsteps),
                             C.byref(opt))
        if rc:
            self._h = _vp(None)
            raise ScIvrError(rc, L.sc_ivr_last_error(None).decode())
        self.F, self.nsteps, self.dt = int(F), int(nsteps), float(dt)

    @classmethod
    def from_workload(cls, w, **kw):
        return cls(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, **kw)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value and _lib is not None:
            _lib.sc_ivr_destroy(self._h)
            self._h = _vp(None)

    __del__ = close

    def _check(self, rc, allow=()):
        if rc and rc not in allow:
            raise ScIvrError(rc, lib().sc_ivr_last_error(self._h).decode())
        return rc

    def min_batch(self):
        return int(lib().sc_ivr_min_batch(self._h))

    def workspace_bytes(self, ntraj, k, max_batch=0):
        return int(lib().sc_ivr_workspace_bytes(self._h, int(ntraj), int(k), int(max_batch)))

    def host_staging_bytes(self, ntraj, k):
        return int(lib().sc_ivr_host_staging_bytes(self._h, int(ntraj), int(k)))

    def last_fallbacks(self):
        """Trajectory-steps of the last synchronising run that needed the pivoted eliminations (-1: not read back)."""
        return int(lib().sc_ivr_last_fallbacks(self._h))

    def set_timing(self, on=True):
        lib().sc_ivr_set_timing(self._h, 1 if on else 0)

    def last_timings(self):
        out = (C.c_double * 6)()
        self._check(lib().sc_ivr_last_timings(self._h, out))
        t = list(out)
        return dict(propagate_ms=t[0], zassemble_ms=t[1], twiddle_ms=t[2], fourier_ms=t[3], reduce_ms=t[4], launches=int(t[5]))

    def run(self, p0q0, chi, E, weights=None, I_out=None, workspace=None, max_batch=0, want_n_good=True):
        """sc_ivr_run: p0q0 DEVICE torch [2F, ntraj] float64 -> (I DEVICE torch [k], n_good or None, status)."""
        import torch
        assert p0q0.is_cuda and p0q0.dtype == torch.float64 and p0q0.is_contiguous()
        ntraj = p0q0.shape[1]
        chi, E = _host(chi), _host(E)
        k = E.size
        if I_out is None:
            I_out = torch.empty(k, dtype=torch.float64, device=p0q0.device)
        if workspace is None:
            workspace = _workspace(self.workspace_bytes(ntraj, k, max_batch), p0q0.device)
        ng = C.c_longlong(-1)
        rc = lib().sc_ivr_run(self._h, _dev(p0q0), _dev(weights), ntraj, _hp(chi), _hp(E), k, _dev(I_out),
                              C.byref(ng) if want_n_good else None, _dev(workspace), workspace.numel(), _stream())
        self._check(rc, allow=(ENOGOOD,))
        return I_out, (int(ng.value) if want_n_good else None), rc

    def run_host(self, p0q0, chi, E, weights=None, I_out=None, workspace=None, max_batch=0):
        """sc_ivr_run_host: p0q0 HOST numpy/pinned torch [2F, ntraj] -> (I HOST numpy [k], n_good, status)."""
        import torch
        if isinstance(p0q0, torch.Tensor):
            assert not p0q0.is_cuda and p0q0.dtype == torch.float64 and p0q0.is_contiguous()
            pq_ptr, ntraj = C.c_void_p(p0q0.data_ptr()), p0q0.shape[1]
        else:
            p0q0 = _host(p0q0)
            pq_ptr, ntraj = C.c_void_p(p0q0.ctypes.data), p0q0.shape[1]
        chi, E = _host(chi), _host(E)
        k = E.size
        if I_out is None:
            I_out = np.empty(k, dtype=np.float64)
        I_ptr = C.c_void_p(I_out.data_ptr() if isinstance(I_out, torch.Tensor) else I_out.ctypes.data)
        w_ptr = None
        if weights is not None:
            weights = weights if isinstance(weights, torch.Tensor) else _host(weights)
            w_ptr = C.c_void_p(weights.data_ptr() if isinstance(weights, torch.Tensor) else weights.ctypes.data)
        if workspace is None:
            workspace = _workspace(self.workspace_bytes(ntraj, k, max_batch) + self.host_staging_bytes(ntraj, k), "cuda")
        ng = C.c_longlong(-1)
        rc = lib().sc_ivr_run_host(self._h, pq_ptr, w_ptr, ntraj, _hp(chi), _hp(E), k, I_ptr, C.byref(ng),
                                   _dev(workspace), workspace.numel(), _stream())
        self._check(rc, allow=(ENOGOOD,))
        return I_out, int(ng.value), rc

    def propagate(self, p0q0, nsteps_run, chi=None, want_M=True, want_theta=True, want_z=False):
        """sc_ivr_propagate: returns dict of DEVICE tensors pq [2F,n], S [n], M [4,F,F,n], theta [n], good [n], z [c,n] complex."""
        import torch
        assert p0q0.is_cuda and p0q0.dtype == torch.float64 and p0q0.is_contiguous()
        F, n, dev = self.F, p0q0.shape[1], p0q0.device
        pq = torch.empty((2 * F, n), dtype=torch.float64, device=dev)
        S = torch.empty(n, dtype=torch.float64, device=dev)
        M = torch.empty((4, F, F, n), dtype=torch.float64, device=dev) if want_M else None
        th = torch.empty(n, dtype=torch.float64, device=dev) if want_theta else None
        good = torch.empty(n, dtype=torch.uint8, device=dev)
        z = torch.empty((nsteps_run + 1, n, 2), dtype=torch.float64, device=dev) if want_z else None
        ws = _workspace(lib().sc_ivr_propagate_workspace_bytes(self._h, n, int(nsteps_run)), dev)
        chi_h = None if chi is None else _host(chi)
        rc = lib().sc_ivr_propagate(self._h, _dev(p0q0), n, int(nsteps_run), None if chi_h is None else _hp(chi_h),
                                    _dev(pq), _dev(S), _dev(M), _dev(th), _dev(good), _dev(z), _dev(ws), ws.numel(), _stream())
        self._check(rc)
        out = dict(pq=pq, S=S, M=M, theta=th, good=good)
        if want_z:
            out["z"] = torch.view_as_complex(z)
        return out

    def eval_pes(self, q):
        """sc_ivr_eval_pes: q DEVICE [F, n] -> V [n], g [F, n], H [F, F, n]."""
        import torch
        assert q.is_cuda and q.dtype == torch.float64 and q.is_contiguous()
        F, n, dev = self.F, q.shape[1], q.device
        V = torch.empty(n, dtype=torch.float64, device=dev)
        g = torch.empty((F, n), dtype=torch.float64, device=dev)
        H = torch.empty((F, F, n), dtype=torch.float64, device=dev)
        self._check(lib().sc_ivr_eval_pes(self._h, _dev(q), n, _dev(V), _dev(g), _dev(H), _stream()))
        return V, g, H

    def assemble_z(self, raw, want_theta=True):
        """sc_ivr_assemble_z: raw DEVICE float64 [nsteps_run+1, n, 4] -> (z DEVICE complex [nsteps_run+1, n], theta [n] or None)."""
        import torch
        assert raw.is_cuda and raw.dtype == torch.float64 and raw.is_contiguous() and raw.dim() == 3 and raw.shape[2] == 4
        rows, n = raw.shape[0], raw.shape[1]
        z = torch.empty((rows, n, 2), dtype=torch.float64, device=raw.device)
        th = torch.empty(n, dtype=torch.float64, device=raw.device) if want_theta else None
        self._check(lib().sc_ivr_assemble_z(self._h, _dev(raw), n, rows - 1, _dev(z), _dev(th), _stream()))
        return torch.view_as_complex(z), th

    def _lib_multi_bytes(self, ntraj, k, ncs, max_batch=0):
        return int(lib().sc_ivr_multi_workspace_bytes(self._h, int(ntraj), int(k), int(ncs), int(max_batch)))

    def run_multi(self, p0q0, chis, eps, E, weights=None, workspace=None, max_batch=0):
        """sc_ivr_run_multi: reference states |chi_n> = sum_m eps[n][m] |chis[m]>; p0q0 DEVICE [2F, ntraj];
        chis [ncs, 2F], eps [nchi, ncs] complex (host) -> (I DEVICE [nchi, k], n_good, status)."""
        import torch
        assert p0q0.is_cuda and p0q0.dtype == torch.float64 and p0q0.is_contiguous()
        ntraj = p0q0.shape[1]
        chis = _host(np.asarray(chis, dtype=np.float64).reshape(-1, 2 * self.F))
        ncs = chis.shape[0]
        e = np.asarray(eps, dtype=np.complex128).reshape(-1, ncs)
        nchi = e.shape[0]
        ee = _host(np.stack([e.real, e.imag], axis=2))
        E = _host(E)
        I = torch.empty((nchi, E.size), dtype=torch.float64, device=p0q0.device)
        if workspace is None:
            workspace = _workspace(self._lib_multi_bytes(ntraj, E.size, ncs, max_batch), p0q0.device)
        ng = C.c_longlong(0)
        rc = lib().sc_ivr_run_multi(self._h, _dev(p0q0), _dev(weights) if weights is not None else None, ntraj, _hp(chis), ncs,
                                    _hp(ee), nchi, _hp(E), E.size, _dev(I), C.byref(ng), _dev(workspace), workspace.numel(),
                                    _stream())
        self._check(rc, allow=(5,))
        return I, int(ng.value), rc

    def fourier_power(self, z, E):
        """sc_ivr_fourier_power (chirp-z kernels): z DEVICE complex [nsteps+1, n] -> |A|^2 DEVICE [n, k]."""
        import torch
        assert z.is_cuda and z.dtype == torch.complex128 and z.is_contiguous() and z.shape[0] == self.nsteps + 1
        n, dev = z.shape[1], z.device
        E = _host(E)
        P = torch.empty((n, E.size), dtype=torch.float64, device=dev)
        ws = _workspace(lib().sc_ivr_fourier_power_workspace_bytes(self._h, n, E.size), dev)
        self._check(lib().sc_ivr_fourier_power(self._h, _dev(z), n, _hp(E), E.size, _dev(P), _dev(ws), ws.numel(), _stream()))
        return P

    def fourier(self, z, E):
        """sc_ivr_fourier: z DEVICE complex [nsteps+1, n] (time-major) -> A DEVICE complex [n, k]."""
        import torch
        assert z.is_cuda and z.dtype == torch.complex128 and z.is_contiguous() and z.shape[0] == self.nsteps + 1
        n, dev = z.shape[1], z.device
        E = _host(E)
        A = torch.empty((n, E.size), dtype=torch.complex128, device=dev)
        ws = _workspace(lib().sc_ivr_fourier_workspace_bytes(self._h, n, E.size), dev)
        self._check(lib().sc_ivr_fourier(self._h, _dev(z), n, _hp(E), E.size, _dev(A), _dev(ws), ws.numel(), _stream()))
        return A
