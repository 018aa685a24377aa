"""Brute-force numpy restatement of the path for TINY inputs.  TEST INFRASTRUCTURE ONLY.

A second implementation, independent of oracle/sc_ivr_oracle.c, that leans on library
routines wherever the paper's object has a plain definition:

  * the potential is the UNRESTRICTED tensor sum of the force-field definition
    V = 1/2 w^2 q^2 + 1/6 Phi_ijk q_i q_j q_k + 1/24 Phi_ijkl q_i q_j q_k q_l  (full rank-3 and
    rank-4 arrays, numpy.einsum), its gradient and Hessian the tensor contractions;
  * det K and det M are numpy.linalg.det (LAPACK);
  * the prefactor phase is numpy.unwrap(angle(det K)) / 2  (continuous branch, R6);
  * the Fourier sum is the definition: z @ exp(i outer(c dt, E))  (Eq. 11).

Pure-Python loops over steps: use only for a handful of trajectories and a few hundred steps.
"""
from __future__ import annotations

import itertools

import numpy as np

VV = ((0.5, 1.0), (0.5, 0.0))
MCLACHLAN_ATELA_4 = (
    (0.1344961992774310892, 0.5153528374311229364),
    (-0.2248198030794208058, -0.085782019412973646),
    (0.7563200005156682911, 0.4415830236164665242),
    (0.3340036032863214255, 0.1288461583653841854),
)


def qff_tensors(F, coeffs):
    """Full symmetric tensors (omega[F], Phi3[F,F,F], Phi4[F,F,F,F]) from the packed block."""
    coeffs = np.asarray(coeffs, dtype=np.float64)
    omega = coeffs[:F]
    n3 = F * (F + 1) * (F + 2) // 6
    cub = coeffs[F:F + n3]
    qua = coeffs[F + n3:]
    Phi3 = np.zeros((F, F, F))
    n = 0
    for i in range(F):
        for j in range(i, F):
            for k in range(j, F):
                for perm in set(itertools.permutations((i, j, k))):
                    Phi3[perm] = cub[n]
                n += 1
    Phi4 = np.zeros((F, F, F, F))
    n = 0
    for i in range(F):
        for j in range(i, F):
            for perm in set(itertools.permutations((i, i, j, j))):
                Phi4[perm] = qua[n]
            n += 1
    return omega, Phi3, Phi4


class QFF:
    def __init__(self, F, coeffs):
        self.F = F
        self.omega, self.Phi3, self.Phi4 = qff_tensors(F, coeffs)
        self.mass = np.ones(F)

    def V(self, q):
        return (0.5 * np.sum(self.omega ** 2 * q ** 2)
                + np.einsum("ijk,i,j,k->", self.Phi3, q, q, q) / 6.0
                + np.einsum("ijkl,i,j,k,l->", self.Phi4, q, q, q, q) / 24.0)

    def grad(self, q):
        return (self.omega ** 2 * q + 0.5 * np.einsum("ajk,j,k->a", self.Phi3, q, q)
                + np.einsum("ajkl,j,k,l->a", self.Phi4, q, q, q) / 6.0)

    def hess(self, q):
        return (np.diag(self.omega ** 2) + np.einsum("abk,k->ab", self.Phi3, q)
                + 0.5 * np.einsum("abkl,k,l->ab", self.Phi4, q, q))


class Morse:
    """Uncoupled Morse oscillators; coeffs = {D, a, q_e, m} per mode (F = 1: config 1)."""

    def __init__(self, F, coeffs):
        c = np.asarray(coeffs, dtype=np.float64).reshape(F, 4)
        self.F = F
        self.D, self.a, self.qe, self.mass = c[:, 0], c[:, 1], c[:, 2], c[:, 3]

    def V(self, q):
        y = np.exp(-self.a * (q - self.qe))
        return np.sum(self.D * (1 - y) ** 2)

    def grad(self, q):
        y = np.exp(-self.a * (q - self.qe))
        return 2 * self.D * self.a * y * (1 - y)

    def hess(self, q):
        y = np.exp(-self.a * (q - self.qe))
        return np.diag(2 * self.D * self.a ** 2 * y * (2 * y - 1))


def make_pes(F, kind, coeffs):
    return QFF(F, coeffs) if kind == 1 else Morse(F, coeffs)


def trajectory(pes, gamma, dt, nsteps, p0, q0, chi, scheme=VV):
    """One trajectory.  Returns dict with per-step arrays (length nsteps+1):
    p, q [.,F], S, M [.,2F,2F] in (p,q) order, detK, detM, phi (continuous), ovl (complex), z."""
    F = pes.F
    gamma = np.asarray(gamma, dtype=np.float64)
    p = np.array(p0, dtype=np.float64)
    q = np.array(q0, dtype=np.float64)
    p_eq, q_eq = np.asarray(chi[:F]), np.asarray(chi[F:])
    M = np.eye(2 * F)
    S = 0.0
    rec = dict(p=[], q=[], S=[], M=[], detK=[], detM=[], ovl=[])
    G = np.diag(gamma)
    Gi = np.diag(1.0 / gamma)
    minv = np.diag(1.0 / pes.mass)
    for c in range(nsteps + 1):
        Mpp, Mpq, Mqp, Mqq = M[:F, :F], M[:F, F:], M[F:, :F], M[F:, F:]
        K = 0.5 * (Mqq + Gi @ Mpp @ G - 1j * Mqp @ G + 1j * Gi @ Mpq)
        rec["detK"].append(np.linalg.det(K))
        rec["detM"].append(np.linalg.det(M))
        dq, dp = q_eq - q, p_eq - p
        rec["ovl"].append(np.exp(np.sum(-0.25 * gamma * dq ** 2 - dp ** 2 / (4 * gamma))
                                 + 0.5j * np.sum((p_eq + p) * dq)))
        rec["p"].append(p.copy()); rec["q"].append(q.copy()); rec["S"].append(S); rec["M"].append(M.copy())
        if c == nsteps:
            break
        for b, a in scheme:
            if b != 0.0:
                H = pes.hess(q)
                S -= b * dt * pes.V(q)
                p = p - b * dt * pes.grad(q)
                kick = np.eye(2 * F)
                kick[:F, F:] = -b * dt * H
                M = kick @ M
            if a != 0.0:
                S += a * dt * 0.5 * np.sum(p * p / pes.mass)
                q = q + a * dt * p / pes.mass
                drift = np.eye(2 * F)
                drift[F:, :F] = a * dt * minv
                M = drift @ M
    out = {k: np.array(v) for k, v in rec.items()}
    out["phi"] = 0.5 * np.unwrap(np.angle(out["detK"]))
    out["z"] = out["ovl"] * np.exp(1j * (out["S"] + out["phi"]))
    return out


def spectrum(pes, gamma, dt, nsteps, p0q0, chi, E, weights=None, det_tol=1e-6, scheme=VV):
    """Eq. 11 by the definition, for a tiny batch.  p0q0 [2F][n].  Returns (I [k], n_good, A [n][k])."""
    F = pes.F
    p0q0 = np.asarray(p0q0, dtype=np.float64).reshape(2 * F, -1)
    n = p0q0.shape[1]
    E = np.asarray(E, dtype=np.float64)
    tw = np.exp(1j * np.outer(np.arange(nsteps + 1) * dt, E))
    I = np.zeros(E.size)
    A_all = np.zeros((n, E.size), dtype=np.complex128)
    n_good = 0
    for j in range(n):
        t = trajectory(pes, gamma, dt, nsteps, p0q0[:F, j], p0q0[F:, j], chi, scheme)
        good = np.all(np.isfinite(t["z"])) and np.all(np.abs(t["detM"] - 1.0) <= det_tol)
        A = t["z"] @ tw
        A_all[j] = A
        if good:
            n_good += 1
            I += (1.0 if weights is None else weights[j]) * np.abs(A) ** 2
    if n_good == 0:
        return np.zeros(E.size), 0, A_all
    T = nsteps * dt
    return I * dt ** 2 / ((2 * np.pi) ** (F + 1) * T * n_good), n_good, A_all


def spectrum_combo(pes, gamma, dt, nsteps, p0q0, chis, eps, E, scheme=VV):
    """Eq. 11 by the definition for the reference state |chi> = sum_m eps[m] |p_m, q_m>:
    <chi|p q> = sum_m conj(eps[m]) <p_m q_m|p q>, each overlap from Eq. 3 in closed form.  Returns (I [k], n_good)."""
    F = pes.F
    gamma = np.asarray(gamma, dtype=np.float64)
    p0q0 = np.asarray(p0q0, dtype=np.float64).reshape(2 * F, -1)
    chis = np.asarray(chis, dtype=np.float64).reshape(-1, 2 * F)
    eps = np.asarray(eps, dtype=np.complex128).reshape(-1)
    E = np.asarray(E, dtype=np.float64)
    tw = np.exp(1j * np.outer(np.arange(nsteps + 1) * dt, E))
    I = np.zeros(E.size)
    n_good = 0
    for j in range(p0q0.shape[1]):
        t = trajectory(pes, gamma, dt, nsteps, p0q0[:F, j], p0q0[F:, j], chis[0], scheme)
        ovl = np.zeros(nsteps + 1, dtype=np.complex128)
        for m in range(chis.shape[0]):
            dq = chis[m, F:][None, :] - t["q"]
            dp = chis[m, :F][None, :] - t["p"]
            a = np.sum(-0.25 * gamma * dq ** 2 - dp ** 2 / (4 * gamma), axis=1)
            b = 0.5 * np.sum((chis[m, :F][None, :] + t["p"]) * dq, axis=1)
            ovl += np.conj(eps[m]) * np.exp(a + 1j * b)
        z = ovl * np.exp(1j * (t["S"] + t["phi"]))
        if np.all(np.isfinite(z)) and np.all(np.abs(t["detM"] - 1.0) <= 1e-6):
            n_good += 1
            I += np.abs(z @ tw) ** 2
    if n_good == 0:
        return np.zeros(E.size), 0
    return I * dt ** 2 / ((2 * np.pi) ** (F + 1) * nsteps * dt * n_good), n_good
