"""Seeded synthetic workloads for the TA-SC-IVR hot path (numpy only).

This module holds DATA recipes and nothing of the method's arithmetic: it draws
potential-energy-surface coefficients and Husimi-distributed initial conditions
and packs them in the layouts the C ABI (include/sc_ivr.h) and the CPU oracle
(oracle/) both take. It is the only module the CUDA path and the oracle share.

The paper's workloads are four molecules with F = 1, 3, 6, 9 vibrational modes
(PAPER.md:157), 128..65536 trajectories, ~4000 steps
(PAPER.md:206), a Morse surface for H2 and fitted ab-initio surfaces for the
rest.  The fitted surfaces are not available; BASELINE.json's synthetic quartic
force fields of the same shape stand in for them ("Input recipe").

Generator: numpy default_rng (PCG64), seed = 13124698 + config number.
Draw order (fixed): (1) frequency splittings xi[F] (configs 4, 5 only);
(2) cubic constants, one standard normal per i<=j<=k in lexicographic order;
(3) q0 = q_eq + N(0,1)[ntraj,F]/sqrt(gamma); (4) p0 = p_eq + N(0,1)[ntraj,F]*sqrt(gamma).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

CM1_PER_HARTREE = 219474.6313632  # CODATA; 1 E_h in cm^-1 (not in the paper)
SEED_BASE = 13124698

PES_MORSE1D = 0
PES_QFF = 1
PES_MORSE_UNCOUPLED = 2


def n_cubic(F: int) -> int:
    return F * (F + 1) * (F + 2) // 6


def n_quartic(F: int) -> int:
    return F * (F + 1) // 2


def cubic_index_list(F: int):
    """(i, j, k) with i <= j <= k in lexicographic order: layout of the cubic block."""
    return [(i, j, k) for i in range(F) for j in range(i, F) for k in range(j, F)]


def quartic_index_list(F: int):
    """(i, j) with i <= j in lexicographic order: layout of the Phi_iijj block."""
    return [(i, j) for i in range(F) for j in range(i, F)]


@dataclass
class Workload:
    """One problem instance, in the units and layouts of include/sc_ivr.h."""

    name: str
    F: int
    pes_kind: int
    pes_coeffs: np.ndarray  # float64, layout per pes_kind (see include/sc_ivr.h)
    gamma: np.ndarray  # [F]
    dt: float
    nsteps: int
    chi: np.ndarray  # [2F] = p_eq[F] then q_eq[F]
    E: np.ndarray  # [k] atomic units, equally spaced end points included
    p0q0: np.ndarray  # [2F, ntraj] SoA: rows 0..F-1 = p_k, rows F..2F-1 = q_k
    seed: int
    meta: dict = field(default_factory=dict)

    @property
    def ntraj(self) -> int:
        return self.p0q0.shape[1]

    @property
    def k(self) -> int:
        return self.E.shape[0]

    def prefix(self, n: int) -> "Workload":
        """Same problem on the first n trajectories."""
        w = Workload(**{**self.__dict__})
        w.p0q0 = np.ascontiguousarray(self.p0q0[:, :n])
        w.name = f"{self.name}[:{n}]"
        return w

    def with_steps(self, nsteps: int) -> "Workload":
        w = Workload(**{**self.__dict__})
        w.nsteps = int(nsteps)
        return w

    def with_grid(self, k: int, e_min_cm=0.0, e_max_cm=20000.0) -> "Workload":
        w = Workload(**{**self.__dict__})
        w.E = energy_grid(k, e_min_cm, e_max_cm)
        return w


def energy_grid(k: int, e_min_cm: float = 0.0, e_max_cm: float = 20000.0) -> np.ndarray:
    """k equally spaced energies, E_1 = E_min ... E_k = E_max, atomic units."""
    return np.linspace(e_min_cm, e_max_cm, k) / CM1_PER_HARTREE


def husimi_sample(rng: np.random.Generator, ntraj: int, gamma, p_eq, q_eq) -> np.ndarray:
    """Draw (p0, q0) from the Husimi density of |p_eq, q_eq>.

    q0 ~ N(q_eq, 1/gamma), p0 ~ N(p_eq, gamma) per mode; q is drawn first, then p.
    Returns the SoA block [2F, ntraj] (rows p_1..p_F, q_1..q_F; PAPER.md:139 layout).
    """
    gamma = np.asarray(gamma, dtype=np.float64)
    F = gamma.shape[0]
    q0 = np.asarray(q_eq) + rng.standard_normal((ntraj, F)) / np.sqrt(gamma)
    p0 = np.asarray(p_eq) + rng.standard_normal((ntraj, F)) * np.sqrt(gamma)
    out = np.empty((2 * F, ntraj), dtype=np.float64)
    out[:F] = p0.T
    out[F:] = q0.T
    return np.ascontiguousarray(out)


def qff_coeffs(omega, phi3_reduced, quartic_scale: float = 5e-4) -> np.ndarray:
    """Pack a quartic force field for the library (mass-weighted normal coordinates, m = 1).

    omega[F] in E_h; phi3_reduced: one value per i<=j<=k (lexicographic), the cubic
    constant in dimensionless normal coordinates, energy units.  Mass-weighted tensors:
    Phi_ijk = phi_ijk sqrt(w_i w_j w_k); Phi_iijj = phi_iijj w_i w_j with
    phi_iijj = quartic_scale * sqrt(w_i w_j) (BASELINE.json configs 2-4; R16).
    Layout: omega[F], cubic block, quartic block.
    """
    omega = np.asarray(omega, dtype=np.float64)
    F = omega.shape[0]
    cub = np.empty(n_cubic(F))
    for n, (i, j, k) in enumerate(cubic_index_list(F)):
        cub[n] = phi3_reduced[n] * np.sqrt(omega[i] * omega[j] * omega[k])
    qua = np.empty(n_quartic(F))
    for n, (i, j) in enumerate(quartic_index_list(F)):
        qua[n] = quartic_scale * np.sqrt(omega[i] * omega[j]) * omega[i] * omega[j]
    return np.concatenate([omega, cub, qua])


_QFF_OMEGA_CM = {
    2: [1648.0, 3832.0, 3943.0],
    3: [1187.0, 1257.0, 1529.0, 1782.0, 2843.0, 2897.0],
    4: [1367.0] * 3 + [1583.0] * 2 + [3036.0] + [3157.0] * 3,
}
_DEFAULTS = {
    1: dict(ntraj=1024, nsteps=3000, k=2000),
    2: dict(ntraj=16384, nsteps=4000, k=4000),
    3: dict(ntraj=65536, nsteps=4000, k=4000),
    4: dict(ntraj=131072, nsteps=4000, k=4000),
    5: dict(ntraj=1 << 20, nsteps=4000, k=4000),
}


def make_config(config: int, ntraj: int | None = None, nsteps: int | None = None,
                k: int | None = None) -> Workload:
    """BASELINE.json config 1..5.  Smaller ntraj takes a PREFIX of the full seeded draw
    only for config 5 (as BASELINE.json's sweep needs); for configs 1-4 the draw has
    exactly `ntraj` rows, so the default sizes reproduce the named workload."""
    if config not in _DEFAULTS:
        raise ValueError("config must be 1..5")
    d = _DEFAULTS[config]
    ntraj = d["ntraj"] if ntraj is None else int(ntraj)
    nsteps = d["nsteps"] if nsteps is None else int(nsteps)
    k = d["k"] if k is None else int(k)
    dt = 10.0
    E = energy_grid(k)
    if config == 1:
        seed = SEED_BASE + 1
        rng = np.random.default_rng(seed)
        D, a, mu, qe = 0.1744, 1.02, 918.6, 1.4
        omega = a * np.sqrt(2.0 * D / mu)
        gamma = np.array([mu * omega])
        p_eq = np.array([np.sqrt(mu * omega)])
        q_eq = np.array([qe])
        coeffs = np.array([D, a, qe, mu])
        p0q0 = husimi_sample(rng, ntraj, gamma, p_eq, q_eq)
        return Workload("config1_morse_h2", 1, PES_MORSE1D, coeffs, gamma, dt, nsteps,
                        np.concatenate([p_eq, q_eq]), E, p0q0, seed,
                        dict(omega=np.array([omega]), mass=np.array([mu])))
    surf = 4 if config == 5 else config
    seed = SEED_BASE + surf
    rng = np.random.default_rng(seed)
    omega = np.array(_QFF_OMEGA_CM[surf]) / CM1_PER_HARTREE
    F = omega.shape[0]
    if surf == 4:
        xi = rng.standard_normal(F)
        omega = omega * (1.0 + 1e-3 * xi)
    phi3 = rng.standard_normal(n_cubic(F)) * (0.02 * omega.min())
    coeffs = qff_coeffs(omega, phi3)
    gamma = omega.copy()
    p_eq = np.sqrt(omega)
    q_eq = np.zeros(F)
    if config == 5:
        full = husimi_sample(rng, _DEFAULTS[5]["ntraj"], gamma, p_eq, q_eq)
        p0q0 = np.ascontiguousarray(full[:, :ntraj])
    else:
        p0q0 = husimi_sample(rng, ntraj, gamma, p_eq, q_eq)
    names = {2: "config2_qff_h2o", 3: "config3_qff_ch2o", 4: "config4_qff_ch4", 5: "config5_qff_ch4_sweep"}
    return Workload(names[config], F, PES_QFF, coeffs, gamma, dt, nsteps,
                    np.concatenate([p_eq, q_eq]), E, p0q0, seed,
                    dict(omega=omega, mass=np.ones(F)))


def make_harmonic(omega, ntraj: int, nsteps: int, dt: float, E: np.ndarray, seed: int = 7,
                  q_eq=None, p_eq=None) -> Workload:
    """Purely harmonic QFF (all Phi = 0), gamma_k = omega_k: the north star's closed-form case."""
    omega = np.asarray(omega, dtype=np.float64)
    F = omega.shape[0]
    coeffs = np.concatenate([omega, np.zeros(n_cubic(F)), np.zeros(n_quartic(F))])
    q_eq = np.zeros(F) if q_eq is None else np.asarray(q_eq, dtype=np.float64)
    p_eq = np.sqrt(omega) if p_eq is None else np.asarray(p_eq, dtype=np.float64)
    rng = np.random.default_rng(seed)
    p0q0 = husimi_sample(rng, ntraj, omega, p_eq, q_eq)
    return Workload("harmonic", F, PES_QFF, coeffs, omega.copy(), dt, nsteps,
                    np.concatenate([p_eq, q_eq]), np.asarray(E, dtype=np.float64), p0q0, seed,
                    dict(omega=omega, mass=np.ones(F)))


def make_random_qff(F: int, ntraj: int, nsteps: int, k: int, seed: int, dt: float = 10.0,
                    omega_cm_range=(1000.0, 3500.0)) -> Workload:
    """A random weakly anharmonic QFF of any F (same recipe as configs 2-4); for tests."""
    rng = np.random.default_rng(seed)
    omega = np.sort(rng.uniform(*omega_cm_range, size=F)) / CM1_PER_HARTREE
    phi3 = rng.standard_normal(n_cubic(F)) * (0.02 * omega.min())
    coeffs = qff_coeffs(omega, phi3)
    gamma = omega.copy()
    p_eq = np.sqrt(omega)
    q_eq = np.zeros(F)
    p0q0 = husimi_sample(rng, ntraj, gamma, p_eq, q_eq)
    return Workload(f"random_qff_F{F}", F, PES_QFF, coeffs, gamma, dt, nsteps,
                    np.concatenate([p_eq, q_eq]), energy_grid(k), p0q0, seed,
                    dict(omega=omega, mass=np.ones(F)))


def make_uncoupled_morse(F: int, ntraj: int, nsteps: int, k: int, seed: int = 11,
                         dt: float = 10.0) -> Workload:
    """F uncoupled Morse oscillators (Fig. 6): mode 0 is config 1's H2
    oscillator; the others scale its depth and range mildly.  coeffs: {D,a,q_e,m} per mode."""
    rng = np.random.default_rng(seed)
    D = 0.1744 * (1.0 + 0.05 * np.arange(F))
    a = 1.02 * (1.0 - 0.03 * np.arange(F))
    qe = np.full(F, 1.4)
    mu = 918.6 * (1.0 + 0.1 * np.arange(F))
    omega = a * np.sqrt(2.0 * D / mu)
    gamma = mu * omega
    p_eq = np.sqrt(mu * omega)
    q_eq = qe.copy()
    coeffs = np.stack([D, a, qe, mu], axis=1).reshape(-1)
    p0q0 = husimi_sample(rng, ntraj, gamma, p_eq, q_eq)
    return Workload(f"uncoupled_morse_F{F}", F, PES_MORSE_UNCOUPLED, coeffs, gamma, dt, nsteps,
                    np.concatenate([p_eq, q_eq]), energy_grid(k), p0q0, seed,
                    dict(omega=omega, mass=mu))
