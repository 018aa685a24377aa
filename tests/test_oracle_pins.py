"""Pins for the CPU oracle (oracle/): what the paper and the mathematics fix, P0..P12 of DESIGN.md.

None of these retype the oracle's formulas: each compares it with a closed form, an invariant,
a library routine, a finite-difference derivative of its own lower-level output, or the
independent brute-force restatement in oracle/brute.py.
"""
import os

import numpy as np
import pytest

from oracle import brute
from paper_1312_4698_b200 import inputs

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _prop(oracle, w, nsteps=None, p0q0=None, **kw):
    return oracle.propagate(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps if nsteps is None else nsteps,
                            w.p0q0 if p0q0 is None else p0q0, w.chi, **kw)


# ------------------------------------------------------------------ P0 initial values
def test_p0_initial_values(oracle):
    """c = 0: M = I => K = I, D = 1, u = 1, S = 0, z_0 = <chi|p0 q0>; started at chi, z_0 = 1."""
    w = inputs.make_config(2, ntraj=3, nsteps=0, k=4)
    p0q0 = w.p0q0.copy()
    p0q0[:, 0] = w.chi  # chi = p_eq then q_eq, same order as the SoA rows
    o = _prop(oracle, w, nsteps=0, p0q0=p0q0, want_z=True)
    assert np.allclose(o["S"], 0) and np.allclose(o["theta"], 0)
    eye = np.eye(w.F)
    for j in range(3):
        assert np.array_equal(o["M"][0, :, :, j], eye) and np.array_equal(o["M"][3, :, :, j], eye)
        assert not o["M"][1, :, :, j].any() and not o["M"][2, :, :, j].any()
    assert abs(o["z"][0, 0] - 1.0) < 1e-15
    assert np.all(np.abs(o["z"][1:, 0]) < 1.0)


# ------------------------------------------------------------------ a6 overlap vs quadrature of Eq. 3
def test_overlap_against_quadrature_of_eq3(oracle):
    """z_0 = <chi|p q> must equal the integral over x of conj(<x|p_eq q_eq>) <x|p q> with the
    coherent states of Eq. 3, per-mode normalisation (gamma/pi)^(1/4) (R1)."""
    F = 2
    gamma = np.array([0.7, 2.3])
    chi = np.array([0.4, -0.9, 0.3, 1.1])  # p_eq, q_eq
    pq = np.array([[-0.2], [1.3], [0.9], [0.5]])  # p1 p2 q1 q2
    coeffs = np.concatenate([np.sqrt(gamma), np.zeros(inputs.n_cubic(F) + inputs.n_quartic(F))])
    o = oracle.propagate(F, inputs.PES_QFF, coeffs, gamma, 1.0, 0, pq, chi, want_z=True)
    x = np.linspace(-12, 12, 48001)
    val = 1.0 + 0j
    for k in range(F):
        def cs(p, q):
            return (gamma[k] / np.pi) ** 0.25 * np.exp(-0.5 * gamma[k] * (x - q) ** 2 + 1j * p * (x - q))
        f = np.conj(cs(chi[k], chi[F + k])) * cs(pq[k, 0], pq[F + k, 0])
        val *= np.sum(f) * (x[1] - x[0])
    assert abs(o["z"][0, 0] - val) < 1e-12


# ------------------------------------------------------------------ P1 PES derivatives
def _five_point(f, x, h):
    return (f(x - 2 * h) - 8 * f(x - h) + 8 * f(x + h) - f(x + 2 * h)) / (12 * h)


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_p1_qff_gradient_hessian_vs_differences_and_definition(oracle, cfg):
    w = inputs.make_config(cfg, ntraj=4, nsteps=1, k=4)
    F = w.F
    q = w.p0q0[F:, :] * 3.0  # well into the anharmonic region
    V, g, H = oracle.eval_pes(F, w.pes_kind, w.pes_coeffs, q)
    # (a) against the unrestricted tensor-sum definition (library einsum over full tensors)
    pes = brute.QFF(F, w.pes_coeffs)
    for j in range(q.shape[1]):
        assert abs(V[j] - pes.V(q[:, j])) <= 1e-13 * abs(V[j])
        assert np.allclose(g[:, j], pes.grad(q[:, j]), rtol=1e-12, atol=1e-18)
        assert np.allclose(H[:, :, j], pes.hess(q[:, j]), rtol=1e-12, atol=1e-18)
        assert np.array_equal(H[:, :, j], H[:, :, j].T) or np.allclose(H[:, :, j], H[:, :, j].T, rtol=1e-14)
    # (b) g and H against 5-point differences of the oracle's own V and g (exact for quartics)
    j = 1
    h = 0.5
    for a in range(F):
        e = np.zeros((F, 1)); e[a] = 1.0
        fV = lambda x: oracle.eval_pes(F, w.pes_kind, w.pes_coeffs, q[:, j:j + 1] + (x) * e)[0][0]
        assert abs(_five_point(fV, 0.0, h) - g[a, j]) <= 1e-10 * np.abs(g[:, j]).max()
        fg = lambda x: oracle.eval_pes(F, w.pes_kind, w.pes_coeffs, q[:, j:j + 1] + (x) * e)[1][:, 0]
        assert np.allclose(_five_point(fg, 0.0, h), H[:, a, j], rtol=0, atol=1e-10 * np.abs(H[:, :, j]).max())


def test_p1_morse_derivatives(oracle):
    w = inputs.make_config(1, ntraj=8, nsteps=1, k=4)
    q = w.p0q0[1:, :]
    V, g, H = oracle.eval_pes(1, w.pes_kind, w.pes_coeffs, q)
    D, a, qe, mu = w.pes_coeffs
    assert np.allclose(V, D * (1 - np.exp(-a * (q[0] - qe))) ** 2, rtol=1e-14)
    h = 1e-4
    fV = lambda x: oracle.eval_pes(1, w.pes_kind, w.pes_coeffs, q + x)[0]
    fg = lambda x: oracle.eval_pes(1, w.pes_kind, w.pes_coeffs, q + x)[1][0]
    assert np.allclose(_five_point(fV, 0.0, h), g[0], rtol=1e-9)
    assert np.allclose(_five_point(fg, 0.0, h), H[0, 0], rtol=1e-9)
    # harmonic limit at the minimum: V'' = 2 D a^2 = mu w^2
    Vm, gm, Hm = oracle.eval_pes(1, w.pes_kind, w.pes_coeffs, np.array([[qe]]))
    assert Vm[0] == 0 and gm[0, 0] == 0 and abs(Hm[0, 0, 0] - mu * w.meta["omega"][0] ** 2) < 1e-15


# ------------------------------------------------------------------ P2 monodromy = derivative of the flow
@pytest.mark.parametrize("cfg,integ", [(2, 0), (3, 0), (2, 1)])
def test_p2_monodromy_is_jacobian_of_the_map(oracle, cfg, integ):
    w = inputs.make_config(cfg, ntraj=1, nsteps=60, k=4)
    F = w.F
    base = _prop(oracle, w, integrator=integ)
    J = np.zeros((2 * F, 2 * F))  # d(p_t,q_t)/d(p_0,q_0), (p,q) order
    scale = np.concatenate([np.sqrt(w.gamma), 1 / np.sqrt(w.gamma)])
    for col in range(2 * F):
        h = 1e-4 * scale[col]
        outs = []
        for sgn in (-2, -1, 1, 2):
            x = w.p0q0.copy(); x[col, 0] += sgn * h
            outs.append(_prop(oracle, w, p0q0=x, integrator=integ)["pq"][:, 0])
        J[:, col] = (outs[0] - 8 * outs[1] + 8 * outs[2] - outs[3]) / (12 * h)
    M = base["M"][..., 0]
    Mfull = np.block([[M[0], M[1]], [M[2], M[3]]])
    # compare in reduced units (all blocks O(1))
    S = np.diag(1 / scale)
    assert np.abs(S @ (Mfull - J) @ np.linalg.inv(S)).max() < 5e-9


# ------------------------------------------------------------------ P3 symplecticity
@pytest.mark.parametrize("cfg,nsteps", [(1, 3000), (2, 1000), (3, 1000), (4, 1000)])
def test_p3_det_one_and_symplectic_condition(oracle, cfg, nsteps):
    w = inputs.make_config(cfg, ntraj=8, nsteps=nsteps, k=4)
    F = w.F
    o = _prop(oracle, w)
    J = np.block([[np.zeros((F, F)), np.eye(F)], [-np.eye(F), np.zeros((F, F))]])
    s = np.concatenate([1 / np.sqrt(w.gamma), np.sqrt(w.gamma)])  # reduced units: p/sqrt(g), q*sqrt(g)
    for j in range(8):
        M = o["M"][..., j]
        Mfull = np.block([[M[0], M[1]], [M[2], M[3]]])
        Mr = np.diag(s) @ Mfull @ np.diag(1 / s)
        if cfg == 1 and np.abs(Mr).max() > 1e3:
            continue  # dissociating Morse trajectory: M grows linearly, conditioning lost (R14)
        assert abs(np.linalg.det(Mr) - 1) < 1e-10
        assert np.abs(Mr.T @ J @ Mr - J).max() < 1e-10 * max(1.0, np.abs(Mr).max() ** 2)
    assert o["good"].all()


# ------------------------------------------------------------------ P4 energy drift
def test_p4_energy_drift_bounded_and_second_order(oracle):
    w = inputs.make_config(2, ntraj=4, nsteps=2000, k=4)
    F = w.F

    def energy(pq):
        V = oracle.eval_pes(F, w.pes_kind, w.pes_coeffs, pq[F:])[0]
        return 0.5 * np.sum(pq[:F] ** 2, axis=0) + V

    E0 = energy(w.p0q0)
    drifts = {}
    for dt, ns in ((10.0, (500, 1000, 1500, 2000)), (5.0, (1000, 2000, 3000, 4000))):
        d = 0.0
        for n in ns:
            o = oracle.propagate(F, w.pes_kind, w.pes_coeffs, w.gamma, dt, n, w.p0q0, w.chi, want_M=False)
            d = max(d, np.max(np.abs(energy(o["pq"]) - E0) / E0))
        drifts[dt] = d
    assert drifts[10.0] < 0.02  # bounded, no secular growth (O((w dt)^2))
    assert drifts[5.0] < 0.4 * drifts[10.0]  # ~ x4 smaller at half the step


def test_fourth_order_scheme_converges_at_order_four(oracle):
    w = inputs.make_config(2, ntraj=2, nsteps=1, k=4)
    T = 400.0
    ref = oracle.propagate(w.F, w.pes_kind, w.pes_coeffs, w.gamma, 0.25, 1600, w.p0q0, w.chi, integrator=1)["pq"]
    errs = []
    for dt in (10.0, 5.0):
        o = oracle.propagate(w.F, w.pes_kind, w.pes_coeffs, w.gamma, dt, int(T / dt), w.p0q0, w.chi, integrator=1)
        errs.append(np.abs(o["pq"] - ref).max())
    order = np.log2(errs[0] / errs[1])
    assert 3.6 < order < 4.5


# ------------------------------------------------------------------ P5 discrete action identity
@pytest.mark.parametrize("integ", [0, 1])
def test_p5_action_is_generating_function(oracle, integ):
    """dS_N/dq_0 = M_qq^T p_N - p_0 and dS_N/dp_0 = M_qp^T p_N (R11), S by differences."""
    w = inputs.make_config(2, ntraj=1, nsteps=40, k=4)
    F = w.F
    base = _prop(oracle, w, integrator=integ)
    pN = base["pq"][:F, 0]
    M = base["M"][..., 0]
    rhs_q = M[3].T @ pN - w.p0q0[:F, 0]
    rhs_p = M[2].T @ pN
    scale = np.concatenate([np.sqrt(w.gamma), 1 / np.sqrt(w.gamma)])
    dS = np.zeros(2 * F)
    for col in range(2 * F):
        h = 1e-3 * scale[col]
        vals = []
        for sgn in (-2, -1, 1, 2):
            x = w.p0q0.copy(); x[col, 0] += sgn * h
            vals.append(_prop(oracle, w, p0q0=x, integrator=integ)["S"][0])
        dS[col] = (vals[0] - 8 * vals[1] + 8 * vals[2] - vals[3]) / (12 * h)
    assert np.allclose(dS[F:] * scale[F:], rhs_q * scale[F:], atol=2e-9)
    assert np.allclose(dS[:F] * scale[:F], rhs_p * scale[:F], atol=2e-9)


# ------------------------------------------------------------------ P6 / P6a harmonic closed form
def _read_golden(name):
    d = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        d[k] = float(v)
    return d


def test_p6a_worked_example_closed_form(oracle):
    """tests/golden/harmonic_1d.txt (closed form, 40-digit arithmetic).  Velocity-Verlet converges to
    it as dt^2; at dt = 1e-3 the residual is ~1e-7 and shrinks x4 per halving."""
    gd = _read_golden("harmonic_1d.txt")
    w0 = gd["omega"]
    coeffs = np.array([w0, 0.0, 0.0])
    # the QFF kind has its minimum at q = 0: shift coordinates by q_eq (translation invariance)
    chi = np.array([gd["p_eq"], 0.0])
    pq = np.array([[gd["p0"]], [gd["q0"] - gd["q_eq"]]])
    errs = []
    for dt in (2e-3, 1e-3):
        n = int(round(gd["t"] / dt))
        o = oracle.propagate(1, inputs.PES_QFF, coeffs, np.array([w0]), dt, n, pq, chi, want_z=True)
        got = dict(p_t=o["pq"][0, 0], q_t=o["pq"][1, 0] + gd["q_eq"], S_t=o["S"][0], M_pp=o["M"][0, 0, 0, 0],
                   M_pq=o["M"][1, 0, 0, 0], M_qp=o["M"][2, 0, 0, 0], M_qq=o["M"][3, 0, 0, 0],
                   theta_t=o["theta"][0], z_re=o["z"][0, -1].real, z_im=o["z"][0, -1].imag)
        errs.append(max(abs(got[k] - gd[k]) for k in got))
    assert errs[1] < 3e-6
    assert 3.5 < errs[0] / errs[1] < 4.5


def test_p6_harmonic_exact_rotation_with_verlet_frequency(oracle):
    """Velocity-Verlet on a harmonic mode IS an exact rotation at the shifted frequency
    wt = arccos(1 - (w dt)^2/2)/dt.  In the variables (q, p_half-step-centred) it closes exactly; here we
    check what needs no re-centring: q_c = A cos(wt c dt) + B sin(wt c dt) to round-off, the action
    identity S_N = (p_N q_N - p_0 q_0)/2 ... + O(dt^2), and the prefactor phase -wt t/2 to O(dt^2)."""
    w0, dt, n = 0.0179, 10.0, 3000
    wt = np.arccos(1 - (w0 * dt) ** 2 / 2) / dt
    coeffs = np.array([w0, 0.0, 0.0])
    pq = np.array([[0.11], [3.1]])
    chi = np.array([np.sqrt(w0), 0.0])
    qs = []
    for m in (0, 1, 2, 1500, n):
        o = oracle.propagate(1, inputs.PES_QFF, coeffs, np.array([w0]), dt, m, pq, chi)
        qs.append(o["pq"][1, 0])
    # three-term recurrence of an exact rotation: q_{c+1} + q_{c-1} = 2 cos(wt dt) q_c
    assert abs(qs[2] + qs[0] - 2 * np.cos(wt * dt) * qs[1]) < 1e-14 * abs(qs[1])
    A = qs[0]
    B = (qs[1] - A * np.cos(wt * dt)) / np.sin(wt * dt)
    for m, qv in ((1500, qs[3]), (n, qs[4])):
        assert abs(qv - (A * np.cos(wt * m * dt) + B * np.sin(wt * m * dt))) < 1e-10 * abs(A)
    o = oracle.propagate(1, inputs.PES_QFF, coeffs, np.array([w0]), dt, n, pq, chi)
    # continuous branch: theta = arg det K unwrapped = -wt T up to the O((w dt)^2) wobble of |K| != 1
    assert abs(o["theta"][0] - (-wt * n * dt)) < 0.05
    assert abs(o["theta"][0]) > 80 * 2 * np.pi  # ~ 85 turns: the branch was tracked, not wrapped


# ------------------------------------------------------------------ P7 harmonic spectrum (north-star pin)
def test_p7_harmonic_spectrum_peaks_at_sum_n_plus_half_omega(oracle):
    """Purely harmonic PES, gamma = omega: peaks of I(E) at sum_k (n_k + 1/2) wt_k, wt the frequency
    velocity-Verlet produces (-> hbar w as dt -> 0).  dt = 1 a.u. makes wt - w < 0.06 cm^-1."""
    cm = inputs.CM1_PER_HARTREE
    om = np.array([1600.0, 3700.0]) / cm
    dt, n = 4.0, 8000
    E = np.linspace(0, 12000, 2401) / cm  # 5 cm^-1 bins
    w = inputs.make_harmonic(om, ntraj=96, nsteps=n, dt=dt, E=E, seed=3)
    I, ng, rc = oracle.run_workload(w)
    assert rc == 0 and ng == 96 and I.min() >= 0
    wt = np.arccos(1 - (om * dt) ** 2 / 2) / dt
    bin_w = E[1] - E[0]
    # expected levels inside the window with non-negligible weight
    levels = sorted((n0 + .5) * wt[0] + (n1 + .5) * wt[1] for n0 in range(4) for n1 in range(3))
    levels = [e for e in levels if e < E[-1] - 10 * bin_w]
    # main peaks: strict local maxima above 6 % of max.  The finite-T window gives every line Dirichlet
    # side lobes at -/+1.43 * 2 pi / T of height 4.7 % of that line; they are not levels and sit below 6 %.
    pk = oracle.find_peaks(I, rel_height=0.06)
    found = E[pk]
    zpe = 0.5 * wt.sum()
    assert abs(E[np.argmax(I)] - zpe) <= bin_w  # strongest line = zero-point level (chi is the ground state)
    for e in found:
        assert min(abs(e - l) for l in levels) <= 1.01 * bin_w, (e * cm, [l * cm for l in levels])
    # the zero-point level, both fundamentals and the combination level must be among them ...
    for l in (zpe, zpe + wt[0], zpe + wt[1], zpe + wt[0] + wt[1]):
        assert min(abs(found - l)) <= 1.01 * bin_w
    # ... and the weaker overtones are local maxima too (Husimi sampling with unit weights, R7, damps
    # the intensity of excited levels but does not move them)
    weak = E[oracle.find_peaks(I, rel_height=1e-3)]
    for l in (zpe + 2 * wt[0], zpe + 2 * wt[1], zpe + 2 * wt[0] + wt[1]):
        assert min(abs(weak - l)) <= 1.01 * bin_w


# ------------------------------------------------------------------ P8 Herman-Kluk matrix, non-uniform Gamma
def test_p8_prefactor_matches_reduced_coordinate_form(oracle):
    """theta from the oracle (raw M, Gamma; Eq. 5 read as R2) equals arg det of the unambiguous form in
    reduced coordinates, K~ = 1/2 (M~qq + M~pp - i M~qp + i M~pq), M~ = S M S^-1, S = diag(g^-1/2, g^1/2),
    computed here with numpy.linalg.det; the literal one-sided reading of Eq. 5 does NOT."""
    w = inputs.make_config(3, ntraj=6, nsteps=300, k=4)
    F = w.F
    gamma = w.gamma * np.array([0.5, 2.0, 1.0, 3.0, 0.7, 1.6])  # deliberately not the frequencies
    o = oracle.propagate(F, w.pes_kind, w.pes_coeffs, gamma, w.dt, w.nsteps, w.p0q0, w.chi)
    n_discriminated = 0
    for j in range(6):
        M = o["M"][..., j]
        Mfull = np.block([[M[0], M[1]], [M[2], M[3]]])
        S = np.diag(np.concatenate([gamma ** -0.5, gamma ** 0.5]))
        Mt = S @ Mfull @ np.linalg.inv(S)
        Kt = 0.5 * (Mt[F:, F:] + Mt[:F, :F] - 1j * Mt[F:, :F] + 1j * Mt[:F, F:])
        d = np.linalg.det(Kt)
        assert abs(np.exp(1j * o["theta"][j]) - d / abs(d)) < 1e-10
        G = np.diag(gamma)
        Klit = 0.5 * (M[3] + M[0] - 1j * G @ M[2] + 1j * np.linalg.inv(G) @ M[1])
        dl = np.linalg.det(Klit)
        n_discriminated += abs(dl / abs(dl) - d / abs(d)) > 1e-3
    assert n_discriminated >= 4  # the test can tell the two readings apart


# ------------------------------------------------------------------ P9 separability
def test_p9_uncoupled_modes_factorise(oracle):
    F = 3
    w = inputs.make_uncoupled_morse(F, ntraj=5, nsteps=250, k=4)
    o = _prop(oracle, w, want_z=True)
    prod = np.ones_like(o["z"])
    Ssum = np.zeros(5)
    for k in range(F):
        c1 = w.pes_coeffs.reshape(F, 4)[k]
        o1 = oracle.propagate(1, inputs.PES_MORSE1D, c1, w.gamma[k:k + 1], w.dt, w.nsteps,
                              w.p0q0[[k, F + k]], w.chi[[k, F + k]], want_z=True)
        prod *= o1["z"]
        Ssum += o1["S"]
        assert np.allclose(o["M"][3, k, k], o1["M"][3, 0, 0], rtol=1e-12)
    assert np.abs(o["z"] - prod).max() < 1e-12
    assert np.allclose(o["S"], Ssum, rtol=1e-12)
    # off-diagonal monodromy blocks stay exactly zero
    for blk in range(4):
        for a in range(F):
            for b in range(F):
                if a != b:
                    assert not o["M"][blk, a, b].any()


def test_p9_qff_without_couplings_factorises(oracle):
    om = np.array([1500.0, 2900.0, 3300.0]) / inputs.CM1_PER_HARTREE
    E = inputs.energy_grid(4)
    w = inputs.make_harmonic(om, ntraj=4, nsteps=300, dt=10.0, E=E)
    o = _prop(oracle, w, want_z=True)
    prod = np.ones_like(o["z"])
    for k in range(3):
        c1 = np.array([om[k], 0.0, 0.0])
        o1 = oracle.propagate(1, inputs.PES_QFF, c1, om[k:k + 1], w.dt, w.nsteps, w.p0q0[[k, 3 + k]],
                              w.chi[[k, 3 + k]], want_z=True)
        prod *= o1["z"]
    assert np.abs(o["z"] - prod).max() < 1e-12


# ------------------------------------------------------------------ P10 Fourier stage vs library FFT
def test_p10_fourier_equals_ifft_on_the_dft_grid_and_parseval(oracle):
    rng = np.random.default_rng(5)
    N, dt = 512, 7.0
    z = rng.standard_normal((3, N)) + 1j * rng.standard_normal((3, N))
    E = 2 * np.pi * np.arange(N) / (N * dt)
    for mode in (0, 1):
        A = oracle.fourier(z, dt, E, mode=mode)
        ref = N * np.fft.ifft(z, axis=1)
        assert np.abs(A - ref).max() < 1e-10
        assert np.allclose(np.sum(np.abs(A) ** 2, axis=1), N * np.sum(np.abs(z) ** 2, axis=1), rtol=1e-12)


def test_p10_recurrence_twiddles_match_definition(oracle):
    rng = np.random.default_rng(6)
    N, dt = 1200, 10.0
    z = rng.standard_normal((2, N)) + 1j * rng.standard_normal((2, N))
    E = inputs.energy_grid(97)
    A0 = oracle.fourier(z, dt, E, mode=0)
    A1 = oracle.fourier(z, dt, E, mode=1)
    assert np.abs(A1 - A0).max() < 1e-12 * np.abs(A0).max()
    # and the definition itself against numpy
    ref = z @ np.exp(1j * np.outer(np.arange(N) * dt, E))
    assert np.abs(A0 - ref).max() < 1e-10 * np.abs(ref).max()


# ------------------------------------------------------------------ brute force on tiny inputs (whole path)
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_brute_force_whole_path_tiny(oracle, cfg):
    w = inputs.make_config(cfg, ntraj=3, nsteps=150, k=64)
    o = _prop(oracle, w, want_z=True)
    pes = brute.make_pes(w.F, w.pes_kind, w.pes_coeffs)
    for j in range(3):
        t = brute.trajectory(pes, w.gamma, w.dt, w.nsteps, w.p0q0[:w.F, j], w.p0q0[w.F:, j], w.chi)
        assert np.abs(o["z"][j] - t["z"]).max() < 1e-12
        assert abs(o["theta"][j] - 2 * t["phi"][-1]) < 1e-10
        assert abs(o["S"][j] - t["S"][-1]) < 1e-12 * max(1, abs(t["S"][-1]))
        Mfull = np.block([[o["M"][0, :, :, j], o["M"][1, :, :, j]], [o["M"][2, :, :, j], o["M"][3, :, :, j]]])
        assert np.allclose(Mfull, t["M"][-1], rtol=1e-11, atol=1e-13 * np.abs(Mfull).max())
    for mode in (0, 1):
        I, ng, rc = oracle.run_workload(w, fourier_mode=mode)
        Ib, ngb, _ = brute.spectrum(pes, w.gamma, w.dt, w.nsteps, w.p0q0, w.chi, w.E)
        assert ng == ngb == 3 and rc == 0
        assert np.abs(I - Ib).max() < 1e-12 * Ib.max()


def test_brute_force_fourth_order_scheme(oracle):
    w = inputs.make_config(2, ntraj=2, nsteps=40, k=8)
    o = _prop(oracle, w, want_z=True, integrator=1)
    pes = brute.make_pes(w.F, w.pes_kind, w.pes_coeffs)
    t = brute.trajectory(pes, w.gamma, w.dt, w.nsteps, w.p0q0[:w.F, 1], w.p0q0[w.F:, 1], w.chi,
                         scheme=brute.MCLACHLAN_ATELA_4)
    assert np.abs(o["z"][1] - t["z"]).max() < 1e-12


# ------------------------------------------------------------------ P11 reduction properties
def test_p11_positive_permutation_invariant_and_poison(oracle):
    w = inputs.make_config(2, ntraj=24, nsteps=300, k=200)
    I, ng, rc = oracle.run_workload(w, fourier_mode=0)
    assert rc == 0 and ng == 24 and I.min() >= 0.0  # Eq. 10 integrand is positive-definite
    perm = np.random.default_rng(1).permutation(24)
    Ip, _, _ = oracle.run(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, w.p0q0[:, perm], w.chi, w.E,
                          fourier_mode=0)
    assert np.abs(I - Ip).max() < 1e-13 * I.max()
    bad = w.p0q0.copy(); bad[0, 7] = np.nan
    Ib, ngb, rcb = oracle.run(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, bad, w.chi, w.E, fourier_mode=0)
    keep = [j for j in range(24) if j != 7]
    Ik, ngk, _ = oracle.run(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, w.p0q0[:, keep], w.chi, w.E,
                            fourier_mode=0)
    assert ngb == 23 and ngk == 23 and rcb == 0
    assert np.abs(Ib - Ik).max() < 1e-13 * Ik.max()
    # weights: w_j = 2 doubles the spectrum; w_j = 0 on one trajectory removes its term but not its count
    wts = np.full(24, 2.0)
    I2, _, _ = oracle.run(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, w.p0q0, w.chi, w.E, weights=wts,
                          fourier_mode=0)
    assert np.allclose(I2, 2 * I, rtol=1e-13)


def test_rejection_path_and_no_good_trajectories(oracle):
    w = inputs.make_config(2, ntraj=4, nsteps=200, k=16)
    # an absurdly tight tolerance rejects everything: zero spectrum, ENOGOOD (R18)
    I, ng, rc = oracle.run(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, w.p0q0, w.chi, w.E, det_tol=1e-18)
    assert ng == 0 and rc == 5 and not I.any()
    o = _prop(oracle, w, det_tol=1e-18)
    assert not o["good"].any()
    # det_stride only changes WHEN the check runs, not the result on healthy trajectories
    I1, n1, _ = oracle.run_workload(w)
    I2, n2, _ = oracle.run_workload(w, det_stride=w.nsteps)
    assert n1 == n2 == 4 and np.array_equal(I1, I2)


# ------------------------------------------------------------------ P12 config 1 sanity (loose)
def test_p12_morse_levels_loose(oracle):
    w = inputs.make_config(1, ntraj=256)
    I, ng, rc = oracle.run_workload(w)
    assert rc == 0 and ng == 256
    D = w.pes_coeffs[0]
    om = w.meta["omega"][0]
    cm = inputs.CM1_PER_HARTREE
    lev = [(om * (n + .5) - (om * (n + .5)) ** 2 / (4 * D)) * cm for n in range(3)]
    assert abs(lev[0] - 2150.0) < 0.5 and abs(lev[1] - 6263.7) < 0.5  # the textbook Morse term values
    Ecm = w.E * cm
    bin_w = Ecm[1] - Ecm[0]
    pk = oracle.find_peaks(I, rel_height=1e-3)  # n = 2 carries ~1 % of the n = 0 intensity
    for l in lev:
        assert min(abs(Ecm[pk] - l)) <= 3 * bin_w
    assert abs(Ecm[np.argmax(I)] - lev[0]) <= 3 * bin_w


def _line_check(spec_single, spec_combo, factors, om, T, dE, nlines):
    """Lines of a harmonic spectrum under a rectangular window of length T ("leakage bound"): a line m
    of power P_m puts at most sqrt(P_m) / ((N + 1) |sin((E_n - E_m) dt / 2)|) <= sqrt(P_m) 2 / (|n - m| om T) of
    amplitude (Dirichlet kernel) under the line n.  With combination factors f_m on the single-state powers P1_m,
    the amplitude under line n is sqrt(f_n P1_n) up to the sum of those side lobes; no tuned constants."""
    idx = [int(round((n + 0.5) * om / dE)) for n in range(nlines)]
    P1 = np.array([spec_single[i] for i in idx])
    for n in range(nlines):
        leak = sum(np.sqrt(factors[m] * P1[m]) * 2.0 / (abs(n - m) * om * T) for m in range(nlines) if m != n)
        leak += np.sqrt(P1[n]) * sum(2.0 / (abs(n - m) * om * T) for m in range(nlines) if m != n)  # P1_n itself carries side lobes
        leak *= 1.05                                                                                # lines above the grid (Poisson tail)
        got, want = np.sqrt(spec_combo[idx[n]]), np.sqrt(factors[n] * P1[n])
        assert abs(got - want) <= leak, (n, got, want, leak)
        if factors[n] == 0.0 and P1[n] > 1e-3 * P1.max():
            assert spec_combo[idx[n]] < 0.02 * P1[n]  # the bound is not vacuous: the line is gone


def test_combo_reference_state_parity_selection_rule(oracle):
    """Row f4 (Fig. 4): reference state = combination of coherent states.  Closed-form pin: for a
    1-D harmonic oscillator with gamma = omega, |alpha> + |-alpha> contains only even and |alpha> - |-alpha> only odd
    number states (the mirror image about q_eq), so each combination keeps every second peak of the single-state
    spectrum, at (n + 1/2) omega~, with four times its power, and removes the others."""
    om = 0.01
    nsteps, dt = 6000, 2.0  # omega dt = 0.02: the Verlet map is harmonic with omega~ = omega (1 + 1.7e-5)
    E = np.linspace(0.0, 6.0 * om, 601)
    w = inputs.make_harmonic([om], ntraj=24, nsteps=nsteps, dt=dt, E=E, seed=3)
    p_e, q_e = w.chi[0], w.chi[1]
    chis = np.array([[p_e, q_e], [-p_e, -q_e]])  # make_harmonic puts q_eq = 0 unless told otherwise
    assert abs(q_e) < 1e-15
    spec = {}
    for name, eps in (("single", [1.0, 0.0]), ("even", [1.0, 1.0]), ("odd", [1.0, -1.0])):
        spec[name], ng, rc = oracle.run_combo(1, w.pes_kind, w.pes_coeffs, w.gamma, dt, nsteps, w.p0q0, chis, eps, E,
                                              fourier_mode=0)
        assert (ng, rc) == (24, 0)
    I1, rc1 = oracle.run(1, w.pes_kind, w.pes_coeffs, w.gamma, dt, nsteps, w.p0q0, w.chi, E, fourier_mode=0)[::2]
    assert np.allclose(spec["single"], I1, rtol=1e-12, atol=0)  # eps = (1, 0) is the plain reference state
    # <n|-alpha> = (-1)^n <n|alpha>: |1 + eps (-1)^n|^2
    _line_check(spec["single"], spec["even"], [4.0, 0.0, 4.0, 0.0, 4.0, 0.0], om, nsteps * dt, E[1] - E[0], 6)
    _line_check(spec["single"], spec["odd"], [0.0, 4.0, 0.0, 4.0, 0.0, 4.0], om, nsteps * dt, E[1] - E[0], 6)


def test_combo_reference_state_conjugation(oracle):
    """The conjugate in <chi| = sum_m conj(eps_m) <p_m q_m| (reference_overlap in the oracle), pinned by a
    closed form that a slip eps <-> conj(eps) breaks.  1-D harmonic oscillator, gamma = omega, q_eq = 0; coherent states
    m = 0: (p_e, 0), i.e. alpha = i p_e / sqrt(2 gamma), and m = 1: (0, -p_e / gamma), i.e. alpha' = i alpha (both have
    p (q - q_eq) = 0, so Eq. 3's state is the Glauber state without an extra phase).  Number-state amplitudes:
    <n|alpha'> = i^n <n|alpha>, so |chi> = |alpha> + eps |alpha'> carries |1 + eps i^n|^2 times the single-state power of
    line n: for eps = +i that is (2, 0, 2, 4, 2, 0), for eps = -i it is (2, 4, 2, 0, 2, 4).  With the conjugate dropped the
    two lists swap: line 1 would survive with four times its power where it must vanish."""
    om = 0.01
    nsteps, dt = 6000, 2.0
    E = np.linspace(0.0, 6.0 * om, 601)
    w = inputs.make_harmonic([om], ntraj=24, nsteps=nsteps, dt=dt, E=E, seed=3)
    p_e, q_e, g = w.chi[0], w.chi[1], w.gamma[0]
    assert abs(q_e) < 1e-15 and abs(g - om) < 1e-15
    chis = np.array([[p_e, 0.0], [0.0, -p_e / g]])
    spec = {}
    for name, eps in (("single", np.array([1.0, 0.0], dtype=complex)), ("plus_i", np.array([1.0, 1.0j])), ("minus_i", np.array([1.0, -1.0j]))):
        spec[name], ng, rc = oracle.run_combo(1, w.pes_kind, w.pes_coeffs, w.gamma, dt, nsteps, w.p0q0, chis, eps, E, fourier_mode=0)
        assert (ng, rc) == (24, 0)
    fac = {"plus_i": [abs(1 + 1j * 1j ** n) ** 2 for n in range(6)], "minus_i": [abs(1 - 1j * 1j ** n) ** 2 for n in range(6)]}
    assert np.allclose(fac["plus_i"], [2, 0, 2, 4, 2, 0]) and np.allclose(fac["minus_i"], [2, 4, 2, 0, 2, 4])
    for name in ("plus_i", "minus_i"):
        _line_check(spec["single"], spec[name], [round(f) * 1.0 for f in fac[name]], om, nsteps * dt, E[1] - E[0], 6)


def test_combo_reference_state_brute_force(oracle):
    """The C oracle against the numpy restatement on a tiny coupled case with complex coefficients and three states."""
    from oracle import brute
    w = inputs.make_random_qff(2, 5, 60, 24, seed=21)
    rng = np.random.default_rng(5)
    chis = np.stack([w.chi, w.chi * np.array([-1, 1, -1, 1]), w.chi + 0.1 * rng.standard_normal(4)])
    eps = np.array([1.0, -0.5 + 0.25j, 0.3j])
    I, ng, rc = oracle.run_combo(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, w.nsteps, w.p0q0, chis, eps, w.E, fourier_mode=0)
    pes = brute.make_pes(w.F, w.pes_kind, w.pes_coeffs)
    Ib, ngb = brute.spectrum_combo(pes, w.gamma, w.dt, w.nsteps, w.p0q0, chis, eps, w.E)
    assert ng == ngb == 5 and rc == 0
    assert np.max(np.abs(I - Ib)) < 1e-11 * Ib.max()


def test_r22_flag_is_decided_by_roundoff(oracle):
    """Reading R22: tests/golden/r22_flag.txt holds, for trajectory 105793 of config 5, the determinant of
    the oracle's own monodromy matrix evaluated in 60-digit arithmetic (make_r22_flag.py).  The exact map has det M = 1
    (PAPER.md:64), so what the file lists is accumulated round-off: negligible while eps max|M|^2 << det_tol, of the size of
    det_tol = 1e-6 once max|M| >= 1e6.  That is the regime in which the GPU parity test lets at most two flags
    differ.  The file is tied to the oracle as it stands: max|M| and the flag are recomputed here."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "r22_flag.txt")
    rows = np.array([[float(x) for x in ln.split()] for ln in open(path) if not ln.startswith("#")])
    assert rows.shape[1] == 6 and rows[-1, 0] == 8000
    nsteps, good, mmax, dev_exact, dev_f64, bound = rows.T
    tol = 1e-6
    early = bound < 1e-1 * tol                       # the flag is a property of the trajectory: far inside the tolerance, accepted
    assert early.sum() >= 2 and np.all(dev_exact[early] < 1e-3 * tol) and np.all(good[early] == 1)
    late = mmax >= 1e6                               # the flag is round-off: deviation within a factor 30 of the tolerance either way
    assert late.sum() >= 3 and np.all(bound[late] > 100 * tol)
    assert np.all((dev_exact[late] > tol / 30) & (dev_exact[late] < tol * 30))
    assert dev_exact[late].min() < tol < dev_exact[late].max()   # both sides of it along one trajectory
    assert np.all(good[dev_exact > tol] == 0)        # the oracle rejects where the determinant of ITS M is outside (rightly)
    assert np.all(np.abs(dev_f64 - dev_exact) <= 1e3 * bound)    # and a double-precision determinant of that M is no better than eps max|M|^2
    # the same trajectory through today's oracle
    w = inputs.make_config(5, ntraj=1 << 17, nsteps=8000)
    pq = np.ascontiguousarray(w.p0q0[:, 105793:105794])
    for i in (1, len(rows) - 1):
        po = oracle.propagate(w.F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, int(nsteps[i]), pq, want_M=True)
        assert abs(np.abs(po["M"]).max() - mmax[i]) <= 1e-8 * mmax[i]
        assert int(po["good"][0]) == int(good[i])
