"""Writes tests/golden/harmonic_1d.txt: the worked example P6a of DESIGN.md.

The paper prints no worked example, so this one comes from the CLOSED FORM of the 1-D harmonic
oscillator (exact classical rotation, S_t = (p_t q_t - p_0 q_0)/2 in displaced coordinates,
C_t = e^{-i w t / 2} for gamma = m w), evaluated in 40-digit arithmetic with mpmath.  It calls
neither oracle/ nor the CUDA path.  Eq. 3 gives the overlap; Eq. 5
 the prefactor; Eq. 10 the integrand z(t).

V = 1/2 w^2 (q - q_eq)^2, m = 1, w = gamma = 1.3, q_eq = 0.2, p_eq = sqrt(1.3),
(p_0, q_0) = (0.7, -0.4), t = 10.
"""
import os

import mpmath as mp

mp.mp.dps = 40
w = mp.mpf("1.3")
q_eq = mp.mpf("0.2")
p_eq = mp.sqrt(w)
p0, q0, t = mp.mpf("0.7"), mp.mpf("-0.4"), mp.mpf(10)
x0 = q0 - q_eq
c, s = mp.cos(w * t), mp.sin(w * t)
xt = x0 * c + p0 / w * s
pt = p0 * c - w * x0 * s
qt = xt + q_eq
# S = int (p^2/2 - w^2 x^2/2) dt = (p_t x_t - p_0 x_0)/2 for the harmonic oscillator
S = (pt * xt - p0 * x0) / 2
Mqq, Mqp, Mpq, Mpp = c, s / w, -w * s, c
phi = -w * t / 2  # continuous phase of sqrt(det K), K = e^{-i w t}
dq, dp = q_eq - qt, p_eq - pt
ovl = mp.e ** (-w / 4 * dq ** 2 - dp ** 2 / (4 * w)) * mp.e ** (mp.j / 2 * (p_eq + pt) * dq)
z = ovl * mp.e ** (mp.j * (S + phi))
rows = [("omega", w), ("q_eq", q_eq), ("p_eq", p_eq), ("p0", p0), ("q0", q0), ("t", t),
        ("p_t", pt), ("q_t", qt), ("S_t", S), ("M_pp", Mpp), ("M_pq", Mpq), ("M_qp", Mqp), ("M_qq", Mqq),
        ("theta_t", 2 * phi), ("ovl_re", ovl.real), ("ovl_im", ovl.imag), ("z_re", z.real), ("z_im", z.imag)]
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "harmonic_1d.txt")
with open(out, "w") as f:
    f.write("# 1-D harmonic worked example, closed form in 40-digit arithmetic (make_harmonic_golden.py)\n")
    f.write("# cites: Eq. 3 PAPER.md:49-52, Eq. 5 PAPER.md:61, Eq. 10 PAPER.md:88-93\n")
    for k, v in rows:
        f.write(f"{k} {mp.nstr(v, 25)}\n")
print(open(out).read())
