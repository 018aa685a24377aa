"""Writes tests/golden/r22_flag.txt: the evidence behind reading R22 of DESIGN.md (section 4).

R22 says: once max|M_ij| of a trajectory reaches ~1e6, the quality flag |det M - 1| <= 1e-6 is decided by
round-off, not by the mathematics, so the CUDA path and the oracle may disagree on it.  The case on record is trajectory 105793
of config 5 (CH4-like surface, 2^17 trajectories) at 8000 steps, which the oracle rejects.  This script

  1. propagates that one trajectory with the ORACLE (oracle/, nothing else) to a few step counts up to 8000,
  2. takes the oracle's own 2F x 2F monodromy matrix M (IEEE doubles, i.e. exact rationals) at each of them,
  3. evaluates det M in 60-digit arithmetic (mpmath LU; M's condition ~1e12 leaves > 40 correct digits), and
  4. writes |det M - 1| exact, the double-precision value numpy.linalg.det gives for the same M, max|M| and eps max|M|^2.

What the table shows.  The exact map is symplectic, det M = 1, so ANY deviation of det M from 1 is round-off accumulated in M
itself, amplified by the stretching: the EXACT determinant of the oracle's M drifts as 2e-14, 2e-12, 3e-9, 3e-7 at 2000, 4000,
6000, 7000 steps (following eps max|M|^2 three to four orders below it), crosses the tolerance 1e-6 near step 7750 (1.3e-6: there
the oracle rejects, rightly for ITS M) and is back at 5.1e-7 at step 8000.  A second implementation whose M differs from the
oracle's in the last digits (6e-10 relative at this point for the CUDA path) has its own drift of the same size, above or
below 1e-6: once max|M| >= 1e6 the flag is not a property of the trajectory.  It calls no CUDA code.

    python tests/golden/make_r22_flag.py
"""
import os
import sys

import mpmath as mp
import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import capi  # noqa: E402
from paper_1312_4698_b200 import inputs  # noqa: E402  (seeded input generators only)

J = 105793
STEPS = [2000, 4000, 6000, 7000, 7500, 7750, 8000]
mp.mp.dps = 60


def main():
    capi.build()
    w = inputs.make_config(5, ntraj=1 << 17, nsteps=8000)
    pq = np.ascontiguousarray(w.p0q0[:, J:J + 1])
    F = w.F
    rows = []
    for n in STEPS:
        po = capi.propagate(F, w.pes_kind, w.pes_coeffs, w.gamma, w.dt, n, pq, want_M=True)
        Mb = po["M"][..., 0]                                     # [4][F][F]: pp, pq, qp, qq
        M = np.block([[Mb[0], Mb[1]], [Mb[2], Mb[3]]])
        exact = mp.det(mp.matrix([[mp.mpf(float(x)) for x in r] for r in M]))
        rows.append((n, int(po["good"][0]), float(np.abs(M).max()), float(abs(exact - 1)), float(abs(np.linalg.det(M) - 1.0)),
                     float(np.finfo(float).eps * np.abs(M).max() ** 2)))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "r22_flag.txt")
    with open(out, "w") as f:
        f.write("# reading R22 (DESIGN.md section 4): trajectory %d of config 5 (2^17 trajectories), oracle's own M, det in 60-digit arithmetic\n" % J)
        f.write("# written by tests/golden/make_r22_flag.py (oracle/ + mpmath only); flag rule: PAPER.md:64, :111\n")
        f.write("# nsteps  oracle_good  max|M|  |det M - 1| exact  |det M - 1| numpy float64  eps*max|M|^2\n")
        for r in rows:
            f.write("%d %d %.9e %.6e %.6e %.6e\n" % r)
    print(open(out).read())


if __name__ == "__main__":
    main()
