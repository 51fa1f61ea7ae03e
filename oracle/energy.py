"""Demagnetizing energy (oracle, test infrastructure).

PAPER.md:L293 relates a field term to its energy density by
H = -(1/(mu0 Ms)) d(eps)/d(m).  For the (quadratic, self-adjoint) demag term
this integrates to the standard magnetostatic self-energy

    E = -(mu0/2) * sum_cells M(t) . H(t) * dV,      dV = hx hy hz

(reading R13; the 1/2 is the double counting of pairs).  SI units:
M, H in A/m, h in m, E in J, mu0 = 4 pi 1e-7 (reading R8).
"""
import numpy as np

MU0 = 4e-7 * np.pi


def demag_energy(M, H, h):
    M = np.asarray(M, np.float64)
    H = np.asarray(H, np.float64)
    dV = float(h[0]) * float(h[1]) * float(h[2])
    return -0.5 * MU0 * dV * float(np.sum(M * H))
