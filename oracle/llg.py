"""Landau-Lifshitz-Gilbert evaluation around the demag path (oracle, TEST INFRASTRUCTURE: only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg may import this).

Plain fp64 numpy, written from the paper:

* PAPER.md:L33, Eq. (1):  dm/dt = -gamma m x H_eff + alpha m x dm/dt, m the unit magnetization direction,
  gamma = mu0 g_rel |gamma_e| (L36).  Solved for dm/dt (cross the equation with m, use m . dm/dt = 0):
      dm/dt = -gamma / (1 + alpha^2) * [ m x H + alpha m x (m x H) ].
* H_eff = "additive field contributions" (L36): the demagnetizing field (L323; oracle/demag_fft.py), the direct
  exchange field H = 2A / (mu0 Ms) * laplacian(m) with the homogeneous Neumann condition dm/dn = 0 (L306-L308), and
  a uniform applied field (Zeeman term, L36).
* RK4 with a fixed time step (L36, L40: "the RK4 method with a fixed time-step"); m is renormalised after each
  step (reading: the paper does not say; a unit vector field is what Eq. (1) evolves, and fp32 drift must not
  accumulate — the library does the same, so the comparison is like for like).

The Laplacian is the second-order 6-neighbour (4 in 2-D: nz = 1) finite difference on the cell centres; the Neumann
condition mirrors the boundary cell (a missing neighbour contributes nothing).  Readings listed in DESIGN.md.
"""
import numpy as np

from .demag_fft import demag_fft, kernel_spectrum

MU0 = 4e-7 * np.pi
GAMMA = 2.212761569e5          # mu0 |gamma_e| for g = 2.0023, m / (A s)


def exchange_field(m, h, A, Ms):
    """H_ex [3][nz][ny][nx] (A/m) of the unit field m: 2A/(mu0 Ms) * laplacian(m), dm/dn = 0."""
    m = np.asarray(m, np.float64)
    lap = np.zeros_like(m)
    for axis, d in ((3, h[0]), (2, h[1]), (1, h[2])):
        n = m.shape[axis]
        if n == 1:
            continue
        lo = [slice(None)] * 4
        hi = [slice(None)] * 4
        lo[axis], hi[axis] = slice(0, n - 1), slice(1, n)
        diff = (m[tuple(hi)] - m[tuple(lo)]) / (d * d)      # (m[i+1] - m[i]) / d^2 on the n - 1 interior faces
        lap[tuple(lo)] += diff                               # cell i gains from its upper neighbour
        lap[tuple(hi)] -= diff                               # cell i + 1 from its lower one; boundary faces add 0
    return 2.0 * A / (MU0 * Ms) * lap


def effective_field(m, h, Ms, A, Hext, Khat=None):
    """H_eff = H_demag(Ms m) + H_exchange(m) + H_applied."""
    m = np.asarray(m, np.float64)
    H = demag_fft(Ms * m, h, Khat=Khat)
    H += exchange_field(m, h, A, Ms)
    H += np.asarray(Hext, np.float64).reshape(3, 1, 1, 1)
    return H


def llg_rhs(m, H, gamma, alpha):
    """dm/dt of Eq. (1) in explicit form."""
    mxH = np.cross(m, H, axis=0)
    return -gamma / (1.0 + alpha * alpha) * (mxH + alpha * np.cross(m, mxH, axis=0))


def rk4_step(m, dt, h, Ms, A, Hext, gamma, alpha, Khat=None):
    """One classical Runge-Kutta step of Eq. (1) (4 effective-field evaluations, L283), then renormalisation."""
    f = lambda u: llg_rhs(u, effective_field(u, h, Ms, A, Hext, Khat), gamma, alpha)
    k1 = f(m)
    k2 = f(m + 0.5 * dt * k1)
    k3 = f(m + 0.5 * dt * k2)
    k4 = f(m + dt * k3)
    out = m + dt / 6.0 * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
    return out / np.sqrt((out * out).sum(axis=0, keepdims=True))


def total_energy(m, h, Ms, A, Hext, Khat=None):
    """E = E_demag + E_exchange + E_zeeman in joules: -(mu0/2) sum M.Hd dV - (mu0/2) sum M.Hex dV - mu0 sum M.Hext dV
    (the exchange term is quadratic like the demag term, hence its 1/2)."""
    m = np.asarray(m, np.float64)
    dV = h[0] * h[1] * h[2]
    M = Ms * m
    Hd = demag_fft(M, h, Khat=Khat)
    Hx = exchange_field(m, h, A, Ms)
    Hz = np.asarray(Hext, np.float64).reshape(3, 1, 1, 1)
    return float(-MU0 * dV * (0.5 * (M * Hd).sum() + 0.5 * (M * Hx).sum() + (M * Hz).sum()))


def precompute(shape, h):
    return kernel_spectrum(shape, h)
