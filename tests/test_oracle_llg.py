"""Pins of the LLG evaluation oracle (oracle/llg.py) against what the paper and the mathematics fix (CPU only)."""
import numpy as np

from oracle import llg

MU0 = 4e-7 * np.pi


def test_explicit_form_satisfies_the_paper_equation_1():
    """dm/dt = -gamma m x H + alpha m x dm/dt, retyped here in its implicit form."""
    rng = np.random.default_rng(1)
    m = rng.standard_normal((3, 2, 3, 4))
    m /= np.sqrt((m * m).sum(0))
    H = rng.standard_normal(m.shape) * 1e5
    gamma, alpha = llg.GAMMA, 0.3
    d = llg.llg_rhs(m, H, gamma, alpha)
    res = d + gamma * np.cross(m, H, axis=0) - alpha * np.cross(m, d, axis=0)
    assert np.abs(res).max() <= 1e-12 * np.abs(d).max()
    assert np.abs((m * d).sum(0)).max() <= 1e-12 * np.abs(d).max()          # |m| is conserved


def test_exchange_field_of_polynomials_and_the_neumann_boundary():
    """H = 2A/(mu0 Ms) laplacian(m), dm/dn = 0."""
    A, Ms = 1.3e-11, 8e5
    h = (2e-9, 3e-9, 4e-9)
    c = 2 * A / (MU0 * Ms)
    nz, ny, nx = 5, 6, 7
    z, y, x = np.meshgrid(np.arange(nz) * h[2], np.arange(ny) * h[1], np.arange(nx) * h[0], indexing="ij")
    f = np.stack([x * x + 2 * y * y, 3 * z * z, np.ones_like(x)])            # laplacians 2 + 4, 6, 0
    H = llg.exchange_field(f, h, A, Ms)
    inner = (slice(None), slice(1, -1), slice(1, -1), slice(1, -1))
    assert np.allclose(H[inner][0], 6 * c, rtol=1e-9) and np.allclose(H[inner][1], 6 * c, rtol=1e-9)
    assert np.abs(H[2]).max() == 0.0                                         # uniform field: no exchange field
    g = np.stack([x, np.zeros_like(x), np.zeros_like(x)])                    # linear: only the mirrored boundary cells feel it
    Hg = llg.exchange_field(g, h, A, Ms)[0]
    assert np.abs(Hg[:, :, 1:-1]).max() <= 1e-9 * c / h[0]
    assert np.allclose(Hg[:, :, 0], c / h[0]) and np.allclose(Hg[:, :, -1], -c / h[0])
    # 2-D mode: a single layer has no z neighbours
    assert np.array_equal(llg.exchange_field(f[:, :1], h, A, Ms)[2], np.zeros((1, ny, nx)))


def test_single_cubic_cell_follows_the_closed_form_damped_precession():
    """One cubic cell: N = 1/3 I, the demag field is parallel to m and exerts no torque, so m precesses about the
    applied field H z^ with m_z(t) = tanh(a t + atanh m_z(0)), a = alpha gamma H / (1 + alpha^2), and azimuth
    phi(t) = phi(0) + gamma H t / (1 + alpha^2) (textbook solution of the LLG equation in a constant field)."""
    h = (2e-9, 2e-9, 2e-9)
    Ms, A, alpha, gamma = 8e5, 1.3e-11, 0.1, llg.GAMMA
    Hz = 2e5
    th0 = 1.0
    m = np.array([np.sin(th0), 0.0, np.cos(th0)]).reshape(3, 1, 1, 1)
    Khat = llg.precompute((1, 1, 1), h)
    dt, n = 5e-14, 400
    for _ in range(n):
        m = llg.rk4_step(m, dt, h, Ms, A, (0.0, 0.0, Hz), gamma, alpha, Khat)
    t = n * dt
    a = alpha * gamma * Hz / (1 + alpha ** 2)
    mz = np.tanh(a * t + np.arctanh(np.cos(th0)))
    phi = gamma * Hz * t / (1 + alpha ** 2)
    ref = np.array([np.sqrt(1 - mz ** 2) * np.cos(phi), np.sqrt(1 - mz ** 2) * np.sin(phi), mz])
    assert np.abs(m.ravel() - ref).max() <= 1e-8


def test_energy_is_conserved_without_damping_and_decreases_with_it():
    """Eq. (1) gives dE/dt = -mu0 Ms alpha gamma/(1+alpha^2) sum |m x H|^2 dV <= 0, = 0 for alpha = 0."""
    rng = np.random.default_rng(3)
    shape, h = (2, 4, 6), (3e-9, 3e-9, 2e-9)
    Ms, A, Hext = 8e5, 1.3e-11, (1e4, -2e4, 3e4)
    m0 = rng.standard_normal((3,) + shape)
    m0 /= np.sqrt((m0 * m0).sum(0))
    Khat = llg.precompute(shape, h)
    for alpha in (0.0, 0.5):
        m, E = m0.copy(), [llg.total_energy(m0, h, Ms, A, Hext, Khat)]
        for _ in range(20):
            m = llg.rk4_step(m, 2e-14, h, Ms, A, Hext, llg.GAMMA, alpha, Khat)
            E.append(llg.total_energy(m, h, Ms, A, Hext, Khat))
            assert np.abs((m * m).sum(0) - 1).max() <= 1e-14
        E = np.array(E)
        if alpha == 0.0:
            assert np.abs(E - E[0]).max() <= 1e-7 * np.abs(E[0])
        else:
            assert np.all(np.diff(E) < 0)
