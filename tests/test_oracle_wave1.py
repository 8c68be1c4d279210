"""Pins for the oracle's system 2, the fully first-order wave system of the paper's Sample 1:
(W1) the exact solution of the *discrete* scheme, per Fourier mode, from the closed-form symbols of the centred
first-derivative and KO stencils -- no stencil code involved; (W2) the discrete energy identity: with centred
(skew-symmetric) differences on a periodic grid  sum(rho * d_t rho + v_i * d_t v_i) = 0  to round-off, which is
what conserves the paper's `eps = 1/2 (rho^2 + v_i v_i)`; (W3) a Gaussian pulse keeps that energy over 20 steps
to the RK4 truncation level.  CPU only."""
import numpy as np
import pytest

from paper_1307_6488_b200 import inputs


def dsym(theta, order):
    """h/i * symbol of the centred first-derivative stencil (reading S2)."""
    if order == 4:
        return (8.0 * np.sin(theta) - np.sin(2 * theta)) / 6.0
    return (672.0 * np.sin(theta) - 168.0 * np.sin(2 * theta) + 32.0 * np.sin(3 * theta) - 3.0 * np.sin(4 * theta)) / 420.0


def exact_discrete(state, order, h, dt, eps, nsteps):
    _, nz, ny, nx = state.shape
    th = [2 * np.pi * np.fft.fftfreq(n) for n in (nz, ny, nx)]
    TZ, TY, TX = np.meshgrid(*th, indexing="ij")
    kx, ky, kz = (1j * dsym(T, order) / h for T in (TX, TY, TZ))
    s = (eps / h) * (np.sin(TX / 2) ** 6 + np.sin(TY / 2) ** 6 + np.sin(TZ / 2) ** 6)
    M = np.zeros(TX.shape + (5, 5), dtype=complex)
    for c in range(5):
        M[..., c, c] = -s
    M[..., 0, 1] = 1.0
    M[..., 1, 2], M[..., 1, 3], M[..., 1, 4] = kx, ky, kz
    M[..., 2, 1], M[..., 3, 1], M[..., 4, 1] = kx, ky, kz
    Z = dt * M
    I = np.broadcast_to(np.eye(5), Z.shape)
    Z2 = Z @ Z
    P = I + Z + Z2 / 2 + (Z2 @ Z) / 6 + (Z2 @ Z2) / 24
    Pn = np.linalg.matrix_power(P, nsteps)
    f = np.stack([np.fft.fftn(state[c]) for c in range(5)], axis=-1)[..., None]
    g = (Pn @ f)[..., 0]
    return np.stack([np.fft.ifftn(g[..., c]).real for c in range(5)])


def relerr(a, b):
    return max(np.max(np.abs(a[v] - b[v])) / max(np.max(np.abs(b[v])), 1e-300) for v in range(a.shape[0]))


@pytest.mark.parametrize("order,g,eps,dims", [(4, 2, 0.0, (16, 12, 20)), (8, 4, 0.1, (16, 20, 12)), (4, 3, 0.1, (12, 12, 12))])
def test_W1_exact_discrete_solution(oracle, order, g, eps, dims):
    nx, ny, nz = dims
    u0 = np.random.default_rng(43).standard_normal((5, nz, ny, nx))   # white noise excites every mode
    h, nsteps = 1.0 / 16, 5
    dt = 0.25 * h
    got = oracle.interior(oracle.rk4(oracle.SYS_WAVE1, oracle.with_ghosts(u0, g), g, order, h, dt,
                                     oracle.params(eps_diss=eps), nsteps), g)
    assert relerr(got, exact_discrete(u0, order, h, dt, eps, nsteps)) < 2e-13


@pytest.mark.parametrize("order,g", [(4, 2), (8, 4)])
def test_W2_energy_identity(oracle, order, g):
    u0 = np.random.default_rng(44).standard_normal((5, 10, 12, 14))
    st = oracle.fill_ghosts(oracle.with_ghosts(u0, g), g)
    r = oracle.interior(oracle.rhs(oracle.SYS_WAVE1, st, g, order, 0.1, oracle.params()), g)
    terms = u0[1] * r[1] + sum(u0[2 + a] * r[2 + a] for a in range(3))
    assert abs(terms.sum()) < 1e-12 * np.abs(terms).sum()
    assert np.array_equal(r[0], u0[1])                                  # D_t u = rho exactly


def test_W3_gaussian_pulse_keeps_energy(oracle):
    """the paper's own initial data: u = 0, rho = A exp(-1/2 (r/W)^2), v_i = 0"""
    n, g, order = 32, 2, 4
    u0 = inputs.wave1_gaussian(n, n, n)
    h = 1.0 / n
    e0 = 0.5 * (u0[1] ** 2 + (u0[2:] ** 2).sum(0)).sum()
    st = oracle.rk4(oracle.SYS_WAVE1, oracle.with_ghosts(u0, g), g, order, h, 0.25 * h, oracle.params(), 20)
    u1 = oracle.interior(st, g)
    e1 = 0.5 * (u1[1] ** 2 + (u1[2:] ** 2).sum(0)).sum()
    assert abs(e1 / e0 - 1.0) < 1e-6 and np.abs(u1[2:]).max() > 1e-3     # conserved, and something did propagate


def test_W4_energy_closed_forms(oracle):
    """eps = 1/2 (rho^2 + v_i v_i): u does not enter, every v_i enters once with weight 1/2"""
    g = 2
    u = np.zeros((5, 4, 5, 6))
    u[0] = 7.0                                   # u must not contribute
    u[1], u[2], u[3], u[4] = 3.0, 1.0, 2.0, 2.0
    assert np.array_equal(oracle.energy(oracle.with_ghosts(u, g), g), np.full((4, 5, 6), 9.0))
    for c, val in [(1, 2.0), (2, 4.0), (3, 6.0), (4, 8.0)]:
        e = np.zeros((5, 4, 5, 6)); e[c] = val
        assert np.array_equal(oracle.energy(oracle.with_ghosts(e, g), g), np.full((4, 5, 6), 0.5 * val * val))
    # the energy the conservation pin W3 sums is this field
    w = inputs.wave1_gaussian(8, 8, 8)
    assert np.isclose(oracle.energy(oracle.with_ghosts(w, g), g).sum(), 0.5 * (w[1] ** 2).sum(), rtol=1e-15)
