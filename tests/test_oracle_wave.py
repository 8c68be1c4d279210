"""Pins O2 / O3 for the wave system: the oracle's RHS + KO + ghost fill + RK4 against
(O2) the exact solution of the *discrete* scheme, computed per Fourier mode with numpy FFTs and the
closed-form symbols of the stencils -- no stencil code involved -- and (O3) the continuum standing
wave, for the convergence order.  CPU only."""
import numpy as np
import pytest

from paper_1307_6488_b200 import inputs


def lam(theta, order):
    """h^2 * symbol of the centred second-derivative stencil (S2)."""
    if order == 4:
        return -5.0 / 2 + (8.0 / 3) * np.cos(theta) - (1.0 / 6) * np.cos(2 * theta)
    return (-205.0 / 72 + (16.0 / 5) * np.cos(theta) - (2.0 / 5) * np.cos(2 * theta)
            + (16.0 / 315) * np.cos(3 * theta) - (1.0 / 280) * np.cos(4 * theta))


def exact_discrete(state, order, h, dt, eps, nsteps, ko_order=5):
    """Each Fourier mode evolves by P(dt M)^n, M = [[-s, 1], [-L, -s]], P = RK4 stability polynomial."""
    _, nz, ny, nx = state.shape
    th = [2 * np.pi * np.fft.fftfreq(n) for n in (nz, ny, nx)]
    TZ, TY, TX = np.meshgrid(*th, indexing="ij")
    L = -(lam(TX, order) + lam(TY, order) + lam(TZ, order)) / h ** 2
    p = ko_order + 1   # S6: sin^6 ; S6b: sin^10
    s = (eps / h) * (np.sin(TX / 2) ** p + np.sin(TY / 2) ** p + np.sin(TZ / 2) ** p)
    M = np.empty(L.shape + (2, 2))
    M[..., 0, 0] = -s; M[..., 0, 1] = 1.0; M[..., 1, 0] = -L; M[..., 1, 1] = -s
    Z = dt * M
    I = np.broadcast_to(np.eye(2), Z.shape)
    Z2 = Z @ Z
    P = I + Z + Z2 / 2 + (Z2 @ Z) / 6 + (Z2 @ Z2) / 24
    Pn = np.linalg.matrix_power(P, nsteps)
    fphi, fpi = np.fft.fftn(state[0]), np.fft.fftn(state[1])
    out = np.empty_like(state)
    out[0] = np.fft.ifftn(Pn[..., 0, 0] * fphi + Pn[..., 0, 1] * fpi).real
    out[1] = np.fft.ifftn(Pn[..., 1, 0] * fphi + Pn[..., 1, 1] * fpi).real
    return out


def relerr(a, b):
    """S11: per variable max|a-b| / max|b|, then max over variables."""
    return max(np.max(np.abs(a[v] - b[v])) / max(np.max(np.abs(b[v])), 1e-300) for v in range(a.shape[0]))


@pytest.mark.parametrize("order,g,eps,dims", [(4, 2, 0.0, (16, 12, 20)), (8, 4, 0.1, (16, 20, 12)),
                                              (4, 3, 0.1, (12, 12, 12)), (8, 4, 0.0, (16, 16, 16))])
def test_O2_exact_discrete_solution(oracle, order, g, eps, dims):
    nx, ny, nz = dims
    rng = np.random.default_rng(42)
    u0 = rng.standard_normal((2, nz, ny, nx))   # white noise excites every mode
    h, nsteps = 1.0 / 16, 5
    dt = 0.25 * h
    got = oracle.interior(oracle.rk4(oracle.SYS_WAVE, oracle.with_ghosts(u0, g), g, order, h, dt,
                                     oracle.params(eps_diss=eps), nsteps), g)
    want = exact_discrete(u0, order, h, dt, eps, nsteps)
    assert relerr(got, want) < 2e-13


def test_O2_exact_discrete_solution_ko9(oracle):
    """S6b through the whole path: 8th order, 5 ghost zones, 9th-order KO, against the per-mode solution."""
    nx, ny, nz = 16, 12, 20
    rng = np.random.default_rng(43)
    u0 = rng.standard_normal((2, nz, ny, nx))
    h, nsteps, g, eps = 1.0 / 16, 5, 5, 0.1
    dt = 0.25 * h
    got = oracle.interior(oracle.rk4(oracle.SYS_WAVE, oracle.with_ghosts(u0, g), g, 8, h, dt,
                                     oracle.params(eps_diss=eps, ko_order=9), nsteps), g)
    want = exact_discrete(u0, 8, h, dt, eps, nsteps, ko_order=9)
    assert relerr(got, want) < 2e-13
    # and it is not the 5th-order operator
    assert relerr(got, exact_discrete(u0, 8, h, dt, eps, nsteps, ko_order=5)) > 1e-4


def test_O2_config0_and_config1_shapes(oracle):
    """the two wave configs of BASELINE.json (config 1 scaled to 32^3), own data, 20 / 3 steps."""
    c = inputs.config(0)
    u0 = c["state"]()
    got = oracle.interior(oracle.rk4(oracle.SYS_WAVE, oracle.with_ghosts(u0, c["ghost"]), c["ghost"], c["order"],
                                     c["dx"], 0.25 * c["dx"], oracle.params(eps_diss=c["eps_diss"]), 20), c["ghost"])
    want = exact_discrete(u0, c["order"], c["dx"], 0.25 * c["dx"], c["eps_diss"], 20)
    assert relerr(got, want) < 1e-12
    c = inputs.config(1, scale=32)
    u0 = c["state"]()
    got = oracle.interior(oracle.rk4(oracle.SYS_WAVE, oracle.with_ghosts(u0, c["ghost"]), c["ghost"], c["order"],
                                     c["dx"], 0.25 * c["dx"], oracle.params(eps_diss=c["eps_diss"]), 3), c["ghost"])
    want = exact_discrete(u0, c["order"], c["dx"], 0.25 * c["dx"], c["eps_diss"], 3)
    assert relerr(got, want) < 1e-12


def test_O3_rhs_convergence_order(oracle):
    """Laplacian of sin sin sin vs -12 pi^2 phi: error ratio 2^4 (O4) and 2^8 (O8) under refinement."""
    for order, g, want_ratio in ((4, 2, 16.0), (8, 4, 256.0)):
        errs = []
        for n in (8, 16, 32):
            u = inputs.wave_standing(n, n, n, noise=0.0)
            st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
            r = oracle.interior(oracle.rhs(oracle.SYS_WAVE, st, g, order, 1.0 / n, oracle.params()), g)
            assert np.array_equal(r[0], u[1])            # d_t phi = pi exactly
            errs.append(np.max(np.abs(r[1] + 12 * np.pi ** 2 * u[0])))
        assert errs[0] / errs[1] == pytest.approx(want_ratio, rel=0.25)
        assert errs[1] / errs[2] == pytest.approx(want_ratio, rel=0.08)


def test_O3_evolution_convergence_order(oracle):
    """standing wave phi = sin sin sin cos(2 pi sqrt3 t): 4th-order scheme + RK4, dt ~ dx -> ratio 16."""
    errs = []
    T = 0.125
    for n in (16, 32, 64):
        h = 1.0 / n
        dt = 0.25 * h
        nsteps = int(round(T / dt))
        u = inputs.wave_standing(n, n, n, noise=0.0)
        got = oracle.interior(oracle.rk4(oracle.SYS_WAVE, oracle.with_ghosts(u, 2), 2, 4, h, dt, oracle.params(),
                                         nsteps), 2)
        want = u[0] * np.cos(2 * np.pi * np.sqrt(3.0) * T)
        errs.append(np.max(np.abs(got[0] - want)))
    assert errs[0] / errs[1] == pytest.approx(16.0, rel=0.15)
    assert errs[1] / errs[2] == pytest.approx(16.0, rel=0.08)
