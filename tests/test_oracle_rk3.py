"""Pins for the oracle's RK3 (reading S9b, Shu-Osher) and BSSN constraint enforcement (reading S10b), SURVEY 8(f)-2.
(R1/R2) on a linear system any 3-stage third-order Runge-Kutta step is P3(dt M) = 1 + z + z^2/2 + z^3/6, so the
exact discrete Fourier solutions of test_oracle_wave / test_oracle_wave1 pin it with that polynomial; (E1-E4)
closed-form properties of the enforcement.  CPU only."""
import numpy as np
import pytest

from tests.test_oracle_wave import lam, relerr
from tests.test_oracle_wave1 import dsym


def _modes(shape):
    nz, ny, nx = shape
    th = [2 * np.pi * np.fft.fftfreq(n) for n in (nz, ny, nx)]
    return np.meshgrid(*th, indexing="ij")


def _p3_power(M, dt, nsteps):
    Z = dt * M
    I = np.broadcast_to(np.eye(M.shape[-1]), Z.shape)
    Z2 = Z @ Z
    return np.linalg.matrix_power(I + Z + Z2 / 2 + (Z2 @ Z) / 6, nsteps)


def _apply(Pn, state):
    V = state.shape[0]
    f = np.stack([np.fft.fftn(state[c]) for c in range(V)], axis=-1)[..., None]
    g = (Pn @ f)[..., 0]
    return np.stack([np.fft.ifftn(g[..., c]).real for c in range(V)])


@pytest.mark.parametrize("order,g,eps", [(4, 2, 0.0), (8, 4, 0.1)])
def test_R1_wave_rk3_exact_discrete(oracle, order, g, eps):
    u0 = np.random.default_rng(51).standard_normal((2, 12, 16, 20))
    h, n = 1.0 / 16, 5
    dt = 0.25 * h
    TZ, TY, TX = _modes(u0.shape[1:])
    L = -(lam(TX, order) + lam(TY, order) + lam(TZ, order)) / h ** 2
    s = (eps / h) * (np.sin(TX / 2) ** 6 + np.sin(TY / 2) ** 6 + np.sin(TZ / 2) ** 6)
    M = np.zeros(L.shape + (2, 2))
    M[..., 0, 0] = -s; M[..., 0, 1] = 1.0; M[..., 1, 0] = -L; M[..., 1, 1] = -s
    got = oracle.interior(oracle.rk3(oracle.SYS_WAVE, oracle.with_ghosts(u0, g), g, order, h, dt,
                                     oracle.params(eps_diss=eps), n), g)
    assert relerr(got, _apply(_p3_power(M, dt, n), u0)) < 2e-13


def test_R2_wave1_rk3_exact_discrete(oracle):
    order, g, eps = 4, 3, 0.1
    u0 = np.random.default_rng(52).standard_normal((5, 12, 12, 16))
    h, n = 1.0 / 16, 4
    dt = 0.25 * h
    TZ, TY, TX = _modes(u0.shape[1:])
    kx, ky, kz = (1j * dsym(T, order) / h for T in (TX, TY, TZ))
    s = (eps / h) * (np.sin(TX / 2) ** 6 + np.sin(TY / 2) ** 6 + np.sin(TZ / 2) ** 6)
    M = np.zeros(TX.shape + (5, 5), dtype=complex)
    for c in range(5):
        M[..., c, c] = -s
    M[..., 0, 1] = 1.0
    M[..., 1, 2], M[..., 1, 3], M[..., 1, 4] = kx, ky, kz
    M[..., 2, 1], M[..., 3, 1], M[..., 4, 1] = kx, ky, kz
    got = oracle.interior(oracle.rk3(oracle.SYS_WAVE1, oracle.with_ghosts(u0, g), g, order, h, dt,
                                     oracle.params(eps_diss=eps), n), g)
    assert relerr(got, _apply(_p3_power(M, dt, n), u0)) < 2e-13


def _mat(p6):
    """packed (11,12,13,22,23,33) arrays -> [..., 3, 3]"""
    a, b, c, d, e, f = p6
    return np.stack([np.stack([a, b, c], -1), np.stack([b, d, e], -1), np.stack([c, e, f], -1)], -2)


def _random_bssn(seed, shape=(6, 5, 7)):
    rng = np.random.default_rng(seed)
    u = rng.standard_normal((25,) + shape)
    u[1:7] = 0.2 * rng.uniform(-1, 1, (6,) + shape)
    u[1] += 1.3; u[4] += 0.9; u[6] += 1.1            # a positive-definite conformal metric, det != 1
    return u


def test_E1_det_one_trace_zero_others_untouched(oracle):
    u = _random_bssn(61)
    g = 3
    out = oracle.interior(oracle.enforce(oracle.with_ghosts(u, g), g), g)
    G, A = _mat(out[1:7]), _mat(out[8:14])
    assert np.max(np.abs(np.linalg.det(G) - 1.0)) < 1e-14
    tr = np.einsum("...ij,...ij->...", np.linalg.inv(G), A)
    assert np.max(np.abs(tr)) < 1e-14 * np.max(np.abs(A))
    for v in [0, 7] + list(range(14, 25)):
        assert np.array_equal(out[v], u[v])
    # the metric is only rescaled and only the trace part of At is removed
    G0, A0 = _mat(u[1:7]), _mat(u[8:14])
    lam0 = np.linalg.det(G0) ** (-1.0 / 3.0)
    assert np.allclose(G, lam0[..., None, None] * G0, rtol=1e-14, atol=0)
    tr0 = np.einsum("...ij,...ij->...", np.linalg.inv(G), A0)
    assert np.allclose(A, A0 - tr0[..., None, None] / 3.0 * G, rtol=1e-13, atol=1e-14)


def test_E2_idempotent_and_conformally_invariant(oracle):
    u = _random_bssn(62)
    g = 3
    once = oracle.interior(oracle.enforce(oracle.with_ghosts(u, g), g), g)
    twice = oracle.interior(oracle.enforce(oracle.with_ghosts(once, g), g), g)
    assert np.max(np.abs(twice - once)) < 1e-14
    v = u.copy()
    v[1:7] *= 2.5                                      # a conformal rescaling of gt does not change the result
    resc = oracle.interior(oracle.enforce(oracle.with_ghosts(v, g), g), g)
    assert np.max(np.abs(resc[1:7] - once[1:7])) < 1e-14


def test_E3_flat_data_bitwise_unchanged(oracle):
    from paper_1307_6488_b200 import inputs
    u = inputs.bssn_minkowski(5, 4, 6)
    g = 3
    assert np.array_equal(oracle.interior(oracle.enforce(oracle.with_ghosts(u, g), g), g), u)


def test_E4_rk3_with_enforcement_keeps_constraints(oracle):
    """a few RK3 steps of BSSN with enforcement: det gt = 1 and tr At = 0 after every step, state stays finite"""
    from paper_1307_6488_b200 import inputs
    n, g, dx = 12, 3, 0.05
    u0 = inputs.bssn_gaussians(n, n, n, amp=1e-3, width_cells=3.0)
    st = oracle.rk3(oracle.SYS_BSSN, oracle.with_ghosts(u0, g), g, 4, dx, 0.25 * dx, oracle.params(eps_diss=0.1), 3, True)
    out = oracle.interior(st, g)
    G, A = _mat(out[1:7]), _mat(out[8:14])
    assert np.isfinite(out).all()
    assert np.max(np.abs(np.linalg.det(G) - 1.0)) < 1e-14
    assert np.max(np.abs(np.einsum("...ij,...ij->...", np.linalg.inv(G), A))) < 1e-18 + 1e-14 * np.max(np.abs(A))
