"""Pins of the radiative (Sommerfeld) outer boundary, reading S16 of DESIGN.md (second boundary kind;
the paper's block faces: PAPER.md:105, :117-123).  CPU only.

B1 the one-sided and centred second-order differences are exact on quadratics: the boundary right-hand side of a
   quadratic field equals its closed form to round-off at every boundary point (pins coefficients, sides, the
   coordinate origin and the 1/r term);
B2 an outgoing spherical wave phi = F(r - t)/r satisfies the condition exactly: the boundary right-hand sides of
   (phi, pi) converge to the analytic time derivatives at second order;
B3 a static 1/r tail on top of u_inf gives zero: d_t (u_inf + c/r) -> 0 at second order, with u_inf = 1 exactly on
   the five BSSN slots whose flat value is 1 and 0 elsewhere;
B4 evolution: a Gaussian pulse of the (phi, pi) system leaves a radiative block (what is left after it has crossed
   the faces is a small fraction of what a periodic block keeps), and exact flat BSSN data stays flat bitwise."""
import numpy as np
import pytest

from paper_1307_6488_b200 import inputs


def coords(n, g, h):
    """x, y, z of every point of the padded block, arrays [tz, ty, tx]"""
    ax = [(np.arange(-g, m + g) - 0.5 * (m - 1)) * h for m in n]
    z, y, x = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return x, y, z


def boundary_mask(n, g):
    m = np.ones((n[2] + 2 * g, n[1] + 2 * g, n[0] + 2 * g), dtype=bool)
    m[g:-g, g:-g, g:-g] = False
    return m


def test_B1_quadratic_fields_closed_form(oracle):
    n, g, h = (9, 7, 8), 3, 0.1
    x, y, z = coords(n, g, h)
    r = np.sqrt(x * x + y * y + z * z)
    u = 0.3 + 0.5 * x - 0.2 * y + 0.7 * z + 0.4 * x * x - 0.6 * y * y + 0.1 * z * z + 0.25 * x * y - 0.35 * y * z
    grad = (0.5 + 0.8 * x + 0.25 * y, -0.2 - 1.2 * y + 0.25 * x - 0.35 * z, 0.7 + 0.2 * z - 0.35 * y)
    want = -((x * grad[0] + y * grad[1] + z * grad[2]) / r + u / r)
    st = np.stack([u, 2.0 * u])
    got = oracle.radiative_rhs(oracle.SYS_WAVE, st, g, h)
    m = boundary_mask(n, g)
    assert np.max(np.abs(got[0][m] - want[m])) < 1e-12 * np.max(np.abs(want[m]))
    assert np.max(np.abs(got[1][m] - 2.0 * want[m])) < 1e-12 * np.max(np.abs(want[m]))
    assert not got[:, ~m].any()                       # interior entries are not this operator's


def test_B2_outgoing_spherical_wave_second_order(oracle):
    errs = []
    for n1, h in ((37, 0.125), (79, 0.0625)):   # the outermost points stay at 2.625 under refinement
        n, g = (n1, n1, n1), 3
        x, y, z = coords(n, g, h)
        r = np.sqrt(x * x + y * y + z * z)
        r0, w = 1.2, 0.6                              # pulse centred on r = r0: well inside, r > 0 on every point used
        F = lambda s: np.exp(-0.5 * ((s - r0) / w) ** 2)
        dF = lambda s: -(s - r0) / w ** 2 * F(s)
        ddF = lambda s: (((s - r0) / w ** 2) ** 2 - 1.0 / w ** 2) * F(s)
        rs = np.maximum(r, 1e-3)
        phi, pi = F(rs) / rs, -dF(rs) / rs            # at t = 0: phi = F(r - t)/r, pi = d_t phi
        got = oracle.radiative_rhs(oracle.SYS_WAVE, np.stack([phi, pi]), g, h)
        m = boundary_mask(n, g)
        e_phi = np.max(np.abs(got[0][m] - pi[m]))                     # d_t phi = pi
        e_pi = np.max(np.abs(got[1][m] - (ddF(rs) / rs)[m]))          # d_t pi = F''(r - t)/r
        errs.append((e_phi, e_pi))
    for a, b in zip(errs[:-1], errs[1:]):
        assert 3.0 < a[0] / b[0] < 5.5 and 3.0 < a[1] / b[1] < 5.5, errs


def test_B3_static_tail_and_u_infinity(oracle):
    errs = []
    for n1, h in ((12, 0.5), (29, 0.25)):           # outermost points at 4.25 in both
        n, g = (n1, n1, n1), 3
        x, y, z = coords(n, g, h)
        r = np.sqrt(x * x + y * y + z * z)
        m = boundary_mask(n, g)
        tail = 0.05 / np.maximum(r, h)
        st = np.stack([tail] * 25)
        for v in (0, 1, 4, 6, 17):
            st[v] += 1.0
        got = oracle.radiative_rhs(oracle.SYS_BSSN, st, g, h)
        errs.append(max(np.max(np.abs(got[v][m])) for v in range(25)))
        # the same tail without the background on a unit-background slot is NOT stationary: u_inf matters
        st[0] -= 1.0
        bad = oracle.radiative_rhs(oracle.SYS_BSSN, st, g, h)
        assert np.max(np.abs(bad[0][m])) > 100 * errs[-1]
    assert 3.0 < errs[0] / errs[1] < 5.5, errs


def test_B4_pulse_leaves_and_flat_stays_flat(oracle):
    n1, g, order = 24, 2, 4
    h = 1.0 / n1
    dt = 0.25 * h
    x, y, z = coords((n1,) * 3, g, h)
    phi = np.exp(-0.5 * (x * x + y * y + z * z) / 0.08 ** 2)
    u0 = np.stack([phi, np.zeros_like(phi)])
    steps = int(1.4 / dt)                             # the pulse (speed 1) crosses the half-width 0.5 and the corners
    rad = oracle.rk4_radiative(oracle.SYS_WAVE, u0.copy(), g, order, h, dt, oracle.params(), steps)
    per = oracle.rk4(oracle.SYS_WAVE, u0.copy(), g, order, h, dt, oracle.params(), steps)
    left = np.max(np.abs(rad[0][g:-g, g:-g, g:-g]))
    kept = np.max(np.abs(per[0][g:-g, g:-g, g:-g]))
    assert np.isfinite(rad).all() and left < 0.02 and left < 0.1 * kept, (left, kept)
    flat = oracle.with_ghosts(inputs.bssn_minkowski(8, 8, 8), 3)
    flat = oracle.fill_ghosts(flat, 3)
    out = oracle.rk4_radiative(oracle.SYS_BSSN, flat.copy(), 3, 4, 0.05, 0.0125, oracle.params(eps_diss=0.1), 2)
    assert np.array_equal(out, flat)
