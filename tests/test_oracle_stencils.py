"""Pin O1: every stencil of the oracle is exact on polynomials up to its order, and has the right
leading error term (reading S2 / S6).  Non-periodic: the ghosts are filled from the
polynomial itself, so only the stencils are under test.  CPU only."""
import numpy as np
import pytest

H = 0.37  # deliberately not a power of two


def poly_grid(cx, cy, cz, n, g, h):
    """f = X(x) * Y(y) * Z(z), each a 1-D polynomial (numpy.polynomial coefficients, low first)."""
    idx = (np.arange(-g, n + g, dtype=np.float64)) * h
    P = np.polynomial.polynomial
    fx, fy, fz = P.polyval(idx, cx), P.polyval(idx, cy), P.polyval(idx, cz)
    return fz[:, None, None] * fy[None, :, None] * fx[None, None, :], idx


def poly_exact(cx, cy, cz, idx, g, nder):
    """exact derivative, nder = (a,b,c) derivative orders along x,y,z, on interior points."""
    P = np.polynomial.polynomial
    ii = idx[g:-g]
    d = [P.polyval(ii, P.polyder(np.asarray(c, dtype=float), m) if m else np.asarray(c, dtype=float))
         for c, m in zip((cx, cy, cz), nder)]
    return d[2][:, None, None] * d[1][None, :, None] * d[0][None, None, :]


def rand_poly(rng, deg):
    return rng.uniform(-1.0, 1.0, size=deg + 1)


@pytest.mark.parametrize("order", [4, 8])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_d1_exact_to_order(oracle, order, axis):
    rng = np.random.default_rng(100 + order + axis)
    g, n = order // 2, 5
    c = [rand_poly(rng, 2), rand_poly(rng, 2), rand_poly(rng, 2)]
    c[axis] = rand_poly(rng, order)  # exact for degree <= order
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_D1, np.ascontiguousarray(f), g, order, H, a=axis)
    nder = [0, 0, 0]; nder[axis] = 1
    want = poly_exact(*c, idx, g, nder)
    assert np.max(np.abs(got - want)) <= 2e-13 * np.max(np.abs(want))
    # degree order+1 is NOT exact: the stencil really has that order, no higher
    c[axis] = np.zeros(order + 2); c[axis][-1] = 1.0
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_D1, np.ascontiguousarray(f), g, order, H, a=axis)
    want = poly_exact(*c, idx, g, nder)
    assert np.max(np.abs(got - want)) > 1e-6 * np.max(np.abs(want))


@pytest.mark.parametrize("order", [4, 8])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_d2_exact_to_order_plus_one(oracle, order, axis):
    rng = np.random.default_rng(200 + order + axis)
    g, n = order // 2, 5
    c = [rand_poly(rng, 2), rand_poly(rng, 2), rand_poly(rng, 2)]
    c[axis] = rand_poly(rng, order + 1)  # symmetric stencil: exact for degree <= order+1
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_DD, np.ascontiguousarray(f), g, order, H, a=axis, b=axis)
    nder = [0, 0, 0]; nder[axis] = 2
    want = poly_exact(*c, idx, g, nder)
    assert np.max(np.abs(got - want)) <= 5e-13 * np.max(np.abs(want))
    c[axis] = np.zeros(order + 3); c[axis][-1] = 1.0
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_DD, np.ascontiguousarray(f), g, order, H, a=axis, b=axis)
    want = poly_exact(*c, idx, g, nder)
    assert np.max(np.abs(got - want)) > 1e-6 * np.max(np.abs(want))


@pytest.mark.parametrize("order", [4, 8])
@pytest.mark.parametrize("a,b", [(0, 1), (0, 2), (1, 2), (1, 0), (2, 0), (2, 1)])
def test_mixed_exact(oracle, order, a, b):
    rng = np.random.default_rng(300 + order + 3 * a + b)
    g, n = order // 2, 4
    c = [rand_poly(rng, order), rand_poly(rng, order), rand_poly(rng, order)]
    other = 3 - a - b
    c[other] = rand_poly(rng, 2)
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_DD, np.ascontiguousarray(f), g, order, H, a=a, b=b)
    nder = [0, 0, 0]; nder[a] = 1; nder[b] = 1
    want = poly_exact(*c, idx, g, nder)
    assert np.max(np.abs(got - want)) <= 5e-13 * np.max(np.abs(want))


@pytest.mark.parametrize("order", [4, 8])
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("side", [+1, -1])
def test_upwind_exact_and_biased(oracle, order, axis, side):
    rng = np.random.default_rng(400 + order + axis + side)
    g, n = order // 2 + 1, 4   # upwinded 8th order needs 5 ghost zones
    c = [rand_poly(rng, 1), rand_poly(rng, 1), rand_poly(rng, 1)]
    c[axis] = rand_poly(rng, order)
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_UPW, np.ascontiguousarray(f), g, order, H, a=axis, b=side)
    nder = [0, 0, 0]; nder[axis] = 1
    want = poly_exact(*c, idx, g, nder)
    assert np.max(np.abs(got - want)) <= 5e-13 * np.max(np.abs(want))
    # the stencil must really be one-sided: a spike at offset +side*(order/2+1) is seen, at the
    # mirrored offset it is not (catches a swapped side / mirrored coefficients)
    reach = order // 2 + 1
    z = np.zeros((n + 2 * g,) * 3)
    p = [g + 1, g + 1, g + 1]
    q = list(p); q[axis] += side * reach
    z[q[2], q[1], q[0]] = 1.0
    got = oracle.apply_op(oracle.OP_UPW, z, g, order, H, a=axis, b=side)
    coef = {4: 1.0 / 12.0, 8: 3.0 / 840.0}[order]  # outermost coefficient, S2
    assert got[1, 1, 1] == pytest.approx(side * coef / H, rel=1e-14)
    q = list(p); q[axis] -= side * reach
    z[:] = 0.0
    z[q[2], q[1], q[0]] = 1.0
    got = oracle.apply_op(oracle.OP_UPW, z, g, order, H, a=axis, b=side)
    assert got[1, 1, 1] == 0.0


def test_ko5_annihilates_degree5_and_sees_degree6(oracle):
    rng = np.random.default_rng(500)
    g, n, eps = 3, 4, 0.1
    c = [rand_poly(rng, 5), rand_poly(rng, 5), rand_poly(rng, 5)]
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_KO, np.ascontiguousarray(f), g, 4, H, eps=eps)
    assert np.max(np.abs(got)) <= 1e-11 * np.max(np.abs(f)) / H
    # on a6 x^6 the 6th undivided difference is 720 a6 h^6: KO = eps * 720 a6 h^5 / 64  (S6)
    a6 = 0.7
    for axis in range(3):
        c = [np.ones(1), np.ones(1), np.ones(1)]
        c[axis] = np.array([0, 0, 0, 0, 0, 0, a6])
        f, idx = poly_grid(*c, n, g, H)
        got = oracle.apply_op(oracle.OP_KO, np.ascontiguousarray(f), g, 4, H, eps=eps)
        want = eps * 720.0 * a6 * H ** 5 / 64.0
        assert np.allclose(got, want, rtol=1e-9, atol=0.0)


def test_ko5_symbol(oracle):
    """S6: on exp(i theta i) the KO operator multiplies by -(eps/h) sin^6(theta/2) per axis."""
    n, g, eps, h = 16, 3, 0.1, 1.0 / 16
    m = 3
    i = np.arange(-g, n + g)
    theta = 2 * np.pi * m / n
    f = np.cos(theta * i)[None, None, :] * np.ones((n + 2 * g, n + 2 * g, 1))
    got = oracle.apply_op(oracle.OP_KO, np.ascontiguousarray(f), g, 4, h, eps=eps)
    want = -(eps / h) * np.sin(theta / 2) ** 6 * f[g:-g, g:-g, g:-g]
    assert np.max(np.abs(got - want)) < 1e-13 * (eps / h)


def test_ko9_annihilates_degree9_and_sees_degree10(oracle):
    """S6b: the 11-point operator is (eps/1024h) times the 10th undivided central difference."""
    rng = np.random.default_rng(501)
    g, n, eps = 5, 4, 0.1
    c = [rand_poly(rng, 9), rand_poly(rng, 9), rand_poly(rng, 9)]
    f, idx = poly_grid(*c, n, g, H)
    got = oracle.apply_op(oracle.OP_KO9, np.ascontiguousarray(f), g, 8, H, eps=eps)
    assert np.max(np.abs(got)) <= 1e-9 * np.max(np.abs(f)) / H
    # on a10 x^10 the 10th undivided difference is 10! a10 h^10: KO9 = eps * 3628800 a10 h^9 / 1024
    a10 = 0.7
    for axis in range(3):
        c = [np.ones(1), np.ones(1), np.ones(1)]
        c[axis] = np.array([0.0] * 10 + [a10])
        f, idx = poly_grid(*c, n, g, H)
        got = oracle.apply_op(oracle.OP_KO9, np.ascontiguousarray(f), g, 8, H, eps=eps)
        want = eps * 3628800.0 * a10 * H ** 9 / 1024.0
        assert np.allclose(got, want, rtol=1e-6, atol=0.0)


def test_ko9_symbol_and_single_point_weights(oracle):
    """S6b: on exp(i theta i) KO9 multiplies by -(eps/h) sin^10(theta/2) per axis; a unit spike at offset k along
    an axis returns eps/(1024 h) * (-1)^(k+1) C(10, 5+k) (a wrong coefficient or sign fails here)."""
    from math import comb
    n, g, eps, h = 16, 5, 0.1, 1.0 / 16
    i = np.arange(-g, n + g)
    for m in (1, 3, 8):
        theta = 2 * np.pi * m / n
        f = np.cos(theta * i)[None, None, :] * np.ones((n + 2 * g, n + 2 * g, 1))
        got = oracle.apply_op(oracle.OP_KO9, np.ascontiguousarray(f), g, 8, h, eps=eps)
        want = -(eps / h) * np.sin(theta / 2) ** 10 * f[g:-g, g:-g, g:-g]
        assert np.max(np.abs(got - want)) < 1e-13 * (eps / h)
    for axis in range(3):
        for k in range(-5, 6):
            z = np.zeros((3 + 2 * g,) * 3)
            q = [g + 1, g + 1, g + 1]
            q[axis] += k
            z[q[2], q[1], q[0]] = 1.0
            got = oracle.apply_op(oracle.OP_KO9, z, g, 8, h, eps=eps)[1, 1, 1]
            w = (-1) ** (abs(k) + 1) * comb(10, 5 + k)
            if k == 0:
                w *= 3      # the centre belongs to all three axes
            assert got == pytest.approx(eps / (1024.0 * h) * w, rel=1e-13)


def test_flat_field_gives_exact_zero(oracle):
    """difference form (reading R-H1): a constant field differentiates to exactly 0.0."""
    g = 5
    f = np.full((4 + 2 * g,) * 3, 1.0 + 2.0 ** -30)
    for order in (4, 8):
        for a in range(3):
            assert not oracle.apply_op(oracle.OP_D1, f, g, order, H, a=a).any()
            assert not oracle.apply_op(oracle.OP_UPW, f, g, order, H, a=a, b=1).any()
            assert not oracle.apply_op(oracle.OP_UPW, f, g, order, H, a=a, b=-1).any()
            for b in range(3):
                assert not oracle.apply_op(oracle.OP_DD, f, g, order, H, a=a, b=b).any()
    assert not oracle.apply_op(oracle.OP_KO, f, g, 4, H, eps=0.1).any()


def test_fill_ghosts_periodic(oracle):
    rng = np.random.default_rng(7)
    nx, ny, nz, g = 5, 4, 6, 3
    a = rng.standard_normal((2, nz, ny, nx))
    st = oracle.fill_ghosts(oracle.with_ghosts(a, g), g)
    want = np.stack([np.pad(a[v], g, mode="wrap") for v in range(2)])
    assert np.array_equal(st, want)
