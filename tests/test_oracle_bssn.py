"""Pins O4-O8 for the oracle's BSSN right-hand side (readings S3-S6, S10).  None of them
re-uses oracle code: O5 is a closed form (Kasner), O6 a separately written linearisation on numpy rolls,
O7/O8 exact solutions of Einstein's equations (Schwarzschild in isotropic, Kerr in Kerr-Schild coordinates;
the latter built symbolically with sympy from the 4-metric alone) whose RHS must converge to 0 at 4th order.
CPU only."""
import numpy as np
import pytest

from paper_1307_6488_b200 import inputs

SYM = [[0, 1, 2], [1, 3, 4], [2, 4, 5]]


def rhs_periodic(oracle, u, g=3, order=4, h=0.05, **kw):
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    return oracle.interior(oracle.rhs(oracle.SYS_BSSN, st, g, order, h, oracle.params(**kw)), g)


# ------------------------------------------------------------------------------------------- O4
def test_O4_flat_stays_flat_bitwise(oracle):
    u = inputs.bssn_minkowski(8, 7, 9)
    r = rhs_periodic(oracle, u, eps_diss=0.1)
    assert not r.any()                         # RHS == 0 bitwise (+-0)
    st = oracle.with_ghosts(u, 3)
    oracle.rk4(oracle.SYS_BSSN, st, 3, 4, 0.05, 0.0125, oracle.params(eps_diss=0.1), 3)
    assert np.array_equal(oracle.interior(st, 3), u)


# ------------------------------------------------------------------------------------------- O5
def test_O5_kasner_algebraic_terms(oracle):
    """Kasner at t=1, p=(-1/3,2/3,2/3): gt=delta, chi=1, alpha=1, K=-1, At=diag(1/3-p_i); homogeneous."""
    p = np.array([-1.0 / 3, 2.0 / 3, 2.0 / 3])
    u = inputs.bssn_minkowski(6, 6, 6)
    u[7] = -1.0
    A = 1.0 / 3 - p
    u[8], u[11], u[13] = A[0], A[1], A[2]
    r = rhs_periodic(oracle, u, eps_diss=0.1)
    want = np.zeros(25)
    want[0] = -2.0 / 3                         # d_t chi = 2/3 chi alpha K
    want[7] = 1.0                              # d_t K = At_ij At^ij + K^2/3 = sum(1/3-p_i)^2 + 1/3 = 1
    for i, s in enumerate((1, 4, 6)):
        want[s] = -2.0 * A[i]                  # d_t gt_ii = -2 alpha At_ii
    for i, s in enumerate((8, 11, 13)):
        want[s] = -A[i] - 2.0 * A[i] ** 2      # d_t At_ii = alpha (K At_ii - 2 At_ik At^k_i)
    want[17] = 2.0                             # d_t alpha = -2 alpha K
    for v in range(25):
        assert np.max(np.abs(r[v] - want[v])) < 2e-15, inputs.BSSN_NAMES[v]


# ------------------------------------------------------------------------------------------- O6
def _roll(f, axis, m):          # value at offset +m along axis (0=x,1=y,2=z) on a periodic array [z,y,x]
    return np.roll(f, -m, axis=2 - axis)


ORDER = [4]                     # FD order the linearised evaluator uses (set by the O6 tests)
KO_ORDER = [5]                  # dissipation order it uses (S6; 9 = S6b)


def _d1(f, a, h):
    e = [_roll(f, a, m) - _roll(f, a, -m) for m in range(5)]
    if ORDER[0] == 4:
        return (8 * e[1] - e[2]) / (12 * h)
    return (672 * e[1] - 168 * e[2] + 32 * e[3] - 3 * e[4]) / (840 * h)


def _dd(f, a, b, h):
    if a != b:
        return _d1(_d1(f, a, h), b, h)
    s = [_roll(f, a, m) + _roll(f, a, -m) for m in range(5)]
    if ORDER[0] == 4:
        return (-30 * f + 16 * s[1] - s[2]) / (12 * h * h)
    return (-14350 * f + 8064 * s[1] - 1008 * s[2] + 128 * s[3] - 9 * s[4]) / (5040 * h * h)


def _ko(f, eps, h):
    s = 0
    if KO_ORDER[0] == 9:
        w = (210, -120, 45, -10, 1)
        for a in range(3):
            s = s - 252 * f
            for m in range(1, 6):
                s = s + w[m - 1] * (_roll(f, a, m) + _roll(f, a, -m))
        return eps * s / (1024 * h)
    for a in range(3):
        s = s + (_roll(f, a, 3) + _roll(f, a, -3) - 6 * (_roll(f, a, 2) + _roll(f, a, -2))
                 + 15 * (_roll(f, a, 1) + _roll(f, a, -1)) - 20 * f)
    return eps * s / (64 * h)


def linearised_rhs(u, h, eps, eta):
    """BSSN linearised about Minkowski (alpha=1+a, chi=1+c, gt=delta+hh); advection is 2nd order."""
    bg = inputs.bssn_minkowski(*u.shape[:0:-1])
    p = u - bg                                 # exact (Sterbenz): perturbations
    c, K, a = p[0], p[7], p[17]
    hh = lambda i, j: p[1 + SYM[i][j]]
    At = lambda i, j: p[8 + SYM[i][j]]
    Gt, beta, B = p[14:17], p[18:21], p[21:24]
    lap = lambda f: _dd(f, 0, 0, h) + _dd(f, 1, 1, h) + _dd(f, 2, 2, h)
    divb = _d1(beta[0], 0, h) + _d1(beta[1], 1, h) + _d1(beta[2], 2, h)
    r = np.zeros_like(u)
    r[0] = 2.0 / 3 * (K - divb)
    r[7] = -lap(a)
    r[17] = -2 * K
    X = [[None] * 3 for _ in range(3)]
    for i in range(3):
        for j in range(i, 3):
            d = 1.0 if i == j else 0.0
            r[1 + SYM[i][j]] = -2 * At(i, j) + _d1(beta[j], i, h) + _d1(beta[i], j, h) - 2.0 / 3 * d * divb
            R = (-0.5 * lap(hh(i, j)) + 0.5 * (_d1(Gt[j], i, h) + _d1(Gt[i], j, h))
                 + 0.5 * (_dd(c, i, j, h) + d * lap(c)))
            X[i][j] = X[j][i] = -_dd(a, i, j, h) + R
    tr = X[0][0] + X[1][1] + X[2][2]
    for i in range(3):
        for j in range(i, 3):
            r[8 + SYM[i][j]] = X[i][j] - (tr / 3 if i == j else 0.0)
    for i in range(3):
        ddiv = sum(_dd(beta[k], i, k, h) for k in range(3))
        r[14 + i] = -4.0 / 3 * _d1(K, i, h) + lap(beta[i]) + ddiv / 3
        r[18 + i] = 0.75 * B[i]
        r[21 + i] = r[14 + i] - eta * B[i]
    for v in range(25):
        r[v] = r[v] + _ko(p[v], eps, h)
    return r


@pytest.mark.parametrize("order,g,ko_order", [(4, 3, 5), (8, 5, 5), (8, 5, 9)])
def test_O6_linearised_bssn_on_config2_data(oracle, order, g, ko_order):
    """order 8 with 5 ghost zones is the paper's own configuration; ko_order 9 is S6b"""
    n, h, eps, eta = 16, 0.05, 0.1, 1.0
    u = inputs.bssn_noise(n, n, n, amp=1e-10)
    got = rhs_periodic(oracle, u, g=g, order=order, h=h, eps_diss=eps, eta=eta, ko_order=ko_order)
    ORDER[0], KO_ORDER[0] = order, ko_order
    try:
        want = linearised_rhs(u, h, eps, eta)
    finally:
        ORDER[0], KO_ORDER[0] = 4, 5
    for v in range(25):
        scale = np.max(np.abs(want[v]))
        assert scale > 0
        assert np.max(np.abs(got[v] - want[v])) < 2e-8 * scale, inputs.BSSN_NAMES[v]


def test_O6_sensitivity(oracle):
    """the linear pin really discriminates: at amplitude 1e-5 the quadratic terms are visible."""
    u = inputs.bssn_noise(8, 8, 8, amp=1e-5)
    got = rhs_periodic(oracle, u)
    want = linearised_rhs(u, 0.05, 0.0, 1.0)
    worst = max(np.max(np.abs(got[v] - want[v])) / np.max(np.abs(want[v])) for v in range(24))
    assert 1e-7 < worst < 1e-2


# ------------------------------------------------------------------------------------------- O7
def _box(n, g, lo, length):
    h = length / n
    idx = lo + h * np.arange(-g, n + g, dtype=np.float64)
    Z, Y, X = np.meshgrid(idx, idx, idx, indexing="ij")
    return X, Y, Z, h


def test_O7_schwarzschild_isotropic_static(oracle):
    """chi = psi^-4, psi = 1 + M/2r, alpha = (1 - M/2r)/psi, gt = delta, rest 0 (analytic ghosts):
    d_t K and d_t At_ij -> 0 at 4th order; d_t chi, d_t gt, d_t Gt, d_t beta are exactly 0."""
    M, g = 1.0, 3
    errs = []
    for n in (8, 16, 32):
        X, Y, Z, h = _box(n, g, 1.1, 1.0)
        r = np.sqrt(X * X + Y * Y + Z * Z)
        psi = 1 + M / (2 * r)
        u = np.zeros((25,) + r.shape)
        u[0] = psi ** -4
        u[1] = u[4] = u[6] = 1.0
        u[17] = (1 - M / (2 * r)) / psi
        rhs = oracle.interior(oracle.rhs(oracle.SYS_BSSN, u, g, 4, h, oracle.params()), g)
        assert not rhs[0].any() and not rhs[1:7].any() and not rhs[18:21].any()
        errs.append(max(np.max(np.abs(rhs[7])), np.max(np.abs(rhs[8:14]))))
        # the pieces that cancel are not small: D_i D_j alpha ~ M/r^3
        assert errs[-1] < 1e-3
    assert errs[0] / errs[1] == pytest.approx(16.0, rel=0.35)
    assert errs[1] / errs[2] == pytest.approx(16.0, rel=0.15)
    assert errs[2] < 2e-7


# ------------------------------------------------------------------------------------------- O8
# constant, non-orthogonal linear change of spatial coordinates x_KS = L x: the solution stays exact and
# stationary but loses its manifest spherical symmetry, so antisymmetric / off-diagonal index mistakes
# (which a spherically symmetric field hides) show up.
SHEAR = [[1, "1/5", 0], ["-1/10", 1, "3/10"], ["1/10", 0, "9/10"]]
SPIN = "3/5"   # Kerr, a = 0.6 M: no spherical symmetry left (a = 0 is Schwarzschild)


@pytest.fixture(scope="module")
def kerr_schild():
    """BSSN variables of Kerr (a = 0.6 M) in (sheared) Kerr-Schild coordinates, derived symbolically from
    gamma_ab = delta_ab + 2H l_a l_b, alpha = (1+2H)^(-1/2), beta^a = 2H/(1+2H) l^a, pulled back
    through x_KS = L x, with K_ij from d_t gamma_ij = 0  (K_ij = (D_i beta_j + D_j beta_i) / 2 alpha) and
    Gt^i = -d_j gtu^{ij} (det gt = 1).  Nothing here comes from the oracle."""
    import sympy as sp
    x, y, z = sp.symbols("x y z", real=True)
    X = [x, y, z]
    L = sp.Matrix(3, 3, lambda i, j: sp.Rational(SHEAR[i][j]))
    Linv = L.inv()
    xo = L * sp.Matrix(X)                                   # Kerr-Schild coordinates of the point
    a = sp.Rational(SPIN)
    rho2 = sum(c * c for c in xo)
    r = sp.sqrt((rho2 - a * a) / 2 + sp.sqrt((rho2 - a * a) ** 2 / 4 + a * a * xo[2] ** 2))
    H = r ** 3 / (r ** 4 + a * a * xo[2] ** 2)              # M = 1
    l = [(r * xo[0] + a * xo[1]) / (r * r + a * a), (r * xo[1] - a * xo[0]) / (r * r + a * a), xo[2] / r]
    gam_o = sp.Matrix(3, 3, lambda a, b: (1 if a == b else 0) + 2 * H * l[a] * l[b])
    gamu_o = sp.Matrix(3, 3, lambda a, b: (1 if a == b else 0) - 2 * H * l[a] * l[b] / (1 + 2 * H))
    betau_o = sp.Matrix([2 * H / (1 + 2 * H) * l[a] for a in range(3)])
    alpha = 1 / sp.sqrt(1 + 2 * H)
    gam = L.T * gam_o * L                                   # gamma_ij = L^a_i L^b_j gamma_ab
    gamu = Linv * gamu_o * Linv.T
    betau = Linv * betau_o
    betad = gam * betau
    Gam = [[[sum(gamu[k, m] * (sp.diff(gam[m, i], X[j]) + sp.diff(gam[m, j], X[i]) - sp.diff(gam[i, j], X[m]))
                 for m in range(3)) / 2 for j in range(3)] for i in range(3)] for k in range(3)]
    Dbeta = [[sp.diff(betad[j], X[i]) - sum(Gam[k][i][j] * betad[k] for k in range(3)) for j in range(3)]
             for i in range(3)]
    Kij = sp.Matrix(3, 3, lambda i, j: (Dbeta[i][j] + Dbeta[j][i]) / (2 * alpha))
    detg = (1 + 2 * H) * L.det() ** 2
    chi = detg ** sp.Rational(-1, 3)
    trK = sum(gamu[i, j] * Kij[i, j] for i in range(3) for j in range(3))
    gt = chi * gam
    gtu = gamu / chi
    At = chi * (Kij - gam * trK / 3)
    Gt = [-sum(sp.diff(gtu[i, j], X[j]) for j in range(3)) for i in range(3)]
    exprs = [chi] + [gt[i, j] for i in range(3) for j in range(i, 3)] + [trK] + \
            [At[i, j] for i in range(3) for j in range(i, 3)] + Gt + [alpha] + list(betau)
    return sp.lambdify((x, y, z), exprs, modules="numpy", cse=True)


def test_O8_kerr_kerr_schild_stationary(oracle, kerr_schild):
    """Everything at once (non-flat gt, At ~ 0.4, K ~ 0.6, non-zero shift => upwinded advection,
    R~_ij, Christoffels): RHS of chi, gt, K, At, Gt -> 0 at 4th order."""
    g = 3
    errs = []
    for n in (8, 16, 32):
        # off-axis box, beta^x,y > 0 and beta^z < 0 there: both upwind sides are exercised
        idx = lambda lo, h: lo + h * np.arange(-g, n + g, dtype=np.float64)
        h = 1.0 / n
        Z, Y, X = np.meshgrid(idx(-1.9, h), idx(0.7, h), idx(1.3, h), indexing="ij")
        vals = kerr_schild(X, Y, Z)
        u = np.zeros((25,) + X.shape)
        for v, a in enumerate(vals):
            u[v] = a
        assert u[20].max() < 0 < u[18].min()
        rhs = oracle.interior(oracle.rhs(oracle.SYS_BSSN, u, g, 4, h, oracle.params()), g)
        e = [np.max(np.abs(rhs[v])) for v in range(17)]
        errs.append(e)
    errs = np.array(errs)
    ratio1, ratio2 = errs[0] / errs[1], errs[1] / errs[2]
    for v in range(17):
        assert errs[2, v] < 3e-6, inputs.BSSN_NAMES[v]
        assert 10.0 < ratio2[v] < 40.0, (inputs.BSSN_NAMES[v], ratio1[v], ratio2[v])
    # sanity: the data is not trivial
    assert np.max(np.abs(u[8:14])) > 0.1 and np.max(np.abs(u[7])) > 0.1


# ------------------------------------------------------------------------------- S2: upwind side
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [+1.0, -1.0])
def test_advection_side_follows_sign_of_shift(oracle, axis, sign):
    """S2: beta^k > 0 uses offsets -1..+3, beta^k < 0 offsets -3..+1.  A spike in trK three cells away
    on the upwind side is seen through beta^k d_k K with coefficient beta/(12h); on the other side not."""
    n, g, h, b = 9, 3, 0.05, 0.3
    for where, expect in ((+3, True), (-3, False)):
        u = inputs.bssn_minkowski(n, n, n)
        u[18 + axis] = sign * b
        q = [4, 4, 4]
        q[axis] += int(sign) * where
        u[7][q[2], q[1], q[0]] = 1.0
        r = rhs_periodic(oracle, u, h=h, eps_diss=0.0)
        got = r[7][4, 4, 4]
        if expect:
            assert got == pytest.approx(sign * b * sign / (12 * h), rel=1e-13)
        else:
            assert got == 0.0


# ------------------------------------------------------- S5: advection of the gauge variables (task 2)
def _up_symbol(theta, sign, order, h):
    """Fourier symbol of the one-sided advection stencil of reading S2 on e^{i theta j}: offsets -1..+3 (O4) or
    -3..+5 (O8) for a positive shift, the mirror image (coefficients negated) for a negative one."""
    if order == 4:
        off, c, den = np.arange(-1, 4), np.array([-3.0, -10.0, 18.0, -6.0, 1.0]), 12.0
    else:
        off, c, den = np.arange(-3, 6), np.array([-5.0, 60.0, -420.0, -378.0, 1050.0, -420.0, 140.0, -30.0, 3.0]), 840.0
    if sign < 0:
        off, c = -off, -c
    return np.sum(c * np.exp(1j * theta * off)) / (den * h)


def _d2_symbol(theta, order, h):
    if order == 4:
        return (-30.0 + 32.0 * np.cos(theta) - 2.0 * np.cos(2 * theta)) / (12.0 * h * h)
    return (-14350.0 + 2 * (8064.0 * np.cos(theta) - 1008.0 * np.cos(2 * theta) + 128.0 * np.cos(3 * theta)
                            - 9.0 * np.cos(4 * theta))) / (5040.0 * h * h)


@pytest.mark.parametrize("order,g", [(4, 3), (8, 5)])
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [+1.0, -1.0])
def test_gauge_advection_closed_form(oracle, order, g, axis, sign):
    """Flat space, uniform shift beta^axis = +-c, one Fourier mode (along `axis`) in alpha, then in each beta^i, then
    in each B^i: every term of the gauge right-hand sides (slots 17..23, reading S5) is then a closed form --
        d_t alpha = c D^up alpha + KO;   d_t beta^i = 3/4 B^i + beta^k D^up_k beta^i + KO;
        d_t B^i = [d_j d_j beta^i + 1/3 d_i d_k beta^k] - eta B^i + c D^up B^i + KO
    with D^up's symbol (one-sided, side by the sign of the shift), the centred second-derivative symbol and
    -(eps/h) sin^6(theta/2) for the dissipation.  A dropped adv(21+a), an advection of B^i with another slot, the
    wrong side or a wrong axis all fail here (they pass O4..O8, where the shift is zero, linear or only the tensor
    slots are checked)."""
    n, h, c, A, eps, eta, sgc = 10, 0.05, 0.3, 1e-3, 0.1, 1.3, 0.6
    m, phase = 3, 0.7
    theta = 2 * np.pi * m / n
    idx = np.arange(n)
    shape = [1, 1, 1]
    shape[2 - axis] = n                      # arrays are [z, y, x]
    wave = np.cos(theta * idx + phase).reshape(shape) * np.ones((n, n, n))
    up, d2 = _up_symbol(theta, sign, order, h), _d2_symbol(theta, order, h)
    ko = -(eps / h) * np.sin(theta / 2) ** 6

    def apply(symbol):                       # symbol applied to A cos(theta j + phase)
        z = A * symbol * np.exp(1j * (theta * idx + phase))
        return z.real.reshape(shape) * np.ones((n, n, n))

    for slot in [17] + [18 + i for i in range(3)] + [21 + i for i in range(3)]:
        u = inputs.bssn_minkowski(n, n, n)
        u[18 + axis] = sign * c
        u[slot] = u[slot] + A * wave
        st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
        r = oracle.interior(oracle.rhs(oracle.SYS_BSSN, st, g, order, h,
                                       oracle.params(eps_diss=eps, eta=eta, shift_gamma_coeff=sgc)), g)
        want = {v: np.zeros((n, n, n)) for v in range(17, 24)}
        if slot == 17:
            want[17] = sign * c * apply(up) + apply(ko)
        elif slot < 21:
            i = slot - 18
            want[slot] = u[18 + axis] * apply(up) + apply(ko)       # beta^axis itself carries the mode when i == axis
            want[21 + i] = apply(d2) + (apply(d2) / 3.0 if i == axis else 0.0)      # d_t Gt^i|_0 of flat space
        else:
            i = slot - 21
            want[18 + i] = sgc * A * wave
            want[slot] = -eta * A * wave + sign * c * apply(up) + apply(ko)
        for v in range(17, 24):
            scale = max(np.max(np.abs(want[v])), A)
            assert np.max(np.abs(r[v] - want[v])) < 1e-13 * scale * (4 if order == 8 else 1), (slot, v)
