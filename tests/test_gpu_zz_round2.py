"""Parity tests added in round 2 (VERDICT r1 "what's missing" 2-4 and task 3): whole-field 256^3 for
10 steps, the configs[4] grids, 10-step runs in which every slot moves, the radiative outer boundary.  GPU access was
closed while they were written, so they sort after the files whose tests ran green on hardware in round 1: under
`pytest -x` a surprise here cannot hide those.  Everything in this file runs on kernels that ran on hardware in round 1
(runtime sweeps bounded to fused ids 0..4 by "autotune_fused_ids") plus the radiative face kernel; the fused ids no
GPU has run yet (5..7) have a file of their own that sorts after this one (tests/test_gpu_zzz_new_fused_ids.py), which
repeats the sweeping tests here with the unbounded sweep.  All need a B200: `pytest -m gpu`."""
import numpy as np
import pytest

from paper_1307_6488_b200 import inputs
from tests.test_gpu_a_parity import ROUND1_FUSED_IDS, TOL_BSSN_10_STEPS, assert_bssn_close, chem, relerr  # noqa: F401  (chem: fixture)
from tests.test_gpu_z_fullsize import check_samples, cut

pytestmark = pytest.mark.gpu


CONFIGS4_GRIDS = [(96, 96, 96), (160, 160, 160), (200, 200, 400)]


@pytest.mark.parametrize("dims", CONFIGS4_GRIDS)
def test_bssn_configs4_grids_sampled(oracle, dims):
    configs4_grid_sampled(oracle, dims, ROUND1_FUSED_IDS, ((0, 1),))


def configs4_grid_sampled(oracle, dims, fused_ids, also):
    """configs[4]'s own grids (96^3, 160^3 and 200 x 200 x 400, whose 206-column rows sit in a 208-double pitch: the
    padding case): configs[2] data, 2 RK4 steps with the variant the runtime sweep picks -- what bench.py --sweep
    times -- and with one split tile, sampled against the oracle; both norms of DESIGN.md S11 / S11b, pro-rated
    2/10 of the 10-step tolerance."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1307_6488_b200 import binding
    nx, ny, nz = dims
    g, dx, eps = 3, 0.05, 0.1
    dt, steps = 0.25 * dx, 2
    u0 = inputs.bssn_noise(nx, ny, nz, seed=13076488 + 4)
    h = binding.Chemora(nx, ny, nz, g, 4, binding.SYS_BSSN, dx)
    h.set_param("eps_diss", eps)
    h.set_state(u0)
    h.set_param("autotune_fused_ids", fused_ids)
    fused, tile, _ = h.autotune()
    assert fused == 1 and tile < fused_ids
    rng = np.random.default_rng(9)
    centres = [(0, 0, 0), (nx - 1, ny // 2, 3), (nx - 3, ny - 2, nz - 1)] + \
              [tuple(int(rng.integers(0, m)) for m in (nx, ny, nz)) for _ in range(2)]
    for f, t in ((fused, tile),) + tuple(also):
        h.set_variant(f, t)
        h.set_state(u0)
        for _ in range(steps):
            h.rk4_step(dt)
        got = h.get_state()
        check_samples(oracle, oracle.SYS_BSSN, u0, got, centres, reach=12 * steps, core=4, g=g, order=4, dx=dx, dt=dt,
                      prm=oracle.params(eps_diss=eps), steps=steps, tol=2e-11)
        # background-subtracted norm on the O(1) slots (chi, gt11, gt22, gt33, alpha), same samples
        reach, core = 12 * steps, 4
        for c in centres:
            blk = cut(u0, c, core + reach)
            st = oracle.rk4(oracle.SYS_BSSN, oracle.with_ghosts(blk, g), g, 4, dx, dt, oracle.params(eps_diss=eps), steps)
            want = oracle.interior(st, g)[:, reach:reach + 2 * core, reach:reach + 2 * core, reach:reach + 2 * core]
            have = cut(got, c, core)
            for v in (0, 1, 4, 6, 17):
                amp = float(np.max(np.abs(got[v] - 1.0)))
                err = float(np.max(np.abs((have[v] - 1.0) - (want[v] - 1.0))))
                assert err < max(2e-11, 8 * 2.220446049250313e-16 / amp) * amp, (f, t, c, v, err, amp)
    h.destroy()
    return fused, tile


def test_zz_bssn_config3_256_full_field_10_steps(oracle):
    """north_star's sentence as written: BSSN 256^3 (configs[3]: Minkowski + 1e-4 Gaussians), 4th order + upwind + KO,
    10 RK4 steps, the WHOLE field against the oracle on all host cores, S11 < 1e-10 and the background-subtracted norm
    of S11b on the O(1) slots.  About 4-5 minutes of host time and 20 GB of host memory."""
    config3_256_full_field(oracle, ROUND1_FUSED_IDS)


_ORACLE_256 = {}     # the oracle's 10 steps at 256^3 (3.6 GB), kept for tests/test_gpu_zzz_new_fused_ids.py


def config3_256_full_field(oracle, fused_ids, only_if_pick_at_least=0):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1307_6488_b200 import binding
    c = inputs.config(3)
    n, g, dx = 256, c["ghost"], c["dx"]
    dt, steps = 0.25 * dx, 10
    u0 = c["state"]()
    h = binding.Chemora(n, n, n, g, c["order"], binding.SYS_BSSN, dx)
    h.set_param("eps_diss", c["eps_diss"])
    h.set_state(u0)
    h.set_param("autotune_fused_ids", fused_ids)
    fused, tile, _ = h.autotune()                       # what bench.py does
    assert fused == 1 and tile < fused_ids
    if tile < only_if_pick_at_least:
        h.destroy()
        return fused, tile, False
    for _ in range(steps):
        h.rk4_step(dt)
    got = h.get_state()
    h.destroy()
    if "st" not in _ORACLE_256:
        _ORACLE_256["st"] = oracle.rk4(oracle.SYS_BSSN, oracle.with_ghosts(u0, g), g, 4, dx, dt,
                                       oracle.params(eps_diss=c["eps_diss"]), steps)
    st = _ORACLE_256["st"]
    del u0
    worst = 0.0
    for v in range(25):
        want = st[v, g:-g, g:-g, g:-g]
        den = float(np.max(np.abs(want)))
        err = float(np.max(np.abs(got[v] - want)))
        if den == 0.0:
            assert err == 0.0, v
            continue
        worst = max(worst, err / den)
        if v in (0, 1, 4, 6, 17):
            amp = float(np.max(np.abs(want - 1.0)))
            ebg = float(np.max(np.abs((got[v] - 1.0) - (want - 1.0))))
            assert ebg < max(1e-10, 8 * 2.220446049250313e-16 / amp) * amp, (v, ebg, amp)
    assert worst < 1e-10, worst
    return fused, tile, True


@pytest.mark.parametrize("data", ["gaussians", "strong"])
def test_bssn_rk4_10_steps_every_slot_moves(chem, oracle, data):
    """10 RK4 steps on data where every slot evolves by far more than 1e-10 of its size (Gaussians of amplitude 1e-4;
    0.02-amplitude strong field), every fused tile id and one split tile: 1e-10 is then meaningful on all 25 slots"""
    nx, ny, nz = 24, 20, 18
    u0 = inputs.bssn_gaussians(nx, ny, nz, width_cells=4.0) if data == "gaussians" else \
        inputs.bssn_minkowski(nx, ny, nz) + 0.02 * np.random.default_rng(23).uniform(-1, 1, size=(25, nz, ny, nx))
    dx, dt, eps = 0.05, 0.0125, 0.1
    st = oracle.rk4(1, oracle.with_ghosts(u0, 3), 3, 4, dx, dt, oracle.params(eps_diss=eps), 10)
    want = oracle.interior(st, 3)
    assert all(np.max(np.abs(want[v] - u0[v])) > 1e-8 * max(np.max(np.abs(want[v])), 1e-300) for v in range(24))
    h = chem.Chemora(nx, ny, nz, 3, 4, 1, dx)
    h.set_param("eps_diss", eps)
    for fused, tile in [(1, t) for t in chem.variants(chem.SYS_BSSN, 4) if t < 5] + [(0, 1)]:
        h.set_variant(fused, tile)
        h.set_state(u0)
        for _ in range(10):
            h.rk4_step(dt)
        assert_bssn_close(h.get_state(), want, TOL_BSSN_10_STEPS)
    h.destroy()


# ------------------------------------------------- radiative outer boundary, reading S16 (second half)
@pytest.mark.parametrize("system,order,g,dims", [(0, 4, 2, (19, 11, 9)), (0, 8, 4, (37, 9, 12)), (1, 4, 3, (21, 12, 10)),
                                                 (2, 4, 3, (9, 33, 8))])
def test_radiative_rhs_at_boundary_points(chem, oracle, system, order, g, dims):
    """the face kernel against the oracle at every boundary point (faces, edges, corners), interior untouched"""
    nx, ny, nz = dims
    V = {0: 2, 1: 25, 2: 5}[system]
    st = np.random.default_rng(51).standard_normal((V, nz + 2 * g, ny + 2 * g, nx + 2 * g))
    dx = 0.07
    want = oracle.radiative_rhs(system, st, g, dx)
    h = chem.Chemora(nx, ny, nz, g, order, system, dx)
    h.set_state_ghosted(st)
    assert np.array_equal(h.get_state_ghosted(), st)                 # the ghosted copies are bit-exact
    out = h.new_state()
    out.fill_(7.0)
    h.radiative_rhs(h.state_view(), out)
    got = h.ghosted(out).cpu().numpy()
    m = np.ones(got.shape[1:], dtype=bool)
    m[g:-g, g:-g, g:-g] = False
    for v in range(V):
        assert np.max(np.abs(got[v][m] - want[v][m])) < 1e-12 * np.max(np.abs(want[v][m])), v
    assert (got[:, ~m] == 7.0).all()
    h.destroy()


@pytest.mark.parametrize("system,order,g,steps,tol", [(0, 4, 2, 10, 1e-11), (2, 8, 4, 5, 5e-12), (1, 4, 3, 10, 1e-10)])
def test_radiative_rk4_whole_block(chem, oracle, system, order, g, steps, tol):
    """RK4 with radiative boundaries: the whole padded block (interior and evolved boundary points) against the
    oracle; the BSSN case on configs[2]-like data with both norms"""
    nx, ny, nz = 22, 18, 13
    dx = 0.05
    dt = 0.25 * dx
    V = {0: 2, 1: 25, 2: 5}[system]
    rng = np.random.default_rng(52)
    if system == 1:
        st = oracle.fill_ghosts(oracle.with_ghosts(inputs.bssn_noise(nx, ny, nz), g), g)
        st += 1e-10 * rng.uniform(-1, 1, size=st.shape)
    else:
        st = rng.standard_normal((V, nz + 2 * g, ny + 2 * g, nx + 2 * g))
    prm = oracle.params(eps_diss=0.1 if g >= 3 else 0.0)
    h = chem.Chemora(nx, ny, nz, g, order, system, dx)
    h.set_param("eps_diss", 0.1 if g >= 3 else 0.0)
    h.set_boundary(chem.BC_RADIATIVE)
    assert h.get_boundary() == chem.BC_RADIATIVE
    h.set_state_ghosted(st)
    for _ in range(steps):
        h.rk4_step(dt)
    got = h.get_state_ghosted()
    want = oracle.rk4_radiative(system, st.copy(), g, order, dx, dt, prm, steps)
    if system == 1:
        assert_bssn_close(got, want, tol)
    else:
        assert relerr(got, want) < tol
    with pytest.raises(chem.ChemoraError):
        h.link_z(h, h)                                      # radiative blocks are not z-linked
    h.destroy()
