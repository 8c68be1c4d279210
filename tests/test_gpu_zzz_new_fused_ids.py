"""The fused BSSN tile ids no GPU has run yet (5, 6, 7: DESIGN.md section 6.6), and the UNBOUNDED runtime sweep that may
pick them -- what bench.py's headline run does.  GPU access was closed for the whole round in which they were written;
what they have is the CTA emulator (tests/test_fused_kernel_emulated.py, tests/test_abi_emulated.py).  This file sorts
after every other `-m gpu` file: a device fault is sticky for the process, so under `pytest -x` a surprise here cannot
hide the tests of the kernels that ran green on hardware in round 1, nor round 2's tests on those kernels."""
import numpy as np
import pytest

from paper_1307_6488_b200 import inputs
from paper_1307_6488_b200.binding import NUM_TILES
from tests.test_gpu_a_parity import ROUND1_FUSED_IDS, TOL_BSSN_10_STEPS, assert_bssn_close, chem, relerr  # noqa: F401  (chem: fixture)
from tests.test_gpu_zz_round2 import CONFIGS4_GRIDS, config3_256_full_field, configs4_grid_sampled

pytestmark = pytest.mark.gpu


# ---- first the tests that survive a new id that is merely wrong (the sweep's guard disqualifies it), then the direct ones
_SWEEP = {}


def test_unbounded_sweep(chem, oracle):
    """chemora_autotune over every fused id: the later ids are timed, or disqualified by the guard (-2: disagrees with
    id 0, -3: a bounded wait gave up) -- never the pick if so; U untouched; two steps with the pick against the oracle"""
    n, dx, eps = 40, 0.05, 0.1
    h = chem.Chemora(n, n, n, 3, 4, chem.SYS_BSSN, dx)
    h.set_param("eps_diss", eps)
    u = inputs.bssn_noise(n, n, n)
    h.set_state(u)
    assert h.get_param("autotune_fused_ids") == chem.NUM_TILES
    fused, tile, ms = h.autotune()
    nt, ids = chem.NUM_TILES, chem.variants(chem.SYS_BSSN, 4)
    assert fused == 1 and tile in ids and ms[nt + tile] > 0
    assert all(ms[nt + t] > 0 for t in range(ROUND1_FUSED_IDS))
    assert all(ms[nt + t] > 0 or ms[nt + t] in (-2.0, -3.0) for t in ids), ms[nt:]
    assert np.array_equal(h.get_state(), u)
    for _ in range(2):
        h.rk4_step(0.25 * dx)
    st = oracle.rk4(1, oracle.with_ghosts(u, 3), 3, 4, dx, 0.25 * dx, oracle.params(eps_diss=eps), 2)
    assert_bssn_close(h.get_state(), oracle.interior(st, 3), 2e-11)
    h.destroy()
    _SWEEP["ms"] = ms[nt:]


@pytest.mark.parametrize("dims", CONFIGS4_GRIDS)
def test_configs4_grids_with_the_unbounded_sweeps_pick(oracle, dims):
    configs4_grid_sampled(oracle, dims, NUM_TILES, ())


def test_zzz_config3_256_full_field_with_the_unbounded_sweeps_pick(oracle):
    """bench.py's launch configuration when its sweep picks a new id: the whole 256^3 field after 10 steps against the
    oracle (whose result tests/test_gpu_zz_round2.py left in memory if it ran in this process).  If the pick is one of
    ids 0..4 that test has already covered it."""
    fused, tile, ran = config3_256_full_field(oracle, NUM_TILES, only_if_pick_at_least=ROUND1_FUSED_IDS)
    if not ran:
        pytest.skip("the unbounded sweep picks fused id %d at 256^3: covered by test_zz_bssn_config3_256_full_field_10_steps" % tile)


# ------------------------------------------- fused tile id 5: the interleaved section layout
@pytest.mark.parametrize("data", ["noise1e-10", "gaussians", "strong"])
def test_interleaved_layout_rhs_and_bit_identity(chem, oracle, data):
    """ids 5 and 6 against the oracle on ragged tiles, and against id 0 (same arithmetic, other section order) at rounding
    level: plain right-hand side and a whole RK4 step"""
    nx, ny, nz, g, dx, eps = 37, 22, 19, 3, 0.05, 0.1
    u = {"noise1e-10": lambda: inputs.bssn_noise(nx, ny, nz),
         "gaussians": lambda: inputs.bssn_gaussians(nx, ny, nz, width_cells=4.0),
         "strong": lambda: inputs.bssn_minkowski(nx, ny, nz) + 0.1 * np.random.default_rng(21).uniform(-1, 1, size=(25, nz, ny, nx))}[data]()
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    want = oracle.interior(oracle.rhs(oracle.SYS_BSSN, st, g, 4, dx, oracle.params(eps_diss=eps)), g)
    h = chem.Chemora(nx, ny, nz, g, 4, chem.SYS_BSSN, dx)
    h.set_param("eps_diss", eps)
    res = {}
    for tile in (0, 5, 6, 7):
        h.set_variant(1, tile)
        pad = h.new_state()
        h.interior(pad).copy_(__import__("torch").from_numpy(u))
        h.fill_ghosts(pad)
        out = h.new_state()
        h.rhs(pad, out)
        rhs = h.interior(out).cpu().numpy()
        assert relerr(rhs, want) < 1e-12, tile
        h.set_state(u)
        h.rk4_step(0.25 * dx)
        res[tile] = (rhs, h.get_state())
    # same arithmetic in another section order: bit-identical under the host emulator; on the device the compiler may
    # contract a product and a sum differently in the two instantiations, so the bar here is rounding level
    for tile in (5, 6, 7):
        assert relerr(res[tile][0], res[0][0]) < 1e-13 and relerr(res[tile][1], res[0][1]) < 1e-14, tile
    h.destroy()


@pytest.mark.parametrize("tile", [5, 6, 7])
def test_interleaved_layout_10_steps_and_rk3(chem, oracle, tile):
    nx, ny, nz, g, dx, eps = 24, 20, 18, 3, 0.05, 0.1
    dt = 0.25 * dx
    u0 = inputs.bssn_noise(nx, ny, nz)
    h = chem.Chemora(nx, ny, nz, g, 4, chem.SYS_BSSN, dx)
    h.set_param("eps_diss", eps)
    h.set_variant(1, tile)
    h.set_state(u0)
    for _ in range(10):
        h.rk4_step(dt)
    st = oracle.rk4(1, oracle.with_ghosts(u0, g), g, 4, dx, dt, oracle.params(eps_diss=eps), 10)
    assert_bssn_close(h.get_state(), oracle.interior(st, g), TOL_BSSN_10_STEPS)
    h.set_state(u0)
    for _ in range(10):
        h.rk3_step(dt)
        h.enforce_constraints()
    st = oracle.rk3(1, oracle.with_ghosts(u0, g), g, 4, dx, dt, oracle.params(eps_diss=eps), 10, True)
    assert_bssn_close(h.get_state(), oracle.interior(st, g), TOL_BSSN_10_STEPS)
    h.destroy()


def test_new_ids_10_steps_every_slot_moves(chem, oracle):
    """as test_bssn_rk4_10_steps_every_slot_moves (tests/test_gpu_zz_round2.py), for ids 5..7"""
    nx, ny, nz = 24, 20, 18
    u0 = inputs.bssn_gaussians(nx, ny, nz, width_cells=4.0)
    dx, dt, eps = 0.05, 0.0125, 0.1
    want = oracle.interior(oracle.rk4(1, oracle.with_ghosts(u0, 3), 3, 4, dx, dt, oracle.params(eps_diss=eps), 10), 3)
    assert all(np.max(np.abs(want[v] - u0[v])) > 1e-8 * max(np.max(np.abs(want[v])), 1e-300) for v in range(24))
    h = chem.Chemora(nx, ny, nz, 3, 4, 1, dx)
    h.set_param("eps_diss", eps)
    for tile in [t for t in chem.variants(chem.SYS_BSSN, 4) if t >= ROUND1_FUSED_IDS]:
        h.set_variant(1, tile)
        h.set_state(u0)
        for _ in range(10):
            h.rk4_step(dt)
        assert_bssn_close(h.get_state(), want, TOL_BSSN_10_STEPS)
    h.destroy()


def test_zzzz_no_new_id_was_disqualified_by_the_guard():
    """last of all: the sweep protects the results from a new id that disagrees with id 0 or whose waits give up, and
    the tests above pass without it -- but it is a defect of that kernel on hardware, and this is where it is reported"""
    if "ms" not in _SWEEP:
        pytest.skip("test_unbounded_sweep did not run")
    assert all(m > 0 or m == -1.0 for m in _SWEEP["ms"]), ("disqualified: -2 disagrees with id 0, -3 a wait gave up", _SWEEP["ms"])
