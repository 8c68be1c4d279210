"""The fused BSSN kernel's SOURCE, executed on the host (no GPU needed): csrc/kernels_bssn_tma.cu is compiled by g++
with -DCHM_EMULATE on top of tests/native/cta_emu.hpp (one OS thread per CUDA thread; real barriers; mbarriers with
the PTX phase/parity/transaction-count semantics; TMA tile loads as synchronous box copies with zero fill) and run
over small periodic blocks with ragged tiles and several tiles per persistent CTA.

What this covers that the host arithmetic test does not: the fused kernel's own transcription of the right-hand side
(its section order and folding), the 5-slot (8th order: 3-slot) box ring with its parities, the warp-wise slot
release and refill, the point-value and Runge-Kutta operand tiles, the two-pass mixed derivatives with their plane
barriers, the At_ij loop and its table, every Runge-Kutta epilogue.  What it cannot cover: hardware timing, and memory
ordering below the emulator's barriers -- the -m gpu parity tests remain the proof on the device.
The device build of the same file is byte-identical in SASS to the one before the emulation hooks went in."""
import os
import subprocess

import numpy as np
import pytest

from paper_1307_6488_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MODE_RHS, MODE_FIRST, MODE_MID, MODE_LAST, MODE_SSP = range(5)


@pytest.fixture(scope="module")
def emu():
    from tests.conftest import build_emulator
    return build_emulator("fused_emu")


def launch(exe, tmp, order, tile, mode, st_in, U, S, g, h, eps, a=0.0, ca=0.0, cb=0.0, grid=3, eta=1.0, sgc=0.75,
           ko_order=5):
    """one emulated launch; returns (out, S, U) as ghosted arrays and the statistics line"""
    V, tz, ty, tx = st_in.shape
    paths = [str(tmp / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
    for arr, p in zip((st_in, U, S), paths):
        np.ascontiguousarray(arr).tofile(p)
    r = subprocess.run([exe, str(order), str(tile), str(mode), str(tx - 2 * g), str(ty - 2 * g), str(tz - 2 * g), str(g),
                        repr(h), repr(eps), repr(eta), repr(sgc), str(ko_order), repr(a), repr(ca), repr(cb), str(grid)]
                       + paths, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    words = r.stdout.split()
    assert words[0] == "err" and int(words[1]) == 0, r.stdout          # no bounded wait gave up
    out = np.fromfile(paths[3]).reshape(3, V, tz, ty, tx)
    return out[0], out[1], out[2], dict(loads=int(words[3]), bytes=int(words[5]))


def relerr(a, b):
    return max(np.max(np.abs(a[v] - b[v])) / max(np.max(np.abs(b[v])), 1e-300) for v in range(a.shape[0]))


def strong(nx, ny, nz, seed=21, amp=0.1):
    return inputs.bssn_minkowski(nx, ny, nz) + amp * np.random.default_rng(seed).uniform(-1, 1, size=(25, nz, ny, nx))


@pytest.mark.parametrize("order,g,tile,dims,grid", [(4, 3, 0, (20, 9, 6), 3), (4, 3, 1, (20, 9, 6), 2), (4, 3, 3, (17, 5, 11), 1),
                                                    (4, 4, 0, (18, 6, 5), 2), (8, 5, 0, (19, 6, 7), 2),
                                                    (4, 3, 5, (20, 9, 6), 3), (4, 4, 5, (18, 6, 9), 1), (4, 3, 6, (20, 9, 6), 2), (4, 3, 7, (20, 9, 6), 3), (4, 4, 7, (18, 6, 9), 1)])
@pytest.mark.parametrize("data", ["strong", "noise1e-10"])
def test_rhs_against_the_oracle(oracle, emu, tmp_path, order, g, tile, dims, grid, data):
    nx, ny, nz = dims
    u = strong(nx, ny, nz) if data == "strong" else inputs.bssn_noise(nx, ny, nz)
    h, eps = 0.05, 0.1
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    z = np.zeros_like(st)
    out, _, _, stats = launch(emu, tmp_path, order, tile, MODE_RHS, st, z, z, g, h, eps, grid=grid, eta=1.3, sgc=0.6)
    want = oracle.rhs(oracle.SYS_BSSN, st, g, order, h, oracle.params(eps_diss=eps, eta=1.3, shift_gamma_coeff=0.6))
    assert relerr(oracle.interior(out, g), oracle.interior(want, g)) < 1e-12
    m = np.ones(out.shape[1:], dtype=bool)
    m[g:-g, g:-g, g:-g] = False
    assert not out[:, m].any()                                  # nothing is written outside the interior
    tx, ty, tz = {0: (16, 4, 4), 1: (16, 8, 2), 3: (16, 2, 8), 5: (16, 4, 4), 6: (16, 4, 4), 7: (16, 4, 4)}[tile]
    ntiles = -(-nx // tx) * -(-ny // ty) * -(-nz // tz)
    assert stats["loads"] == ntiles * (25 + 3)                  # one box per section + three point-value groups


def test_interleaved_layout_is_bit_identical_to_the_plain_one(oracle, emu, tmp_path):
    """tile id 5 evaluates the arithmetic of tile id 0 in another section order: a middle RK4 stage gives the same bits
    (Y and S), and loads the same boxes plus the same operand tiles in fewer, larger requests"""
    nx, ny, nz, g, h, eps = 20, 9, 6, 3, 0.05, 0.1
    st = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz), g), g)
    U = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz, seed=7), g), g)
    S = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz, seed=8), g), g)
    a0 = launch(emu, tmp_path, 4, 0, MODE_MID, st, U, S, g, h, eps, a=0.00625)
    a5 = launch(emu, tmp_path, 4, 5, MODE_MID, st, U, S, g, h, eps, a=0.00625)
    a6 = launch(emu, tmp_path, 4, 6, MODE_MID, st, U, S, g, h, eps, a=0.00625)
    assert np.array_equal(a0[0], a5[0]) and np.array_equal(a0[1], a5[1]) and np.array_equal(a0[2], a5[2])
    a7 = launch(emu, tmp_path, 4, 7, MODE_MID, st, U, S, g, h, eps, a=0.00625)
    assert np.array_equal(a0[0], a6[0]) and np.array_equal(a0[1], a6[1]) and a5[3] == a6[3]
    assert np.array_equal(a0[0], a7[0]) and np.array_equal(a0[1], a7[1]) and a5[3] == a7[3]
    assert a0[3]["bytes"] == a5[3]["bytes"]
    ntiles = 2 * 3 * 2
    assert a0[3]["loads"] == ntiles * (25 + 50 + 3) and a5[3]["loads"] == ntiles * (25 + 2 * 13 + 2 * 2 + 4 + 3)


@pytest.mark.parametrize("col_rows", [2, 4, 8, 64])
def test_tile_traversal_order_does_not_change_the_result(oracle, emu, tmp_path, col_rows, monkeypatch):
    """the tuning parameter col_rows (y-extent of the columns in which the persistent CTAs visit the tiles; the runtime
    sweep tries half and twice its value) only permutes the tiles: same bits, every tile visited once"""
    nx, ny, nz, g, h, eps = 20, 13, 6, 3, 0.05, 0.1
    st = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz), g), g)
    z = np.zeros_like(st)
    ref = launch(emu, tmp_path, 4, 0, MODE_RHS, st, z, z, g, h, eps, grid=3)
    monkeypatch.setenv("CHM_COL_ROWS", str(col_rows))
    got = launch(emu, tmp_path, 4, 5, MODE_RHS, st, z, z, g, h, eps, grid=3)
    assert np.array_equal(ref[0], got[0]) and ref[3]["loads"] == got[3]["loads"]


@pytest.mark.parametrize("tile", [0, 1, 3, 5, 7])
def test_fill_only_mode_moves_what_the_full_kernel_moves(oracle, emu, tmp_path, tile):
    """the benchmark mode behind chemora_measure_box_fill: the same TMA requests and bytes as a middle RK4 stage of
    the full kernel (it runs the same issue / wait / release / refill code), no wait gives up, nothing is written"""
    nx, ny, nz, g, h, eps = 20, 9, 6, 3, 0.05, 0.1
    st = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz), g), g)
    U = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz, seed=7), g), g)
    S = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz, seed=8), g), g)
    full = launch(emu, tmp_path, 4, tile, MODE_MID, st, U, S, g, h, eps, a=0.00625)
    fill = launch(emu, tmp_path, 4, tile, 10 + MODE_MID, st, U, S, g, h, eps, a=0.00625)
    assert fill[3] == full[3]                                        # TMA requests and bytes
    assert not fill[0].any() and np.array_equal(fill[1], S) and np.array_equal(fill[2], U)


def test_flat_space_gives_exactly_zero(oracle, emu, tmp_path):
    st = oracle.fill_ghosts(oracle.with_ghosts(inputs.bssn_minkowski(16, 8, 8), 3), 3)
    z = np.zeros_like(st)
    out, _, _, _ = launch(emu, tmp_path, 4, 0, MODE_RHS, st, z, z, 3, 0.05, 0.1)
    assert not out.any()


@pytest.mark.parametrize("tile", [0, 3, 5, 6, 7])
def test_one_rk4_step_through_the_four_epilogues(oracle, emu, tmp_path, tile):
    """FIRST, MID, MID, LAST chained as chemora_rk4_step chains them (the periodic fill between the stages done by the
    oracle's fill): equals the oracle's RK4 step in both norms of DESIGN.md S11 / S11b"""
    nx, ny, nz, g, h, eps = 20, 6, 9, 3, 0.05, 0.1
    dt = 0.25 * h
    u0 = inputs.bssn_gaussians(nx, ny, nz, width_cells=3.0)
    fill = lambda s: oracle.fill_ghosts(s.copy(), g)
    U = fill(oracle.with_ghosts(u0, g))
    S = np.zeros_like(U)
    Yb, S, _, _ = launch(emu, tmp_path, 4, tile, MODE_FIRST, U, U, S, g, h, eps, a=dt / 2)
    Ya, S, _, _ = launch(emu, tmp_path, 4, tile, MODE_MID, fill(Yb), U, S, g, h, eps, a=dt / 2)
    Yb, S, _, _ = launch(emu, tmp_path, 4, tile, MODE_MID, fill(Ya), U, S, g, h, eps, a=dt)
    _, _, U1, _ = launch(emu, tmp_path, 4, tile, MODE_LAST, fill(Yb), U, S, g, h, eps, a=dt / 6)
    want = oracle.rk4(oracle.SYS_BSSN, oracle.with_ghosts(u0, g), g, 4, h, dt, oracle.params(eps_diss=eps), 1)
    got, want = oracle.interior(U1, g), oracle.interior(want, g)
    assert relerr(got, want) < 1e-13
    for v in (0, 1, 4, 6, 17):                                  # background-subtracted norm on the O(1) slots
        amp = np.max(np.abs(want[v] - 1.0))
        assert np.max(np.abs((got[v] - 1.0) - (want[v] - 1.0))) < max(1e-11, 8 * 2.3e-16 / amp) * amp


@pytest.mark.parametrize("tile", [0, 5, 7])
def test_ssp_epilogue(oracle, emu, tmp_path, tile):
    """MODE_SSP: out = ca U + cb (in + dt k), the Shu-Osher stage"""
    nx, ny, nz, g, h, eps = 16, 8, 4, 3, 0.05, 0.1
    st = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz, seed=5, amp=0.02), g), g)
    U = oracle.fill_ghosts(oracle.with_ghosts(strong(nx, ny, nz, seed=6, amp=0.02), g), g)
    out, _, _, _ = launch(emu, tmp_path, 4, tile, MODE_SSP, st, U, np.zeros_like(U), g, h, eps, a=0.01, ca=0.75, cb=0.25)
    k = oracle.rhs(oracle.SYS_BSSN, st, g, 4, h, oracle.params(eps_diss=eps))
    want = 0.75 * U + 0.25 * (st + 0.01 * k)
    assert relerr(oracle.interior(out, g), oracle.interior(want, g)) < 1e-13
