"""Two whole RK4 steps with nothing but emulated kernels: the stage table of chemora_rk4_step (csrc/chemora.cu,
rk4_plan: fill(U) FIRST -> fill(Yb) MID -> fill(Ya) MID -> fill(Yb) LAST on the buffers U, Ya, Yb, S) driven from
Python, every launch the library's own kernel source under the CTA emulator -- fill_ghosts_kernel, then the fused
kernel (plain layout id 0 and interleaved layout with the six-slot ring, id 7).  Against the oracle's RK4, both norms of DESIGN.md S11/S11b."""
import os
import subprocess

import numpy as np
import pytest

from paper_1307_6488_b200 import inputs
from tests.test_basic_kernels_emulated import run as basic_run
from tests.test_fused_kernel_emulated import MODE_FIRST, MODE_LAST, MODE_MID, launch, relerr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def emus():
    from tests.conftest import build_emulator
    return build_emulator("basic_emu"), build_emulator("fused_emu")


@pytest.mark.parametrize("tile", [0, 7])
def test_two_rk4_steps_all_kernels_emulated(oracle, emus, tmp_path, tile):
    basic, fused = emus
    nx, ny, nz, g, h, eps = 18, 7, 6, 3, 0.05, 0.1
    dt = 0.25 * h
    u0 = inputs.bssn_gaussians(nx, ny, nz, width_cells=3.0) + 1e-10 * np.random.default_rng(2).uniform(-1, 1, size=(25, nz, ny, nx))
    fill = lambda s: basic_run(basic, tmp_path, "fill", 1, 4, s, g)[0]
    U = oracle.with_ghosts(u0, g)                       # ghosts zero: the first fill must produce them
    S = np.zeros_like(U)
    for _ in range(2):
        U = fill(U)
        Yb, S, _, _ = launch(fused, tmp_path, 4, tile, MODE_FIRST, U, U, S, g, h, eps, a=dt / 2)
        Ya, S, _, _ = launch(fused, tmp_path, 4, tile, MODE_MID, fill(Yb), U, S, g, h, eps, a=dt / 2)
        Yb, S, _, _ = launch(fused, tmp_path, 4, tile, MODE_MID, fill(Ya), U, S, g, h, eps, a=dt)
        _, _, U, _ = launch(fused, tmp_path, 4, tile, MODE_LAST, fill(Yb), U, S, g, h, eps, a=dt / 6)
    want = oracle.interior(oracle.rk4(oracle.SYS_BSSN, oracle.with_ghosts(u0, g), g, 4, h, dt,
                                      oracle.params(eps_diss=eps), 2), g)
    got = oracle.interior(U, g)
    assert relerr(got, want) < 1e-12
    for v in (0, 1, 4, 6, 17):
        amp = np.max(np.abs(want[v] - 1.0))
        assert np.max(np.abs((got[v] - 1.0) - (want[v] - 1.0))) < max(1e-10, 8 * 2.3e-16 / amp) * amp, v
