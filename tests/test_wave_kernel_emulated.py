"""The plane-ring kernel's SOURCE (csrc/kernels_wave_tma.cu; the (phi, pi) system and the paper's Sample-1 system),
executed on the host on top of tests/native/cta_emu.hpp (see tests/test_fused_kernel_emulated.py for what the
emulation covers): z-marching work items, the ring of plane boxes with its load sequence numbers and parities, the
release of the oldest plane and the refill by the last warp, the item boundary, the prefetched Runge-Kutta operands."""
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MODE_RHS, MODE_FIRST, MODE_MID, MODE_LAST, MODE_SSP = range(5)


@pytest.fixture(scope="module")
def emu():
    from tests.conftest import build_emulator
    return build_emulator("wave_emu")


def launch(exe, tmp, V, order, ko, which, mode, st_in, U, S, g, h, eps, a=0.0, ca=0.0, cb=0.0, grid=2):
    _, tz, ty, tx = st_in.shape
    paths = [str(tmp / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
    for arr, p in zip((st_in, U, S), paths):
        np.ascontiguousarray(arr).tofile(p)
    r = subprocess.run([exe, str(V), str(order), str(int(ko)), str(which), str(mode), str(tx - 2 * g), str(ty - 2 * g),
                        str(tz - 2 * g), str(g), repr(h), repr(eps), repr(a), repr(ca), repr(cb), str(grid)] + paths,
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    words = r.stdout.split()
    assert words[0] == "err" and int(words[1]) == 0, r.stdout
    out = np.fromfile(paths[3]).reshape(3, V, tz, ty, tx)
    return out[0], out[1], out[2]


def relerr(a, b):
    return max(np.max(np.abs(a[v] - b[v])) / max(np.max(np.abs(b[v])), 1e-300) for v in range(a.shape[0]))


@pytest.mark.parametrize("V,order,g,eps,which,dims", [
    (2, 4, 2, 0.0, 0, (37, 21, 40)),      # two z chunks (nz > 32), ragged x and y
    (2, 4, 3, 0.1, 2, (70, 9, 13)),
    (2, 8, 4, 0.1, 0, (33, 18, 35)),
    (5, 4, 3, 0.1, 0, (19, 11, 70)),      # Sample-1 system, two 64-plane chunks
    (5, 8, 4, 0.0, 0, (17, 9, 12)),
    (5, 4, 3, 0.1, 1, (18, 17, 9)),
])
def test_rhs_against_the_oracle(oracle, emu, tmp_path, V, order, g, eps, which, dims):
    nx, ny, nz = dims
    system = 0 if V == 2 else 2
    u = np.random.default_rng(11).standard_normal((V, nz, ny, nx))
    h = 1.0 / 32
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    z = np.zeros_like(st)
    out, _, _ = launch(emu, tmp_path, V, order, eps != 0.0, which, MODE_RHS, st, z, z, g, h, eps)
    want = oracle.rhs(system, st, g, order, h, oracle.params(eps_diss=eps))
    assert relerr(oracle.interior(out, g), oracle.interior(want, g)) < 1e-12
    m = np.ones(out.shape[1:], dtype=bool)
    m[g:-g, g:-g, g:-g] = False
    assert not out[:, m].any()


def test_one_rk4_step_of_the_wave_system(oracle, emu, tmp_path):
    nx, ny, nz, g, order, eps = 33, 17, 36, 4, 8, 0.1
    h = 1.0 / 32
    dt = 0.25 * h
    u0 = np.random.default_rng(12).standard_normal((2, nz, ny, nx))
    fill = lambda s: oracle.fill_ghosts(s.copy(), g)
    U = fill(oracle.with_ghosts(u0, g))
    S = np.zeros_like(U)
    args = (emu, tmp_path, 2, order, True, 0)
    Yb, S, _ = launch(*args, MODE_FIRST, U, U, S, g, h, eps, a=dt / 2)
    Ya, S, _ = launch(*args, MODE_MID, fill(Yb), U, S, g, h, eps, a=dt / 2)
    Yb, S, _ = launch(*args, MODE_MID, fill(Ya), U, S, g, h, eps, a=dt)
    _, _, U1 = launch(*args, MODE_LAST, fill(Yb), U, S, g, h, eps, a=dt / 6)
    want = oracle.rk4(oracle.SYS_WAVE, oracle.with_ghosts(u0, g), g, order, h, dt, oracle.params(eps_diss=eps), 1)
    assert relerr(oracle.interior(U1, g), oracle.interior(want, g)) < 1e-13
