"""csrc/kernels_boundary.cu executed on the host (tests/native/cta_emu.hpp, launch geometry of the real launchers): the
radiative face kernel (reading S16) against the oracle at every boundary point and through a whole RK4 step, and the
runtime sweep's agreement norm against numpy.  No GPU needed; the -m gpu tests repeat the comparison on the device."""
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
    return build_emulator("boundary_emu")


def rad(exe, tmp, system, st_in, U, S, g, h, mode, a=0.0, ca=0.0, cb=0.0):
    V, tz, ty, tx = st_in.shape
    paths = [str(tmp / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
    for arr, p in zip((st_in, U, S), paths):
        np.ascontiguousarray(arr).tofile(p)
    subprocess.run([exe, "rad", str(system), str(tx - 2 * g), str(ty - 2 * g), str(tz - 2 * g), str(g), repr(h), str(mode),
                    repr(a), repr(ca), repr(cb)] + paths, check=True, timeout=600)
    out = np.fromfile(paths[3]).reshape(3, V, tz, ty, tx)
    return out[0], out[1], out[2]


def boundary(shape, g):
    m = np.ones(shape, dtype=bool)
    m[g:-g, g:-g, g:-g] = False
    return m


@pytest.mark.parametrize("system,g,dims", [(0, 2, (10, 8, 6)), (0, 4, (13, 5, 9)), (2, 3, (7, 9, 5)), (1, 3, (9, 6, 5)),
                                           (1, 4, (8, 5, 6))])
def test_radiative_rhs(oracle, emu, tmp_path, system, g, dims):
    nx, ny, nz = dims
    V = {0: 2, 1: 25, 2: 5}[system]
    st = np.random.default_rng(51).standard_normal((V, nz + 2 * g, ny + 2 * g, nx + 2 * g))
    want = oracle.radiative_rhs(system, st, g, 0.07)
    z = np.zeros_like(st)
    out, _, _ = rad(emu, tmp_path, system, st, z, z, g, 0.07, MODE_RHS)
    m = boundary(st.shape[1:], g)
    for v in range(V):
        assert np.max(np.abs(out[v][m] - want[v][m])) < 1e-12 * np.max(np.abs(want[v][m])), v
    assert (out[:, ~m] == 7.0).all()                    # the interior is not this kernel's


def test_radiative_rk4_boundary_points_near_flat(oracle, emu, tmp_path):
    """the four epilogues at the boundary points on configs[2]-like data (1 + 1e-10 noise): what the oracle's
    radiative RK4 step leaves there, in the background-subtracted norm too (difference-form one-sided stencils)"""
    nx, ny, nz, g, h = 8, 6, 5, 3, 0.05
    dt = 0.25 * h
    rng = np.random.default_rng(52)
    U0 = oracle.fill_ghosts(oracle.with_ghosts(inputs.bssn_noise(nx, ny, nz), g), g) + 1e-10 * rng.uniform(-1, 1, size=(25, nz + 2 * g, ny + 2 * g, nx + 2 * g))
    prm = oracle.params(eps_diss=0.1)
    m = boundary(U0.shape[1:], g)
    # reference: the oracle's radiative step; the interior right-hand sides of its stages are the oracle's too, so
    # drive the emulated face kernel stage by stage with the oracle's stage states
    def stage_states():
        U = U0.copy()
        k = lambda s: oracle.radiative_rhs(1, s, g, h, out=oracle.rhs(1, s, g, 4, h, prm))
        k1 = k(U); Y2 = U + (dt / 2) * k1
        k2 = k(Y2); Y3 = U + (dt / 2) * k2
        k3 = k(Y3); Y4 = U + dt * k3
        return U, Y2, Y3, Y4
    U, Y2, Y3, Y4 = stage_states()
    S = np.zeros_like(U)
    Yb, S, _ = rad(emu, tmp_path, 1, U, U, S, g, h, MODE_FIRST, a=dt / 2)
    assert np.max(np.abs(Yb[:, m] - Y2[:, m])) < 1e-15
    Ya, S, _ = rad(emu, tmp_path, 1, Y2, U, S, g, h, MODE_MID, a=dt / 2)
    Yb, S, _ = rad(emu, tmp_path, 1, Y3, U, S, g, h, MODE_MID, a=dt)
    _, _, U1 = rad(emu, tmp_path, 1, Y4, U, S, g, h, MODE_LAST, a=dt / 6)
    want = oracle.rk4_radiative(1, U0.copy(), g, 4, h, dt, prm, 1)
    for v in range(25):
        bg = 1.0 if v in (0, 1, 4, 6, 17) else 0.0
        amp = np.max(np.abs(want[v][m] - bg))
        assert np.max(np.abs((U1[v][m] - bg) - (want[v][m] - bg))) < max(1e-10, 8 * 2.3e-16 / amp) * amp, v


def test_agreement_norm(emu, tmp_path):
    V, n = 3, 5000
    rng = np.random.default_rng(3)
    a = rng.standard_normal((V, n))
    b = a + 1e-9 * rng.standard_normal((V, n))
    b[2] = a[2]
    a[1, 77] = np.nan
    a.tofile(str(tmp_path / "a.bin")); b.tofile(str(tmp_path / "b.bin"))
    r = subprocess.run([emu, "maxdiff", str(V), str(n), str(tmp_path / "a.bin"), str(tmp_path / "b.bin")], check=True,
                       capture_output=True, text=True)
    got = np.array([float(x) for x in r.stdout.split()]).reshape(V, 2)
    assert got[0, 0] == np.max(np.abs(a[0] - b[0])) and got[0, 1] == np.max(np.abs(b[0]))
    assert np.isinf(got[1, 0])                          # a NaN on either side is an infinite difference
    assert got[2, 0] == 0.0 and got[2, 1] == np.max(np.abs(b[2]))
