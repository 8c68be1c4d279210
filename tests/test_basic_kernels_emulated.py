"""The remaining kernels' SOURCE executed on the host (tests/native/cta_emu.hpp): csrc/kernels_basic.cu and
csrc/kernels_bssn.cu on the grids their launchers give them -- periodic ghost fill (bit-exact), pack/unpack,
constraint enforcement, the L1-path kernels of both wave systems, the derivative-split BSSN variant (136 derivative
arrays, then the right-hand side from them), the Energy calculation of the paper's Sample 1.
Together with the fused-kernel, plane-ring and boundary-kernel tests every __global__ function of the library but
the FP64 peak probe runs against the oracle on a box without a GPU; the -m gpu tests repeat it on the device."""
import os
import subprocess

import numpy as np
import pytest

from paper_1307_6488_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def emu():
    from tests.conftest import build_emulator
    return build_emulator("basic_emu")


def run(exe, tmp, op, system, order, st, g, h=0.05, eps=0.0, tile=0, mode=0, a=0.0, ko_order=5, raw=False):
    V, tz, ty, tx = st.shape
    fin, fout = str(tmp / "in.bin"), str(tmp / "out.bin")
    np.ascontiguousarray(st).tofile(fin)
    subprocess.run([exe, op, str(system), str(order), str(tx - 2 * g), str(ty - 2 * g), str(tz - 2 * g), str(g), repr(h),
                    repr(eps), str(tile), str(mode), repr(a), str(ko_order), fin, fout], check=True, timeout=900)
    out = np.fromfile(fout)
    return out if raw else out.reshape(-1, V, tz, ty, tx)


def relerr(a, b):
    return max(np.max(np.abs(a[v] - b[v])) / max(np.max(np.abs(b[v])), 1e-300) for v in range(a.shape[0]))


@pytest.mark.parametrize("system,g,dims", [(1, 3, (37, 7, 5)), (0, 2, (16, 16, 16)), (0, 4, (5, 4, 9)), (1, 3, (3, 3, 3)),
                                           (1, 4, (9, 6, 7)), (2, 5, (6, 5, 7))])
def test_ghost_fill_bit_exact(oracle, emu, tmp_path, system, g, dims):
    nx, ny, nz = dims
    V = {0: 2, 1: 25, 2: 5}[system]
    u = np.random.default_rng(5).standard_normal((V, nz, ny, nx))
    st = oracle.with_ghosts(u, g)
    st[st == 0.0] = 99.0                       # stale ghost values must all be overwritten
    st[:, g:-g, g:-g, g:-g] = u
    got = run(emu, tmp_path, "fill", system, 4, st, g)[0]
    assert np.array_equal(got, oracle.fill_ghosts(oracle.with_ghosts(u, g), g))


def test_pack_unpack_roundtrip(oracle, emu, tmp_path):
    u = np.random.default_rng(6).standard_normal((25, 9, 10, 11))
    st = oracle.with_ghosts(u, 3)
    got = run(emu, tmp_path, "roundtrip", 1, 4, st, 3)[0]
    assert np.array_equal(got, st)             # interior copied, nothing else touched (ghosts stay 0)


def test_constraint_enforcement(oracle, emu, tmp_path):
    nx, ny, nz, g = 21, 9, 10, 3
    u = inputs.bssn_minkowski(nx, ny, nz) + 0.1 * np.random.default_rng(33).uniform(-1, 1, size=(25, nz, ny, nx))
    st = oracle.with_ghosts(u, g)
    got = run(emu, tmp_path, "enforce", 1, 4, st, g)[0]
    want = oracle.enforce(st.copy(), g)
    assert relerr(oracle.interior(got, g), oracle.interior(want, g)) < 1e-14
    flat = oracle.with_ghosts(inputs.bssn_minkowski(8, 8, 8), g)
    assert np.array_equal(run(emu, tmp_path, "enforce", 1, 4, flat, g)[0], flat)


@pytest.mark.parametrize("system,order,g,eps,tile,dims", [(0, 4, 2, 0.0, 0, (37, 21, 19)), (0, 8, 4, 0.1, 1, (33, 9, 12)),
                                                          (0, 4, 3, 0.1, 5, (16, 17, 9)), (2, 4, 3, 0.1, 0, (37, 9, 10)),
                                                          (2, 8, 4, 0.0, 5, (18, 17, 9))])
def test_l1_path_wave_kernels(oracle, emu, tmp_path, system, order, g, eps, tile, dims):
    nx, ny, nz = dims
    V = 2 if system == 0 else 5
    u = np.random.default_rng(11).standard_normal((V, nz, ny, nx))
    h = 1.0 / 32
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    got = run(emu, tmp_path, "wave", system, order, st, g, h=h, eps=eps, tile=tile)[0]
    want = oracle.rhs(system, st, g, order, h, oracle.params(eps_diss=eps))
    assert relerr(oracle.interior(got, g), oracle.interior(want, g)) < 1e-12
    # a middle RK4 stage with U = S = the state: Y = U + a k, S' = S + 2 k, each product and sum rounded once
    y, s2 = run(emu, tmp_path, "wave", system, order, st, g, h=h, eps=eps, tile=tile, mode=2, a=0.01)
    k = oracle.interior(want, g)
    u0 = oracle.interior(st, g)
    assert relerr(oracle.interior(y, g), u0 + 0.01 * k) < 1e-14 and relerr(oracle.interior(s2, g), u0 + 2.0 * k) < 1e-13


@pytest.mark.parametrize("order,g,tile,ko_order", [(4, 3, 0, 5), (4, 4, 5, 5), (8, 5, 0, 9)])
@pytest.mark.parametrize("data", ["strong", "noise1e-10"])
def test_split_variant(oracle, emu, tmp_path, order, g, tile, ko_order, data):
    nx, ny, nz = 21, 10, 9
    u = inputs.bssn_noise(nx, ny, nz) if data == "noise1e-10" else \
        inputs.bssn_minkowski(nx, ny, nz) + 0.1 * np.random.default_rng(21).uniform(-1, 1, size=(25, nz, ny, nx))
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    got = run(emu, tmp_path, "split", 1, order, st, g, eps=0.1, tile=tile, ko_order=ko_order)[0]
    want = oracle.rhs(1, st, g, order, 0.05, oracle.params(eps_diss=0.1, ko_order=ko_order))
    assert relerr(oracle.interior(got, g), oracle.interior(want, g)) < 1e-12


def test_energy_field_and_sum(oracle, emu, tmp_path):
    nx, ny, nz, g = 37, 5, 6, 3
    u = np.random.default_rng(13).standard_normal((5, nz, ny, nx))
    st = oracle.with_ghosts(u, g)
    out = run(emu, tmp_path, "energy", 2, 4, st, g, raw=True)
    want = oracle.energy(st, g)
    assert np.array_equal(out[:-1].reshape(nz, ny, nx), want)          # the field bit for bit
    assert out[-1] == pytest.approx(want.sum(), rel=1e-13)
