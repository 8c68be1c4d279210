"""The CUDA path's own right-hand-side arithmetic, run on the HOST against the oracle (no GPU needed).

csrc/stencils.cuh (finite-difference templates, dissipation, upwinded advection, 4th and 8th order), its derivative
provider OnTheFly and csrc/bssn_point.cuh (the pointwise BSSN expression: the kernels' second transcription of reading
S4) are __host__ __device__ code; tests/native/rhs_host_probe.cu instantiates them exactly as the derivative-split BSSN
kernels and the L1-path wave kernels do on the device, over a periodic block.  This does not replace the -m gpu parity
tests (launch geometry, staging, the fused kernel's own section order are not covered) but it shows, on any box, that
the product's arithmetic agrees with the oracle's to rounding: tolerance 1e-12 in the norm of reading S11."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from paper_1307_6488_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def probe(tmp_path_factory):
    nvcc = os.environ.get("NVCC") or shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path_factory.mktemp("probe") / "rhs_host_probe")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-o", exe, os.path.join(ROOT, "tests", "native", "rhs_host_probe.cu")],
                   check=True, capture_output=True)
    return exe


def run_probe(exe, tmp, system, order, u, g, h, eps=0.1, eta=1.0, sgc=0.75, ko_order=5):
    V, nz, ny, nx = u.shape
    from oracle import oracle
    st = oracle.fill_ghosts(oracle.with_ghosts(u, g), g)
    fin, fout = str(tmp / "in.bin"), str(tmp / "out.bin")
    st.tofile(fin)
    subprocess.run([exe, str(system), str(order), str(nx), str(ny), str(nz), str(g), repr(h), repr(eps), repr(eta),
                    repr(sgc), str(ko_order), fin, fout], check=True)
    got = np.fromfile(fout).reshape(V, nz, ny, nx)
    want = oracle.interior(oracle.rhs(system, st, g, order, h,
                                      oracle.params(eps_diss=eps, eta=eta, shift_gamma_coeff=sgc, ko_order=ko_order)), g)
    return got, want


def relerr(a, b):
    return max(np.max(np.abs(a[v] - b[v])) / max(np.max(np.abs(b[v])), 1e-300) for v in range(a.shape[0]))


@pytest.mark.parametrize("order,g,ko_order", [(4, 3, 5), (8, 5, 5), (8, 5, 9)])
@pytest.mark.parametrize("data", ["noise1e-10", "gaussians", "strong"])
def test_bssn_pointwise_and_stencils(probe, tmp_path, order, g, ko_order, data):
    nx, ny, nz = 13, 11, 12
    if data == "noise1e-10":
        u = inputs.bssn_noise(nx, ny, nz)
    elif data == "gaussians":
        u = inputs.bssn_gaussians(nx, ny, nz, width_cells=3.0)
    else:
        u = inputs.bssn_minkowski(nx, ny, nz) + 0.1 * np.random.default_rng(21).uniform(-1, 1, size=(25, nz, ny, nx))
    got, want = run_probe(probe, tmp_path, 1, order, u, g, 0.05, eta=1.3, sgc=0.6, ko_order=ko_order)
    assert relerr(got, want) < 1e-12
    if data == "strong":
        assert all(np.max(np.abs(want[v])) > 0 for v in range(25))       # every right-hand side is exercised


def test_bssn_flat_is_exactly_zero(probe, tmp_path):
    got, want = run_probe(probe, tmp_path, 1, 4, inputs.bssn_minkowski(8, 8, 8), 3, 0.05)
    assert not got.any() and not want.any()


@pytest.mark.parametrize("system,order,g,eps", [(0, 4, 2, 0.0), (0, 4, 3, 0.1), (0, 8, 4, 0.1), (2, 4, 3, 0.1), (2, 8, 4, 0.0)])
def test_wave_systems(probe, tmp_path, system, order, g, eps):
    V = 2 if system == 0 else 5
    u = np.random.default_rng(11).standard_normal((V, 9, 10, 11))
    got, want = run_probe(probe, tmp_path, system, order, u, g, 1.0 / 32, eps=eps)
    assert relerr(got, want) < 1e-12
