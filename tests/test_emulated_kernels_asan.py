"""The emulated kernels once more under AddressSanitizer: the CTA's shared memory is one heap block and every state
buffer an exactly sized heap array, so a shared-memory or global access outside its allocation -- which on the device
is a fault (Xid 13/43) or silent corruption -- aborts the emulator here.  Covers the fused kernel in every section
layout (ids 0, 1, 3, 5, 7; a middle RK4 stage, ragged tiles, several tiles per CTA), the 8th-order instance, the
plane-ring kernel and the radiative face kernel.  Part of VERDICT r1 task 1 (no launch may fault)."""
import os
import subprocess

import numpy as np
import pytest

from paper_1307_6488_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def build(tmp, name):
    from tests.conftest import build_emulator
    return build_emulator(name, flags=("-O0", "-fsanitize=address"))


def run(cmd):
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0")
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=900)
    assert r.returncode == 0 and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
    return r.stdout


def test_fused_kernel_under_asan(oracle, tmp_path):
    exe = build(tmp_path, "fused_emu")
    g, h, eps = 3, 0.05, 0.1
    for order, tile, dims, gg in [(4, 0, (20, 9, 6), 3), (4, 1, (17, 9, 3), 3), (4, 3, (17, 3, 9), 3), (4, 5, (20, 5, 6), 3),
                                  (4, 7, (18, 5, 6), 4), (8, 0, (17, 5, 5), 5)]:
        nx, ny, nz = dims
        st = oracle.fill_ghosts(oracle.with_ghosts(inputs.bssn_noise(nx, ny, nz), gg), gg)
        paths = [str(tmp_path / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
        for p in paths[:3]:
            st.tofile(p)
        out = run([exe, str(order), str(tile), "2", str(nx), str(ny), str(nz), str(gg), repr(h), repr(eps), "1.0", "0.75", "5",
                   "0.00625", "0.0", "0.0", "2"] + paths)
        assert out.split()[1] == "0", out


def test_wave_and_boundary_kernels_under_asan(oracle, tmp_path):
    wave, bnd = build(tmp_path, "wave_emu"), build(tmp_path, "boundary_emu")
    rng = np.random.default_rng(3)
    paths = [str(tmp_path / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
    for V, order, g, which, dims in [(2, 8, 4, 0, (33, 18, 35)), (5, 4, 3, 0, (19, 11, 66))]:
        nx, ny, nz = dims
        st = oracle.fill_ghosts(oracle.with_ghosts(rng.standard_normal((V, nz, ny, nx)), g), g)
        for p in paths[:3]:
            st.tofile(p)
        run([wave, str(V), str(order), "1", str(which), "2", str(nx), str(ny), str(nz), str(g), "0.03125", "0.1", "0.01", "0.0",
             "0.0", "2"] + paths)
    for system, g, dims in [(1, 3, (9, 6, 5)), (0, 2, (10, 8, 6))]:
        nx, ny, nz = dims
        V = 25 if system == 1 else 2
        st = rng.standard_normal((V, nz + 2 * g, ny + 2 * g, nx + 2 * g))
        for p in paths[:3]:
            st.tofile(p)
        run([bnd, "rad", str(system), str(nx), str(ny), str(nz), str(g), "0.07", "2", "0.01", "0.0", "0.0"] + paths)


def build_tsan(tmp, name, *defines):
    from tests.conftest import build_emulator
    return build_emulator(name, flags=("-O0", "-fsanitize=thread") + tuple(defines))


def test_fused_kernel_under_thread_sanitizer(oracle, tmp_path):
    """Race detection at the granularity of the emulator's barriers: the emulated CUDA threads are OS threads whose only
    ordering comes from the kernel's own __syncthreads / __syncwarp / bar.sync / mbarrier calls, so a shared-memory
    access pair the kernel's protocol leaves unordered (a slot refilled while a warp still reads it, a first-derivative
    buffer rewritten before the plane's readers are through, the At_ij table laid over those buffers) is a
    ThreadSanitizer report.  Every section layout of the fused kernel runs a middle RK4 stage clean; and, as a
    self-test of the detector, the same kernel with its plane barriers compiled out (CHM_EMU_DROP_NAMED_BARRIERS) IS
    reported."""
    exe = build_tsan(tmp_path, "fused_emu")
    h, eps = 0.05, 0.1
    paths = [str(tmp_path / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
    env = dict(os.environ, TSAN_OPTIONS="halt_on_error=0 report_signal_unsafe=0")

    def go(binary, order, tile, dims, g):
        nx, ny, nz = dims
        st = oracle.fill_ghosts(oracle.with_ghosts(inputs.bssn_noise(nx, ny, nz), g), g)
        for p in paths[:3]:
            st.tofile(p)
        return subprocess.run([binary, str(order), str(tile), "2", str(nx), str(ny), str(nz), str(g), repr(h), repr(eps), "1.0",
                               "0.75", "5", "0.00625", "0.0", "0.0", "2"] + paths, capture_output=True, text=True, env=env,
                              timeout=900)

    for order, tile, dims, g in [(4, 0, (20, 9, 6), 3), (4, 1, (17, 9, 3), 3), (4, 3, (17, 3, 9), 3), (4, 5, (20, 5, 6), 3),
                                 (4, 6, (20, 5, 6), 3), (4, 7, (18, 5, 6), 4), (8, 0, (17, 5, 5), 5)]:
        r = go(exe, order, tile, dims, g)
        assert "ThreadSanitizer" not in r.stderr and r.stdout.split()[1] == "0", (tile, r.stderr[-3000:])
    broken = build_tsan(tmp_path, "fused_emu", "-DCHM_EMU_DROP_NAMED_BARRIERS")
    r = go(broken, 4, 0, (20, 9, 6), 3)
    assert "ThreadSanitizer: data race" in r.stderr


def test_plane_ring_kernel_under_thread_sanitizer(oracle, tmp_path):
    """the plane-ring kernel's slot protocol (release of the oldest plane, refill by the last warp, item boundary).
    Grids are multiples of the (x, y) tile here: on ragged tiles the threads outside the grid prefetch the Runge-Kutta
    operands of a clamped, valid point (which another thread may be updating) and discard them -- harmless, but a
    report; the ragged cases are covered by the parity and AddressSanitizer tests."""
    exe = build_tsan(tmp_path, "wave_emu")
    rng = np.random.default_rng(4)
    paths = [str(tmp_path / n) for n in ("in.bin", "U.bin", "S.bin", "out.bin")]
    env = dict(os.environ, TSAN_OPTIONS="halt_on_error=0 report_signal_unsafe=0")
    for V, order, g, which, dims in [(2, 8, 4, 0, (64, 16, 35)), (2, 4, 3, 2, (64, 16, 13)), (5, 4, 3, 0, (32, 8, 66))]:
        nx, ny, nz = dims
        st = oracle.fill_ghosts(oracle.with_ghosts(rng.standard_normal((V, nz, ny, nx)), g), g)
        for p in paths[:3]:
            st.tofile(p)
        r = subprocess.run([exe, str(V), str(order), "1", str(which), "2", str(nx), str(ny), str(nz), str(g), "0.03125", "0.1",
                            "0.01", "0.0", "0.0", "2"] + paths, capture_output=True, text=True, env=env, timeout=900)
        assert r.returncode == 0 and "ThreadSanitizer" not in r.stderr and r.stdout.split()[1] == "0", r.stderr[-3000:]
