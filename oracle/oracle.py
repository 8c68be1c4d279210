"""ctypes harness around oracle/oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It never imports paper_1307_6488_b200 (the CUDA path) and the CUDA path never
imports it.  Arrays are numpy float64 in the oracle layout: [V, nz+2g, ny+2g, nx+2g].
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

SYS_WAVE, SYS_BSSN, SYS_WAVE1 = 0, 1, 2
NVARS = {SYS_WAVE: 2, SYS_BSSN: 25, SYS_WAVE1: 5}
OP_D1, OP_DD, OP_UPW, OP_KO, OP_KO9 = 0, 1, 2, 3, 4

_lib = None


def build(force=False):
    """g++ -O2 -ffp-contract=off (no FMA contraction: reproducible reference arithmetic)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-std=c++17", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        i, d = ctypes.c_int, ctypes.c_double
        _lib.oracle_apply_op.argtypes = [i, dp, dp, i, i, i, i, i, d, i, i, d]
        _lib.oracle_fill_ghosts.argtypes = [dp, i, i, i, i, i]
        _lib.oracle_rhs.argtypes = [i, dp, dp, i, i, i, i, i, d, dp]
        _lib.oracle_rk4.argtypes = [i, dp, i, i, i, i, i, d, d, dp, i]
        _lib.oracle_rk3.argtypes = [i, dp, i, i, i, i, i, d, d, dp, i, i]
        _lib.oracle_radiative_rhs.argtypes = [i, dp, dp, i, i, i, i, d]
        _lib.oracle_radiative_rhs.restype = None
        _lib.oracle_rk4_radiative.argtypes = [i, dp, i, i, i, i, i, d, d, dp, i]
        _lib.oracle_rk4_radiative.restype = None
        _lib.oracle_enforce.argtypes = [dp, i, i, i, i]
        _lib.oracle_energy.argtypes = [dp, i, i, i, i, dp]
        _lib.oracle_energy.restype = None
        _lib.oracle_rk3.restype = None
        _lib.oracle_enforce.restype = None
        _lib.oracle_set_threads.argtypes = [i]
        _lib.oracle_max_threads.restype = i
        for f in (_lib.oracle_apply_op, _lib.oracle_fill_ghosts, _lib.oracle_rhs, _lib.oracle_rk4,
                  _lib.oracle_set_threads):
            f.restype = None
    return _lib


def _p(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def params(eps_diss=0.0, eta=1.0, shift_gamma_coeff=0.75, ko_order=5):
    assert ko_order in (5, 9)
    return np.array([eps_diss, eta, shift_gamma_coeff, ko_order], dtype=np.float64)


def set_threads(n):
    lib().oracle_set_threads(int(n))


def max_threads():
    return lib().oracle_max_threads()


def with_ghosts(packed, g):
    """[V,nz,ny,nx] interior-packed -> [V,nz+2g,ny+2g,nx+2g] with zero (unfilled) ghosts."""
    V, nz, ny, nx = packed.shape
    out = np.zeros((V, nz + 2 * g, ny + 2 * g, nx + 2 * g), dtype=np.float64)
    out[:, g:g + nz, g:g + ny, g:g + nx] = packed
    return out


def interior(ghosted, g):
    if g == 0:
        return np.ascontiguousarray(ghosted)
    return np.ascontiguousarray(ghosted[..., g:-g, g:-g, g:-g])


def apply_op(op, f_ghosted, g, order, h, a=0, b=0, eps=0.0):
    tz, ty, tx = f_ghosted.shape
    nx, ny, nz = tx - 2 * g, ty - 2 * g, tz - 2 * g
    out = np.empty((nz, ny, nx), dtype=np.float64)
    lib().oracle_apply_op(op, _p(f_ghosted), _p(out), nx, ny, nz, g, order, float(h), a, b, float(eps))
    return out


def fill_ghosts(state, g):
    V, tz, ty, tx = state.shape
    lib().oracle_fill_ghosts(_p(state), V, tx - 2 * g, ty - 2 * g, tz - 2 * g, g)
    return state


def rhs(system, state, g, order, h, prm):
    """state [V,tz,ty,tx] with ghosts already filled -> rhs, same shape (ghost entries zero)."""
    V, tz, ty, tx = state.shape
    assert V == NVARS[system]
    out = np.zeros_like(state)
    lib().oracle_rhs(system, _p(state), _p(out), tx - 2 * g, ty - 2 * g, tz - 2 * g, g, order, float(h), _p(prm))
    return out


def rk4(system, state, g, order, h, dt, prm, nsteps=1):
    """Advance `state` (ghosted; ghosts are filled periodically inside) in place; returns it."""
    V, tz, ty, tx = state.shape
    assert V == NVARS[system]
    lib().oracle_rk4(system, _p(state), tx - 2 * g, ty - 2 * g, tz - 2 * g, g, order, float(h), float(dt), _p(prm),
                     int(nsteps))
    return state


def rk3(system, state, g, order, h, dt, prm, nsteps=1, enforce=False):
    """Shu-Osher RK3 (reading S9b), in place; enforce=True applies the BSSN algebraic constraints after each step."""
    V, tz, ty, tx = state.shape
    assert V == NVARS[system]
    lib().oracle_rk3(system, _p(state), tx - 2 * g, ty - 2 * g, tz - 2 * g, g, order, float(h), float(dt), _p(prm),
                     int(nsteps), int(bool(enforce)))
    return state


def radiative_rhs(system, state, g, h, out=None):
    """Reading S16: the radiative (Sommerfeld) right-hand side at every boundary point (the g ghost layers) of a
    ghosted state; interior entries of the result are those of `out` (zeros when not given)."""
    V, tz, ty, tx = state.shape
    assert V == NVARS[system]
    if out is None:
        out = np.zeros_like(state)
    lib().oracle_radiative_rhs(system, _p(state), _p(out), tx - 2 * g, ty - 2 * g, tz - 2 * g, g, float(h))
    return out


def rk4_radiative(system, state, g, order, h, dt, prm, nsteps=1):
    """RK4 (S9) of a block with radiative outer boundaries: `state` is the whole padded block (its ghost layers are
    evolved boundary points, nothing is filled); advanced in place."""
    V, tz, ty, tx = state.shape
    assert V == NVARS[system]
    lib().oracle_rk4_radiative(system, _p(state), tx - 2 * g, ty - 2 * g, tz - 2 * g, g, order, float(h), float(dt),
                               _p(prm), int(nsteps))
    return state


def enforce(state, g):
    """det gt -> 1, tr At -> 0 on the interior of a ghosted BSSN state (reading S10b), in place."""
    V, tz, ty, tx = state.shape
    assert V == 25
    lib().oracle_enforce(_p(state), tx - 2 * g, ty - 2 * g, tz - 2 * g, g)
    return state


def energy(state, g):
    """eps = 1/2 (rho^2 + v_i v_i) of a ghosted system-2 state on its interior: array [nz, ny, nx]."""
    V, tz, ty, tx = state.shape
    assert V == 5
    out = np.empty((tz - 2 * g, ty - 2 * g, tx - 2 * g), dtype=np.float64)
    lib().oracle_energy(_p(state), tx - 2 * g, ty - 2 * g, tz - 2 * g, g, _p(out))
    return out
