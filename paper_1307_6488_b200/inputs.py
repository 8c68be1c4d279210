"""Seeded synthetic input generators.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests, and therefore
holds none of the method's arithmetic (no stencils, no right-hand sides, no time stepping) and
imports neither side.  Every array is float64, interior-packed [V, nz, ny, nx] (x fastest),
generated on the host with numpy.random.default_rng(seed) so both sides read identical bits.

The paper's own workloads (McLachlan benchmark, QC-0 binary black hole) need
its initial-data solvers and are not reproduced; these inputs have the same structure: V fp64
grid functions on a uniform periodic block, near-vacuum data.
"""
import numpy as np

SEED_BASE = 13076488

SYS_WAVE, SYS_BSSN, SYS_WAVE1 = 0, 1, 2

# BSSN slot order (reading S3)
BSSN_NAMES = ["chi", "gt11", "gt12", "gt13", "gt22", "gt23", "gt33", "trK",
              "At11", "At12", "At13", "At22", "At23", "At33", "Gt1", "Gt2", "Gt3",
              "alpha", "beta1", "beta2", "beta3", "B1", "B2", "B3", "A"]
WAVE_NAMES = ["phi", "pi"]


def _coords(n):
    """Unit periodic cube: x_i = i / n."""
    return np.arange(n, dtype=np.float64) / n


def wave_standing(nx, ny, nz, noise=1e-6, seed=SEED_BASE + 0):
    """configs[0]: phi = sin(2 pi x) sin(2 pi y) sin(2 pi z) + noise * U(-1,1), pi = 0."""
    x, y, z = _coords(nx), _coords(ny), _coords(nz)
    phi = (np.sin(2 * np.pi * z)[:, None, None] * np.sin(2 * np.pi * y)[None, :, None]
           * np.sin(2 * np.pi * x)[None, None, :])
    if noise:
        rng = np.random.default_rng(seed)
        phi = phi + noise * rng.uniform(-1.0, 1.0, size=phi.shape)
    out = np.zeros((2, nz, ny, nx), dtype=np.float64)
    out[0] = phi
    return out


def wave_plane_sum(nx, ny, nz, nwaves=8, seed=SEED_BASE + 1):
    """configs[1]: seeded random-phase sum of `nwaves` plane waves, wavelength 8-64 cells
    (integer mode vectors m with n/64 <= |m| <= n/8, n = min dimension, periodic-compatible):
    phi = sum sin(2 pi m.x + p), pi = -sum w cos(2 pi m.x + p), w = 2 pi |m| (unit cube)."""
    rng = np.random.default_rng(seed)
    n = min(nx, ny, nz)
    lo, hi = max(n / 64.0, 1.0), max(n / 8.0, 1.0)
    modes = []
    while len(modes) < nwaves:
        m = rng.integers(-int(hi), int(hi) + 1, size=3)
        r = float(np.sqrt((m * m).sum()))
        if lo <= r <= hi:
            modes.append(m)
    phases = rng.uniform(0.0, 2 * np.pi, size=nwaves)
    x, y, z = _coords(nx), _coords(ny), _coords(nz)
    phi = np.zeros((nz, ny, nx), dtype=np.float64)
    pi = np.zeros((nz, ny, nx), dtype=np.float64)
    for m, p in zip(modes, phases):
        arg = 2 * np.pi * (m[2] * z[:, None, None] + m[1] * y[None, :, None] + m[0] * x[None, None, :]) + p
        w = 2 * np.pi * float(np.sqrt((m * m).sum()))
        phi += np.sin(arg)
        pi -= w * np.cos(arg)
    out = np.empty((2, nz, ny, nx), dtype=np.float64)
    out[0], out[1] = phi, pi
    return out


WAVE1_NAMES = ["u", "rho", "v1", "v2", "v3"]


def wave1_gaussian(nx, ny, nz, amp=1.0, width_cells=4.0):
    """The paper's Sample-1 initial data: u = 0, rho = A exp(-1/2 (r/W)^2), v_i = 0, centred in the
    unit periodic cube (minimum-image distance), W = width_cells grid spacings."""
    out = np.zeros((5, nz, ny, nx), dtype=np.float64)
    d = []
    for n in (nz, ny, nx):
        x = np.abs(np.arange(n, dtype=np.float64) - n / 2.0)
        d.append(np.minimum(x, n - x))
    r2 = d[0][:, None, None] ** 2 + d[1][None, :, None] ** 2 + d[2][None, None, :] ** 2
    out[1] = amp * np.exp(-0.5 * r2 / width_cells ** 2)
    return out


def bssn_minkowski(nx, ny, nz):
    """chi = 1, gt = delta, alpha = 1, everything else 0."""
    out = np.zeros((25, nz, ny, nx), dtype=np.float64)
    out[0] = 1.0
    out[1] = 1.0
    out[4] = 1.0
    out[6] = 1.0
    out[17] = 1.0
    return out


def bssn_noise(nx, ny, nz, amp=1e-10, seed=SEED_BASE + 2):
    """configs[2] (and the sweep grids of configs[4]): Minkowski + amp * U(-1,1) on all 25 slots."""
    rng = np.random.default_rng(seed)
    out = bssn_minkowski(nx, ny, nz)
    out += amp * rng.uniform(-1.0, 1.0, size=out.shape)
    return out


def bssn_gaussians(nx, ny, nz, amp=1e-4, width_cells=16.0, seed=SEED_BASE + 3):
    """configs[3]: Minkowski + one Gaussian (+-amp) exp(-r^2 / 2 sigma^2), sigma = width_cells cells,
    on each of gt11..gt33 and alpha; seeded centre and sign; minimum-image (periodic) distance."""
    rng = np.random.default_rng(seed)
    out = bssn_minkowski(nx, ny, nz)
    ii = np.arange(nx, dtype=np.float64)
    jj = np.arange(ny, dtype=np.float64)
    kk = np.arange(nz, dtype=np.float64)
    for v in (1, 2, 3, 4, 5, 6, 17):
        c = rng.uniform(0.0, 1.0, size=3) * np.array([nx, ny, nz])
        sign = 1.0 if rng.uniform() < 0.5 else -1.0
        dx = np.abs(ii - c[0]); dx = np.minimum(dx, nx - dx)
        dy = np.abs(jj - c[1]); dy = np.minimum(dy, ny - dy)
        dz = np.abs(kk - c[2]); dz = np.minimum(dz, nz - dz)
        r2 = dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2
        out[v] += sign * amp * np.exp(-r2 / (2.0 * width_cells ** 2))
    return out


# The five BASELINE.json configs as (system, dims, ghost, fd_order, dx, eps_diss, generator)
def bssn_waves_slab(nx, ny, nz, z0, z1, amp=1e-4, seed=SEED_BASE + 6):
    """Planes z0 <= k < z1 (k taken mod nz) of a periodic near-Minkowski state that can be generated slab by slab:
    every slot = its Minkowski value + amp * sin(2 pi (mx i/nx + my j/ny + mz k/nz) + phase), with seeded integer
    mode numbers per slot (wavelength nx/mx >= 8 cells in x and y, about 16..32 cells in z).  Used for blocks too
    large to build on the host in one piece (more than 2^31 elements per buffer)."""
    rng = np.random.default_rng(seed)
    mx = rng.integers(1, max(nx // 8, 1) + 1, size=25)
    my = rng.integers(1, max(ny // 8, 1) + 1, size=25)
    mz = rng.integers(max(nz // 32, 1), max(nz // 16, 1) + 1, size=25)
    ph = rng.uniform(0.0, 2 * np.pi, size=25)
    k = np.arange(z0, z1, dtype=np.int64) % nz
    j = np.arange(ny, dtype=np.int64)
    i = np.arange(nx, dtype=np.int64)
    out = np.empty((25, z1 - z0, ny, nx), dtype=np.float64)
    base = bssn_minkowski(1, 1, 1)[:, 0, 0, 0]
    for v in range(25):
        # integer products reduced modulo the period first, so the phase keeps full precision at large nz
        arg = (2 * np.pi) * (((mz[v] * k) % nz)[:, None, None] / nz + ((my[v] * j) % ny)[None, :, None] / ny
                             + ((mx[v] * i) % nx)[None, None, :] / nx) + ph[v]
        out[v] = base[v] + amp * np.sin(arg)
    return out


def config(index, scale=None):
    """Returns a dict describing BASELINE.json configs[index]; `scale` overrides the cube size
    (for parity tests at sizes the oracle finishes in seconds)."""
    if index == 0:
        n = scale or 32
        return dict(system=SYS_WAVE, dims=(n, n, n), ghost=2, order=4, dx=1.0 / n, eps_diss=0.0,
                    steps=20, state=lambda: wave_standing(n, n, n))
    if index == 1:
        n = scale or 256
        return dict(system=SYS_WAVE, dims=(n, n, n), ghost=4, order=8, dx=1.0 / n, eps_diss=0.1,
                    steps=1, state=lambda: wave_plane_sum(n, n, n))
    if index == 2:
        n = scale or 64
        return dict(system=SYS_BSSN, dims=(n, n, n), ghost=3, order=4, dx=0.05, eps_diss=0.1,
                    steps=10, state=lambda: bssn_noise(n, n, n))
    if index == 3:
        n = scale or 256
        return dict(system=SYS_BSSN, dims=(n, n, n), ghost=3, order=4, dx=0.05, eps_diss=0.1,
                    steps=10, state=lambda: bssn_gaussians(n, n, n))
    raise ValueError("configs[4] is a sweep; see SWEEP_GRIDS")


SWEEP_GRIDS = [(96, 96, 96), (160, 160, 160), (200, 200, 400)]  # (nx, ny, nz)
