"""CPU check of the sampled-parity method of test_gpu_fullsize.py: the oracle run on a periodic block cut around
a sample reproduces, bit for bit, the centre of the oracle run on the whole grid (domain of dependence 12 n cells)."""
import numpy as np

from paper_1307_6488_b200 import inputs
from tests.test_gpu_z_fullsize import cut


def test_cut_block_reproduces_full_run(oracle):
    n, g, dx, steps = 40, 3, 0.05, 1
    u0 = inputs.bssn_gaussians(n, n, n, width_cells=5.0)
    u0 += 1e-6 * np.random.default_rng(3).uniform(-1, 1, u0.shape)
    prm = oracle.params(eps_diss=0.1)
    full = oracle.interior(oracle.rk4(oracle.SYS_BSSN, oracle.with_ghosts(u0, g), g, 4, dx, 0.25 * dx, prm, steps), g)
    reach, core = 12 * steps, 3
    for c in [(0, 0, 0), (39, 20, 5)]:
        blk = cut(u0, c, core + reach)
        st = oracle.interior(oracle.rk4(oracle.SYS_BSSN, oracle.with_ghosts(blk, g), g, 4, dx, 0.25 * dx, prm, steps), g)
        want = st[:, reach:reach + 2 * core, reach:reach + 2 * core, reach:reach + 2 * core]
        assert np.array_equal(cut(full, c, core), want)
        # one cell less of reach is not enough: the method's bound is tight, so it is really being exercised
        assert not np.array_equal(cut(full, c, core + 1)[:, :1], st[:, reach - 1:reach, reach - 1:reach + 2 * core + 1,
                                                                    reach - 1:reach + 2 * core + 1])
