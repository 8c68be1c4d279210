"""the paper's tile cost model for the fused BSSN tiles -- the library's closed
form against the oracle's brute-force enumeration of the sectors a tile touches, and the properties the paper
states for its model.  CPU only: chemora_tile_cost is host arithmetic."""
import pytest

from oracle import tile_cost as oracle_cost

FUSED_IDS = [0, 1, 2, 3, 4]


@pytest.fixture(scope="module")
def binding():
    from paper_1307_6488_b200 import binding as b
    b.load()
    return b


@pytest.mark.parametrize("ghost", [3, 4, 5])
def test_requests_equal_the_enumeration_order4(binding, ghost):
    for tile in FUSED_IDS:
        shape = binding.tile_shape(tile)
        s, r, n = binding.tile_cost(4, ghost, tile)
        assert r == oracle_cost.requests(4, ghost, shape), (tile, shape)
        assert n == shape[0] * shape[1] * shape[2]
        assert s == pytest.approx(oracle_cost.sigma(4, ghost, shape), rel=1e-15)


@pytest.mark.parametrize("ghost", [5, 6])
def test_requests_equal_the_enumeration_order8(binding, ghost):
    shape = binding.tile_shape(0)
    s, r, n = binding.tile_cost(8, ghost, 0)
    assert r == oracle_cost.requests(8, ghost, shape)
    assert s == pytest.approx(oracle_cost.sigma(8, ghost, shape), rel=1e-15)


def test_enumeration_does_not_depend_on_the_tile_column():
    """tx * 8 bytes is a multiple of the sector size for every tile: the alignment is that of column 0"""
    for shape in [(16, 4, 4), (8, 4, 8)]:
        assert len({oracle_cost.requests(4, 3, shape, column=c) for c in (0, 1, 2, 5)}) == 1


def test_hand_count_16x4x4():
    """16 x 4 x 4 at 4th order, g = 3 (xo = 3, boxes start at column 0): a 22-double box row covers 6 sectors, an
    18-double tile-box row starting at column 2 covers 5, a 16-double store row starting at column 3 covers 5:
    25*10*10*6 + 21*16*5 + 50*16*5 + 50*16*5 = 24680."""
    assert oracle_cost.requests(4, 3, (16, 4, 4)) == 25 * 100 * 6 + 21 * 16 * 5 + 50 * 16 * 5 + 50 * 16 * 5


def test_model_properties(binding):
    """what the paper says of its model: partially used lines favour tiles long in x -- among the
    256-point tiles with the same halo volume the 16-wide one requests fewer sectors per useful double in its box
    rows; and the small-tile factor makes the 128-point tile dearer than any 256-point one"""
    cost = {t: binding.tile_cost(4, 3, t) for t in FUSED_IDS}
    eff16 = 22 / (4.0 * 6)      # useful doubles per fetched double in a box row, tx = 16
    eff8 = 14 / (4.0 * 4)
    assert eff16 > eff8
    assert all(cost[4][0] > cost[t][0] for t in (0, 1, 2, 3))
    for t in (5, 6, 8, 11, -1):
        with pytest.raises(binding.ChemoraError):
            binding.tile_cost(4, 3, t)
    with pytest.raises(binding.ChemoraError):
        binding.tile_cost(8, 5, 1)
    with pytest.raises(binding.ChemoraError):
        binding.tile_cost(4, 2, 0)
