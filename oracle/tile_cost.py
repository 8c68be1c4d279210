"""Oracle of the tile cost model (test infrastructure only; nothing in the product imports it).

PAPER.md:254-262: for a candidate tile the number of cache lines requested during the execution of the kernel is
computed ("request size"; under the assumption that all lines survive it is "the number of distinct lines the kernel
will touch, after accounting for many special cases such as alignment"), normalised to the number of grid points,
r / (I tx ty tz), and corrected for "the lower execution efficiency with smaller tiles" by the empirical factor
1 / (1 + 256 / (tx ty tz)).

Written out by brute force: the tile is placed on an actual padded layout, every double it reads or writes is
enumerated access kind by access kind, and the distinct 32-byte sectors of each kind are counted with a set.
Reading S15: the efficiency DIVIDES the cost, sigma = (r / points) * (1 + 256 / (tx ty tz)).
"""


def layout(nx, ghost):
    """x offset of interior point 0 and row pitch in doubles (include/chemora.h, "Conventions")."""
    xo = ghost + 1 if (ghost - 3) % 2 else ghost
    pitch = (xo + nx + ghost + 15) // 16 * 16
    return xo, pitch


def requests(fd_order, ghost, tile, nx=256, ny=64, nz=64, column=1):
    """distinct 32-byte sectors one interior tile of a middle Runge-Kutta stage of the fused BSSN kernel requests"""
    tx, ty, tz = tile
    H = fd_order // 2 + 1
    xo, pitch = layout(nx, ghost)
    tot_y = ny + 2 * ghost
    x0, y0, z0 = xo + column * tx, ghost + ty, ghost + tz        # padded coordinates of the tile's first point

    def count(nvars, xr, yr, zr):
        seen = set()
        for v in range(nvars):
            for k in zr:
                for j in yr:
                    row = ((v * (nz + 2 * ghost) + k) * tot_y + j) * pitch
                    for i in xr:
                        seen.add((row + i) * 8 // 32)
        return len(seen)

    box = count(25, range(x0 - H, x0 + tx + H), range(y0 - H, y0 + ty + H), range(z0 - H, z0 + tz + H))
    wide = (range(x0 - 1, x0 + tx + 1), range(y0, y0 + ty), range(z0, z0 + tz))   # TMA tile boxes: one column each side
    cen = count(21, *wide)
    operands = 2 * count(25, *wide)
    stores = 2 * count(25, range(x0, x0 + tx), range(y0, y0 + ty), range(z0, z0 + tz))
    return box + cen + operands + stores


def sigma(fd_order, ghost, tile, **kw):
    tx, ty, tz = tile
    n = tx * ty * tz            # I = 1
    return (requests(fd_order, ghost, tile, **kw) / n) * (1.0 + 256.0 / n)
