"""Host logic of the cooperative kernel (pf_krylov_coop.cu): the brick decomposition that
pf_coop_plan reports must tile the box exactly with non-empty bricks, respect the block and shared-memory limits it
was given, and say "does not fit" for grids whose bricks are too large.  No device is touched."""
import itertools

import pytest

from paper_1711_04060_b200 import pf

SM, CAP = 148, 223 * 1024


def brick_bounds(n, nb):
    return [(k * n // nb, (k + 1) * n // nb) for k in range(nb)]


def smem_bytes(v, h, nh):
    # six vectors of own nodes, codes, global indices, 16-bit operand indices; diagonal and operand with halo;
    # the halo list (pf_krylov_coop.cu coop_smem_bytes)
    return v * (6 * 8 + 4 + 4 + 2) + h * 16 + nh * 8 + 16


@pytest.mark.parametrize("shape", [(3, 3, 3), (5, 4, 3), (32, 32, 32), (37, 20, 11), (40, 40, 40), (48, 48, 48),
                                   (64, 64, 64), (7, 150, 9), (200, 3, 3), (64, 16, 40), (33, 35, 31)])
def test_plan_tiles_the_box(shape):
    nx, ny, nz = shape
    p = pf.pf_coop_plan(nx, ny, nz, SM, CAP)
    assert p is not None, shape
    nb = (p["nbx"], p["nby"], p["nbz"])
    assert 1 <= nb[0] * nb[1] * nb[2] <= SM
    assert all(1 <= b <= n for b, n in zip(nb, shape))
    # every node belongs to exactly one brick; no brick is empty; extents cover the largest brick
    vmax = hmax = nhmax = 0
    count = 0
    for (x0, x1), (y0, y1), (z0, z1) in itertools.product(brick_bounds(nx, nb[0]), brick_bounds(ny, nb[1]),
                                                          brick_bounds(nz, nb[2])):
        bx, by, bz = x1 - x0, y1 - y0, z1 - z0
        assert bx >= 1 and by >= 1 and bz >= 1
        count += bx * by * bz
        vmax = max(vmax, bx * by * bz)
        hmax = max(hmax, (bx + 2) * (by + 2) * (bz + 2))
        nhmax = max(nhmax, 2 * (bx * by + by * bz + bx * bz))
    assert count == nx * ny * nz
    for axis, n in enumerate(shape):                   # consecutive bricks along an axis share their bounds
        b = brick_bounds(n, nb[axis])
        assert b[0][0] == 0 and b[-1][1] == n and all(b[i][1] == b[i + 1][0] for i in range(len(b) - 1))
    assert p["vmax"] >= vmax and p["vmax"] % 2 == 0 and p["hmax"] >= hmax and p["nhmax"] >= nhmax
    assert p["hmax"] <= 65535                                        # operand indices are 16-bit
    assert p["threads"] in (256, 512, 1024) and p["threads"] >= SM    # one record per thread at the barrier
    assert p["smem"] == smem_bytes(p["vmax"], p["hmax"], p["nhmax"]) <= CAP


def test_plan_limits():
    assert pf.pf_coop_plan(128, 128, 128, SM, CAP) is None            # 14 000 nodes per SM do not fit
    assert pf.pf_coop_plan(64, 64, 64, SM, 64 * 1024) is None         # nor 64^3 in 64 KB per block
    assert pf.pf_coop_plan(64, 64, 64, 8, CAP) is None                # nor on 8 SMs
    small = pf.pf_coop_plan(32, 32, 32, 8, CAP)                       # 32^3 fits neither: 4096 nodes per brick
    assert small is None
    p16 = pf.pf_coop_plan(16, 16, 16, 8, CAP)
    assert p16 is not None and p16["nbx"] * p16["nby"] * p16["nbz"] <= 8
    assert pf.pf_coop_plan(2, 8, 8, SM, CAP) is None                  # invalid grid
    # the fewer blocks, the larger the bricks
    a, b = pf.pf_coop_plan(40, 40, 40, 148, CAP), pf.pf_coop_plan(40, 40, 40, 64, CAP)
    assert a["vmax"] <= b["vmax"]


def test_plan_prefers_long_bricks_in_x_on_ties():
    p = pf.pf_coop_plan(64, 64, 64, SM, CAP)
    assert (p["nbx"], p["nby"], p["nbz"]) == (4, 6, 6)
