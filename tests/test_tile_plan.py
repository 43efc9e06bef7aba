"""Host logic of the persistent tiled kernels (pf_krylov_tma.cu): the decomposition that pf_tile_plan reports -- equal
z chunks taken round-robin, or whole layers in step on most SMs plus the remaining planes split over the other SMs --
must cover every (tile, plane) exactly once, with non-empty segments, within the blocks it launches; the two-group
plan is only chosen where its longest block is shorter.  No device is touched.  The segment walk below restates the
description in include/pf_debug.h; the kernels' own iterator is checked on the GPU (bit-equality with the direct
kernels for every plan, tests/test_gpu_merged.py)."""
import pytest

from paper_1711_04060_b200 import pf

TX = 64


def segments(p, nz):
    """block -> list of (tile, z0, z1) as include/pf_debug.h describes them."""
    out = []
    for b in range(p["blocks"]):
        segs = []
        if p["mode"] == 0:
            for i in range(b, p["nitems"], p["blocks"]):
                z0 = (i // p["ntiles"]) * p["depth"]
                segs.append((i % p["ntiles"], z0, min(z0 + p["depth"], nz)))
        elif p["mode"] == 2:
            T = p["ntiles"]
            R, r = p["blocks"] - T, b - T
            L = T - R
            if b < T:
                segs.append((b, 0, p["depth"]))
            else:
                segs.append((r, p["zrest"], nz))
                dp = -(-p["erest"] // p["q"])
                if r < L * p["q"]:
                    z0 = p["zrest"] + (r // L) * dp
                    assert z0 < nz, "the plan names an empty piece"
                    segs.append((R + r % L, z0, min(z0 + dp, nz)))
        elif b < p["nitems"]:
            z0 = (b // p["ntiles"]) * p["depth"]
            segs.append((b % p["ntiles"], z0, min(z0 + p["depth"], p["zrest"])))
        else:
            pos = (b - p["nitems"]) * p["q"]
            end = min(pos + p["q"], p["ntiles"] * p["erest"])
            while pos < end:
                tile, zz = divmod(pos, p["erest"])
                ln = min(p["erest"] - zz, end - pos)
                segs.append((tile, p["zrest"] + zz, p["zrest"] + zz + ln))
                pos += ln
        out.append(segs)
    return out


def longest(segs):
    return max(sum(z1 - z0 + 2 for _, z0, z1 in s) for s in segs)


SHAPES = [(256, 256, 256), (128, 128, 128), (160, 160, 160), (192, 192, 192), (144, 144, 144), (512, 512, 512),
          (64, 29, 200), (130, 33, 96), (66, 53, 40), (64, 16, 8), (96, 100, 77), (255 + 1, 255, 255), (320, 64, 300),
          (320, 208, 90), (256, 300, 64), (64, 52, 40)]


@pytest.mark.parametrize("rows", [13, 16])
@pytest.mark.parametrize("mode", [-1, 0, 1, 2])
@pytest.mark.parametrize("sms", [148, 132, 7])
def test_plan_covers_every_tile_plane_once(rows, mode, sms):
    for nx, ny, nz in SHAPES:
        p = pf.pf_tile_plan(nx, ny, nz, rows, sms, mode)
        ntx, nty = -(-nx // TX), -(-ny // rows)
        assert p["ntx"] == ntx and p["ntiles"] == ntx * nty
        assert 1 <= p["blocks"] <= max(sms, 1) and p["mode"] in (0, 1, 2)
        if mode in (1, 2):
            assert p["mode"] in (0, mode)
        assert p["mode"] != 2 or rows == 13          # the kernels of mode 2 exist for the 13-row tiles
        if mode == 0:
            assert p["mode"] == 0
        segs = segments(p, nz)
        cover = {}
        for s in segs:
            for tile, z0, z1 in s:
                assert 0 <= tile < p["ntiles"] and 0 <= z0 < z1 <= nz, (nx, ny, nz, tile, z0, z1)
                for z in range(z0, z1):
                    assert (tile, z) not in cover, (nx, ny, nz, tile, z)
                    cover[(tile, z)] = 1
        assert len(cover) == p["ntiles"] * nz
        if p["mode"] == 2:
            # one block per tile for the lower layer; the other blocks start with the upper layer of one tile each
            T = p["ntiles"]
            assert p["blocks"] == sms and T < sms < 2 * T
            assert all(s == [(b, 0, p["depth"])] for b, s in enumerate(segs[:T]))
            assert all(s[0] == (r, p["zrest"], nz) for r, s in enumerate(segs[T:]))
        if p["mode"] == 1:
            # whole layers on tiles * full blocks, in step: equal depth, one segment each
            main = [s for s in segs[:p["nitems"]]]
            assert all(len(s) == 1 and s[0][2] - s[0][1] == p["depth"] for s in main)
            assert p["nitems"] % p["ntiles"] == 0 and p["nitems"] // p["ntiles"] >= 2


def test_two_group_plan_is_chosen_only_where_it_is_shorter():
    # 256^3 with 16-row tiles on 148 SMs: 64 tiles x 9 chunks = 4 rounds of 31 plane steps, against two layers of
    # 112 planes on 128 SMs with the last 32 planes split over the other 20
    eq = pf.pf_tile_plan(256, 256, 256, 16, 148, 0)
    auto = pf.pf_tile_plan(256, 256, 256, 16, 148, -1)
    assert eq["mode"] == 0 and auto["mode"] == 1
    l0, l1 = longest(segments(eq, 256)), longest(segments(auto, 256))
    assert l0 == 124 and l1 <= 0.97 * l0 and l1 >= 256 * 64 / 148
    # more tiles than half the SMs (512^3; 13-row tiles at 256^3): equal chunks
    assert pf.pf_tile_plan(512, 512, 512, 16, 148, -1)["mode"] == 0
    # 256^3 with 13-row tiles: 80 tiles, 11 chunks in 6 rounds = 156 steps against a lower layer on 80 blocks, the upper
    # layer of 68 tiles on the other 68 and the upper layer of the last 12 tiles in 5 pieces afterwards
    deep = pf.pf_tile_plan(256, 256, 256, 13, 148, -1)
    assert deep["mode"] == 2 and longest(segments(pf.pf_tile_plan(256, 256, 256, 13, 148, 0), 256)) == 156
    assert longest(segments(deep, 256)) <= 146
    for shape in SHAPES:
        for rows in (13, 16):
            a, e = pf.pf_tile_plan(*shape, rows, 148, -1), pf.pf_tile_plan(*shape, rows, 148, 0)
            if a["mode"] != 0:
                assert longest(segments(a, shape[2])) <= 0.97 * longest(segments(e, shape[2]))


def test_mode2_pieces_are_never_empty():
    """Every depth of the upper layer must split into non-empty pieces (the kernel derives the piece depth from their number)."""
    for nz in range(16, 400, 3):
        for (nx, ny, rows, sms) in ((256, 256, 13, 148), (320, 208, 13, 148), (256, 250, 13, 148), (64, 52, 13, 7), (256, 256, 13, 132)):
            p = pf.pf_tile_plan(nx, ny, nz, rows, sms, 2)
            segs = segments(p, nz)          # asserts on an empty piece
            assert sum(z1 - z0 for s in segs for _, z0, z1 in s) == p["ntiles"] * nz
