"""CPU test of the decomposition logic: where every ghost cell of every
sub-domain takes its value from (smaug_group_map_cell, the same host/device function the exchange kernel runs), against
numpy: the GLOBAL array padded x first, then y over the padded width (reading c-8) must hold, at the ghost cell's
global position, the value of the source cell the mapping names.  Needs no GPU."""
import numpy as np
import pytest

import paper_1710_06423_b200 as pkg

MODE = {0: "wrap", 1: "edge", 2: "edge"}       # fixed == edge at freeze time (set_state)


def _blocks(n, p):
    return [a * n // p for a in range(p + 1)]


@pytest.mark.parametrize("px,py,nx,ny", [(2, 1, 11, 7), (1, 2, 7, 10), (2, 2, 10, 9), (3, 2, 13, 8), (4, 1, 5, 1), (3, 3, 4, 5)])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 1, 1, 1), (2, 2, 0, 0), (0, 0, 1, 2), (1, 2, 2, 1)])
def test_every_ghost_cell_maps_to_the_cell_numpy_pad_copies(px, py, nx, ny, bc):
    rng = np.random.default_rng(7)
    g = rng.normal(size=(ny, nx))
    pad = np.pad(np.pad(g, ((0, 0), (3, 3)), mode=MODE[bc[0]] if bc[0] == bc[1] else "edge"), ((3, 3), (0, 0)),
                 mode=MODE[bc[2]] if bc[2] == bc[3] else "edge")
    if bc[0] != bc[1] or bc[2] != bc[3]:          # open on one side, fixed on the other: both are 'edge' at freeze
        assert 0 not in (bc[0], bc[1]) or bc[0] == bc[1]
    x0, y0 = _blocks(nx, px), _blocks(ny, py)
    for m in range(px * py):
        a, b = m % px, m // px
        mnx, mny = x0[a + 1] - x0[a], y0[b + 1] - y0[b]
        for j in range(-3, mny + 3):
            for i in range(-3, mnx + 3):
                if 0 <= i < mnx and 0 <= j < mny:
                    continue
                (bx0, by0, bnx, bny), (sm, si, sj) = pkg.group_map_cell(px, py, nx, ny, bc, m, i, j, freeze=1)
                assert (bx0, by0, bnx, bny) == (x0[a], y0[b], mnx, mny)
                assert sm >= 0
                sa, sb = sm % px, sm // px
                assert 0 <= si < x0[sa + 1] - x0[sa] and 0 <= sj < y0[sb + 1] - y0[sb]      # an interior cell of its owner
                assert g[y0[sb] + sj, x0[sa] + si] == pad[y0[b] + j + 3, x0[a] + i + 3]


def test_fixed_sides_are_never_rewritten_and_their_corners_read_frozen_ghosts():
    px, py, nx, ny = 2, 2, 10, 8
    bc = (2, 2, 0, 0)                               # fixed in x, periodic in y
    x0, y0 = _blocks(nx, px), _blocks(ny, py)
    for m in range(4):
        a, b = m % px, m // px
        mnx, mny = x0[a + 1] - x0[a], y0[b + 1] - y0[b]
        for j in range(-3, mny + 3):
            for i in range(-3, mnx + 3):
                if 0 <= i < mnx and 0 <= j < mny:
                    continue
                _, (sm, si, sj) = pkg.group_map_cell(px, py, nx, ny, bc, m, i, j, freeze=0)
                I, J = x0[a] + i, y0[b] + j
                outside_x = I < 0 or I >= nx
                if outside_x and 0 <= J < ny:
                    assert sm == -1                   # a frozen ghost of the global x-side: left alone
                elif outside_x:
                    # corner of the global grid: wraps in y and copies the FROZEN ghost of the member owning that row
                    sa, sb = sm % px, sm // px
                    assert sa == a and (si < 0 or si >= x0[sa + 1] - x0[sa]) and 0 <= sj < y0[sb + 1] - y0[sb]
                    assert x0[sa] + si == I and y0[sb] + sj == J % ny
                else:
                    sa, sb = sm % px, sm // px     # internal boundary or periodic y: an interior cell of the owner
                    assert x0[sa] + si == I and y0[sb] + sj == J % ny
    # fixed in y: whole ghost rows (corners included) stay frozen
    for i in range(-3, 8):
        assert pkg.group_map_cell(2, 1, 10, 8, (0, 0, 2, 2), 0, i, -1, freeze=0)[1][0] == -1


def test_group_argument_validation_needs_no_gpu():
    import ctypes as C
    L = pkg.lib()
    h = C.c_void_p()
    bc = (C.c_int * 4)(0, 0, 0, 0)
    assert L.smaug_group_create(0, 1, 8, 8, 1.4, bc, None, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_group_create(9, 1, 80, 8, 1.4, bc, None, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_group_create(4, 1, 3, 8, 1.4, bc, None, None, C.byref(h)) == pkg.EINVAL       # a block would be empty
    assert L.smaug_group_create(2, 2, 8, 8, 1.4, (C.c_int * 4)(0, 1, 0, 0), None, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_group_step(None, 1, 0.3) == pkg.EINVAL
    L.smaug_group_destroy(None)
