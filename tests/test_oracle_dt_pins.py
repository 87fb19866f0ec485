"""Pins of the one rule of reading c-7 that no other pin reaches: an axis with a single cell takes no part in the CFL
minimum  dt = cfl * min_d(Delta_d / cmax_d)  (oracle/smaug_oracle.cpp cfl_dt, oracle/smaug3d_oracle.cpp cfl_dt;
PAPER.md is silent on dt, north_star wants "a y-invariant 2D Brio-Wu run matching the 1D run cell for cell").

The collapsed axis is made SHORT (L = 1e-3 over one cell), so that Delta_d / cmax_d along it would be the minimum by a
factor of ten or more if it were counted: removing `if (c.ny > 1)` / `if (c.n[d] > 1)` from either oracle fails these.
Expected values are the textbook fast speed of a uniform state typed here, and bit-equality of two runs.  CPU only."""
import numpy as np
import pytest

import oracle
import smaug_inputs as si

RHO, P0, GAMMA = 1.3, 0.7, 1.4


def fast_speed(v_d, b_d, b2):
    a2, s = GAMMA * P0 / RHO, GAMMA * P0 / RHO + b2 / RHO
    return abs(v_d) + np.sqrt(0.5 * (s + np.sqrt(s * s - 4 * a2 * b_d * b_d / RHO)))


@pytest.mark.parametrize("nx,ny,lx,ly", [(64, 1, 1.0, 1e-3), (1, 64, 1e-3, 1.0), (64, 1, 2.0, 1e-4), (5, 4, 1.0, 1e-3)])
def test_dt_of_a_uniform_flow_ignores_a_one_cell_axis_2d(oracle_mod, nx, ny, lx, ly):
    v, B = (0.3, -0.2), (0.4, -0.6)
    w = si.prim_to_cons(RHO * np.ones((ny, nx)), v[0], v[1], P0, B[0], B[1], GAMMA)
    o = oracle_mod.Oracle(nx, ny, GAMMA, (0, 0, 0, 0), lx=lx, ly=ly)
    o.set_state(w)
    o.step(1, 0.4)
    b2 = B[0] ** 2 + B[1] ** 2
    terms = [L / n / fast_speed(v[d], B[d], b2) for d, (n, L) in enumerate(((nx, lx), (ny, ly))) if n > 1]
    assert np.isclose(o.time()[1], 0.4 * min(terms), rtol=1e-13), (o.time(), terms)
    if nx == 5:                                  # both axes count here, and the short y axis decides
        assert min(terms) == terms[1] < 0.1 * terms[0]
    o.close()


def test_brio_wu_1d_does_not_depend_on_the_length_of_its_one_cell_axis(oracle_mod):
    """With ny = 1 every y-difference vanishes, so L_y can only enter through dt: the runs agree bit for bit exactly
    when the y axis is left out of the minimum (and the x <-> y mirrored problem likewise)."""
    w, bc, gamma = si.brio_wu(64, 1)
    runs = []
    for ly in (1.0, 1e-3):
        o = oracle_mod.Oracle(64, 1, gamma, bc, ly=ly)
        o.set_state(w)
        o.step(10, 0.3)
        runs.append((o.get_state(), o.time()))
        o.close()
    assert np.array_equal(runs[0][0], runs[1][0]) and runs[0][1] == runs[1][1]
    wt, bct, _ = si.brio_wu(64, 1, transpose=True)
    o = oracle_mod.Oracle(1, 64, gamma, bct, lx=1e-3)
    o.set_state(wt)
    o.step(10, 0.3)
    assert o.time() == runs[0][1]
    o.close()


@pytest.mark.parametrize("shape,L", [((1, 5, 4), (1.0, 2.0, 1e-3)), ((6, 1, 1), (1e-3, 1e-3, 3.0)), ((5, 1, 4), (1.0, 1e-3, 0.5)),
                                     ((3, 5, 4), (1.0, 2.0, 1e-3))])
def test_dt_of_a_uniform_flow_ignores_one_cell_axes_3d(shape, L):
    nz, ny, nx = shape
    v, B = (0.3, -0.2, 0.5), (0.4, 0.1, -0.6)
    w = si.prim_to_cons3(RHO * np.ones(shape), v, P0, B, GAMMA)
    o = oracle.Oracle3D(nx, ny, nz, GAMMA, (0,) * 6, lx=L[0], ly=L[1], lz=L[2])
    o.set_state(w)
    o.step(1, 0.4)
    n, b2 = (nx, ny, nz), sum(b * b for b in B)
    terms = {d: L[d] / n[d] / fast_speed(v[d], B[d], b2) for d in range(3) if n[d] > 1}
    assert np.isclose(o.time()[1], 0.4 * min(terms.values()), rtol=1e-13), (o.time(), terms)
    if nz == 3:                                  # three cells along z: the short axis counts and decides
        assert min(terms.values()) == terms[2]
    o.close()
