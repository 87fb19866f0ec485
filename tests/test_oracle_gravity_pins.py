"""Pins of the oracle's gravity terms (reading c-10; "rho g", "rho g.v") against
closed forms and invariants -- none re-types the oracle's formula.  All CPU, `-m "not gpu"`.

  G1  a hydrostatic background with zero perturbation stays exactly static (bitwise): in the split form gravity
      acts on the PERTURBED density only (a version using the total density fails this).
  G2  free fall of a uniform gas on a zero background under uniform g: m = rho g t, e = e0 + rho g^2 t^2 / 2,
      rho, B unchanged; RK4 integrates these polynomials exactly (pins sign and coefficient of both sources, for
      both components, and that the energy source uses g.v).
  G3  PAPER.md:35 as printed (zero background): an isothermal hydrostatic column dp/dy = rho g_y is stationary
      up to the truncation error of the 4th-order central difference (pins the sign of g against grad p).
  G4  split == unsplit: the same total stratified state as (background + perturbation) and as (zero background,
      everything in the perturbation) has the same RHS up to O(h^4) (pins rho~ vs rho in both equations).
"""
import numpy as np
import pytest

import smaug_inputs as si

PER = (0, 0, 0, 0)


@pytest.mark.parametrize("hd_on", [0, 1])
def test_G1_hydrostatic_background_is_exactly_static(oracle_mod, hd_on):
    nx, ny = 12, 40
    w, bc, gamma, bg, (gx, gy) = si.stratified_atmosphere(nx, ny, pulse=0.0)
    assert not w.any()
    o = oracle_mod.Oracle(nx, ny, gamma, bc, bg=bg, gx=gx, gy=gy, hd_on=hd_on, fixed_dt=1e-3)
    o.set_state(w)
    assert not o.rhs().any()
    o.step(5)
    assert not o.get_state().any()
    o.close()


@pytest.mark.parametrize("g", [(0.0, -1.3), (0.7, 0.0), (0.4, -0.9)])
def test_G2_free_fall_closed_form(oracle_mod, g):
    nx, ny, gamma = 8, 6, 5.0 / 3.0
    rho, p, bx, by = 0.8, 0.6, 0.2, -0.1
    w = si.prim_to_cons(rho * np.ones((ny, nx)), 0.0, 0.0, p, bx, by, gamma)
    dt, n = 2e-3, 25
    o = oracle_mod.Oracle(nx, ny, gamma, PER, gx=g[0], gy=g[1], fixed_dt=dt)
    o.set_state(w)
    o.step(n)
    out = o.get_state()
    o.close()
    T = n * dt
    e0 = p / (gamma - 1) + 0.5 * (bx * bx + by * by)
    assert np.abs(out[0] - rho).max() == 0.0
    assert np.abs(out[1] - rho * g[0] * T).max() < 1e-15
    assert np.abs(out[2] - rho * g[1] * T).max() < 1e-15
    assert np.abs(out[3] - (e0 + 0.5 * rho * (g[0] ** 2 + g[1] ** 2) * T * T)).max() < 1e-14
    assert np.abs(out[4] - bx).max() == 0.0 and np.abs(out[5] - by).max() == 0.0
    # and the sources really are there (g = 0 leaves the state untouched)
    assert np.abs(out[1]).max() + np.abs(out[2]).max() > 1e-2


def _interior(a, m=4):
    return a[..., m:-m, :]


def test_G3_hydrostatic_column_of_the_printed_equations_to_fourth_order(oracle_mod):
    errs = []
    for ny in (32, 96):
        w, bc, gamma, bg, (gx, gy) = si.stratified_atmosphere(8, ny, pulse=0.0, split=False)
        assert bg is None
        o = oracle_mod.Oracle(8, ny, gamma, bc, gx=gx, gy=gy, hd_on=0)
        o.set_state(w)
        R = o.rhs()
        o.close()
        # away from the open boundaries (whose zero-gradient ghosts are not the analytic continuation)
        scale = np.abs(w[0] * gy).max()                      # |rho g|: the size of each of the two balancing terms
        errs.append(np.abs(_interior(R[2])).max() / scale)
        assert np.abs(_interior(R[[0, 1, 3, 4, 5]])).max() == 0.0      # v = 0: nothing else moves
        # with the sign of g flipped the two terms add instead of cancelling
        o = oracle_mod.Oracle(8, ny, gamma, bc, gx=gx, gy=-gy, hd_on=0)
        o.set_state(w)
        assert np.abs(_interior(o.rhs()[2])).max() / scale > 0.1
        o.close()
    assert errs[0] < 1e-3 and errs[0] / errs[1] > 40, errs            # 3^4 = 81 asymptotically


def test_G4_split_equals_unsplit_on_a_stratified_atmosphere(oracle_mod):
    errs = []
    for n in (32, 96):
        ws, bc, gamma, bg, (gx, gy) = si.stratified_atmosphere(n, n, pulse=5e-2)
        wf = si.stratified_atmosphere(n, n, pulse=5e-2, split=False)[0]
        o_s = oracle_mod.Oracle(n, n, gamma, bc, bg=bg, gx=gx, gy=gy, hd_on=0)
        o_f = oracle_mod.Oracle(n, n, gamma, bc, gx=gx, gy=gy, hd_on=0)
        o_s.set_state(ws); o_f.set_state(wf)
        rs, rf = _interior(o_s.rhs()), _interior(o_f.rhs())
        o_s.close(); o_f.close()
        # per field, relative to that field's own RHS size (my: relative to |rho g|, the balancing terms)
        e = [np.abs(rs[f] - rf[f]).max() / max(np.abs(rf[f]).max(), 1e-300) for f in (0, 1, 3, 5)]
        e.append(np.abs(rs[2] - rf[2]).max() / np.abs(wf[0] * gy).max())
        errs.append(max(e))
    assert errs[0] < 1e-2 and errs[0] / errs[1] > 40, errs
    # a version that applied g to the total density in the split form would differ by rho_b g: O(1) relative
