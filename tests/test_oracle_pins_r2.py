"""Round-2 pins of the CPU oracle: the parts the round-1 review found unpinned by mutation testing.

  M1-M4  energy coupling of the MIXED hyperdiffusive fluxes (DESIGN.md c-5): G(e;k) = v_l G(m_l;k) +
         B_l G(b_l;k).  A uniform drift v_x0 (uniform field B_x0) multiplies the mixed momentum (magnetic) flux
         whose closed form tests/test_oracle_pins.py::test_hd_mixed_terms_closed_form already pins, so the
         viscous (ohmic) part of R_e must contain v_x0 (B_x0) times that closed form; plus the x<->y mirror.
  F1-F2  "fixed" ghosts during the steps (c-8; PAPER.md:59 halo layers): the whole ghost strip of a fixed side,
         corners included, is bitwise what set_state left there after a pulse has run into it, and the interior
         then differs from the open-boundary run of the same state.
  R1     rhs() of a flowing, magnetised, non-linear smooth state (HD off, zero background) against PAPER.md:35
         differentiated analytically (product rule carried by first-order jets), converging at 4th order.

None re-types a formula of oracle/smaug_oracle.cpp: expectations are closed forms (1-D nu ratios pinned by P8-P10,
the modified wavenumber k*), invariants of reading c-8, and the paper's vector equations.  Each was checked to
fail on the seeded mistake it is there for (listed in the docstrings).  All CPU, `-m "not gpu"`.
"""
import math

import numpy as np
import pytest

import smaug_inputs as si

PER = (0, 0, 0, 0)


def _rhs(oracle_mod, prim, gamma, bc=PER, **params):
    w = si.prim_to_cons(prim["rho"], prim["vx"], prim["vy"], prim["p"], prim["bx"], prim["by"], gamma)
    ny, nx = w.shape[1:]
    o = oracle_mod.Oracle(nx, ny, gamma, bc, **params)
    o.set_state(w)
    r = o.rhs()
    o.close()
    return r


def _rhs_t(oracle_mod, prim, gamma, **params):
    """R of the x<->y mirrored problem, mirrored back (so that it can be compared with the same closed form)."""
    t = dict(rho=prim["rho"].T, p=prim["p"].T, vx=prim["vy"].T, vy=prim["vx"].T, bx=prim["by"].T, by=prim["bx"].T)
    t = {k: np.ascontiguousarray(v) for k, v in t.items()}
    return si.transpose_state(_rhs(oracle_mod, t, gamma, **params))


def _kstar(n):
    kh = 2 * math.pi / n
    return (8 * math.sin(kh) - math.sin(2 * kh)) / 6 * n      # L = 1


def _mixed_setup(oracle_mod, nx, ny):
    """a(x) g(y) = sin(2 pi x) (1 + 0.3 cos(2 pi y)) and the 1-D ingredients of its closed forms."""
    x, y = si.centres(nx)[None, :], si.centres(ny)[:, None]
    a, g = np.sin(2 * np.pi * x), 1 + 0.3 * np.cos(2 * np.pi * y)
    line_x = np.sin(2 * np.pi * (np.arange(-3, nx + 3) + 0.5) / nx)
    line_y = 1 + 0.3 * np.cos(2 * np.pi * (np.arange(-3, ny + 3) + 0.5) / ny)
    ratio_x = oracle_mod.hyper_nu_1d(line_x, 1.0, 1.0, 1.0)        # M3/M1 at interfaces -1/2 .. nx-1/2 (P8-P10)
    ratio_y = oracle_mod.hyper_nu_1d(line_y, 1.0, 1.0, 1.0)
    rbar_x = 0.5 * (ratio_x[:-1] + ratio_x[1:])[None, :]
    dcx_a = _kstar(nx) * np.cos(2 * np.pi * x)                      # d^c_x a
    dcy_g = -0.3 * _kstar(ny) * np.sin(2 * np.pi * y)               # d^c_y g
    return a, g, ratio_x, ratio_y, rbar_x, dcx_a, dcy_g


@pytest.mark.parametrize("mirror", [False, True])
def test_M1_mixed_viscous_flux_carries_energy_with_the_drift(oracle_mod, mirror):
    """v_y = a(x) g(y) on a uniform drift v_x = U: the only viscous term that knows about U is the energy flux
    v_x G(m_x; y) of the mixed stress, so [R_e(c_mom) - R_e(0)](U) - [..](0) = U d^c_y{ rho/2 nubar_x(v_y) d^c_x v_y }
    = U * (closed form of the mixed R_mx).  Fails if G(e;k) is dropped, or uses v_k instead of v_l."""
    nx, ny, gamma, c_mom, rho0, p0, U = 32, 16, 1.4, 0.4, 0.8, 0.5, 0.37
    a, g, ratio_x, ratio_y, rbar_x, dcx_a, dcy_g = _mixed_setup(oracle_mod, nx, ny)
    one = np.ones((ny, nx))
    rhs = _rhs_t if mirror else _rhs

    def visc(u):
        prim = dict(rho=rho0 * one, vx=u * one, vy=a * g * one, p=p0 * one, bx=0 * one, by=0 * one)
        return rhs(oracle_mod, prim, gamma, c_mom=c_mom) - rhs(oracle_mod, prim, gamma, c_mom=0.0)

    vt = math.sqrt(gamma * p0 / rho0)
    mixed_mx = 0.5 * rho0 * c_mom * (1.0 / nx) * vt * rbar_x * dcx_a * dcy_g      # pinned for U = 0 in round 1
    d0, dU = visc(0.0), visc(U)
    scale = np.abs(mixed_mx).max()
    assert scale > 1e-6
    assert np.abs(d0[1] - mixed_mx).max() < 1e-9 * scale
    assert np.abs(dU[1] - mixed_mx).max() < 1e-9 * scale                          # momentum part does not see U
    assert np.abs((dU[3] - d0[3]) - U * mixed_mx).max() < 1e-9 * U * scale
    # and in full: R_e = U*mixed + interface work d_x{ vbar_y Phi_x(m_y) } + d_y{ vbar_y Phi_y(m_y) },
    # Phi_x = (rho/2) nu_x (v_y[i+1]-v_y[i])/dx,  Phi_y = rho nu_y (v_y[j+1]-v_y[j])/dy  (nu from the 1-D ratios)
    vy = a * g * one
    nu_x = c_mom * (1.0 / nx) * vt * ratio_x[1:][None, :]
    nu_y = c_mom * (1.0 / ny) * vt * ratio_y[1:][:, None]
    phx = 0.5 * rho0 * nu_x * (np.roll(vy, -1, 1) - vy) * nx
    phy = rho0 * nu_y * (np.roll(vy, -1, 0) - vy) * ny
    wx = 0.5 * (vy + np.roll(vy, -1, 1)) * phx
    wy = 0.5 * (vy + np.roll(vy, -1, 0)) * phy
    work = (wx - np.roll(wx, 1, 1)) * nx + (wy - np.roll(wy, 1, 0)) * ny
    assert np.abs(dU[3] - (U * mixed_mx + work)).max() < 1e-9 * np.abs(work).max()
    assert np.abs(dU[2] - ((phx - np.roll(phx, 1, 1)) * nx + (phy - np.roll(phy, 1, 0)) * ny)).max() < 1e-9 * np.abs(phx).max() * nx
    for f in (0, 4, 5):
        assert not dU[f].any()


@pytest.mark.parametrize("mirror", [False, True])
def test_M2_mixed_resistive_flux_carries_energy_with_the_field(oracle_mod, mirror):
    """b_y = a(x) g(y) in a uniform B_x = B0, gas at rest: R_bx(c_b) - R_bx(0) is the mixed term alone and
    R_e(c_b) - R_e(0) = B0 * (that closed form) + d_x{ Bbar_y Phi_x(b_y) }.  Fails if the ohmic part of G(e;k) is
    dropped or uses B_k instead of B_l."""
    nx, ny, gamma, c_b, rho0, p0, B0 = 32, 16, 1.4, 0.02, 0.8, 0.5, 0.45
    a, g, ratio_x, ratio_y, rbar_x, dcx_a, dcy_g = _mixed_setup(oracle_mod, nx, ny)
    one = np.ones((ny, nx))
    by = a * g * one
    prim = dict(rho=rho0 * one, vx=0 * one, vy=0 * one, p=p0 * one, bx=B0 * one, by=by)
    rhs = _rhs_t if mirror else _rhs
    d = rhs(oracle_mod, prim, gamma, c_b=c_b) - rhs(oracle_mod, prim, gamma, c_b=0.0)
    vt = math.sqrt(gamma * p0 / rho0) + math.sqrt((B0 ** 2 + by ** 2).max() / rho0)
    mixed_bx = -c_b * (1.0 / nx) * vt * rbar_x * dcx_a * dcy_g
    scale = np.abs(mixed_bx).max()
    assert scale > 1e-7
    assert np.abs(d[4] - mixed_bx).max() < 1e-9 * scale
    nu_x = c_b * (1.0 / nx) * vt * ratio_x[1:][None, :]
    phx = nu_x * (np.roll(by, -1, 1) - by) * nx
    ex = 0.5 * (by + np.roll(by, -1, 1)) * phx
    ohm_x = (ex - np.roll(ex, 1, 1)) * nx
    assert np.abs(d[3] - (B0 * mixed_bx + ohm_x)).max() < 1e-9 * max(np.abs(ohm_x).max(), B0 * scale)
    assert np.abs(B0 * mixed_bx).max() > 1e-3 * np.abs(ohm_x).max()             # the coupling is visible in the sum
    assert np.abs(d[5] - (phx - np.roll(phx, 1, 1)) * nx).max() < 1e-9 * np.abs(phx).max() * nx
    for f in (0, 1, 2):
        assert not d[f].any()


# ----------------------------------------------------------------------------- fixed ghosts during the steps (c-8)
def _pulse(nx, ny, gamma=1.4):
    x = si.centres(nx)[None, :] * np.ones((ny, 1))
    y = si.centres(ny)[:, None] * np.ones((1, nx))
    bump = np.exp(-((x - 0.8) ** 2 + (y - 0.75) ** 2) / (2 * 0.07 ** 2))
    return si.prim_to_cons(1.0 + 0.3 * bump, 0.2 * bump, -0.1 * bump, 0.6 * (1 + 0.5 * bump), 0.2 + 0 * x,
                           0.1 + 0.05 * bump, gamma), gamma


@pytest.mark.parametrize("bc", [(2, 2, 0, 0), (0, 0, 2, 2), (1, 2, 1, 2), (2, 2, 2, 2), (1, 2, 0, 0)])
def test_F1_fixed_ghost_strips_are_frozen_bitwise_while_a_pulse_runs_into_them(oracle_mod, bc):
    """Reading c-8: the ghosts of a fixed side hold the nearest-interior value as of set_state and are never
    rewritten.  A pressure pulse next to the x_hi / y_hi sides reaches them within the run, so a fill that treats
    `fixed` like `open` during the steps (the seeded mistake) changes those ghosts and fails this."""
    nx, ny, steps = 40, 36, 60
    w, gamma = _pulse(nx, ny)
    o = oracle_mod.Oracle(nx, ny, gamma, bc)
    o.set_state(w)
    before = [o.padded(f).copy() for f in range(6)]
    o.step(steps, 0.3)
    after = [o.padded(f) for f in range(6)]
    out = o.get_state()
    o.close()
    strips = {0: np.s_[:, :3], 1: np.s_[:, -3:], 2: np.s_[:3, :], 3: np.s_[-3:, :]}      # whole strips: corners too
    for side, kind in enumerate(bc):
        for f in range(6):
            same = np.array_equal(after[f][strips[side]], before[f][strips[side]])
            if kind == 2:
                assert same, (side, f)
        if kind == 1 and side in (1, 3):                      # the pulse did reach this side: open ghosts moved
            assert not np.array_equal(after[0][strips[side]], before[0][strips[side]])
    # the boundary matters: the same state with the fixed sides opened ends up different in the interior
    bc_open = tuple(1 if k == 2 else k for k in bc)
    o = oracle_mod.Oracle(nx, ny, gamma, bc_open)
    o.set_state(w)
    o.step(steps, 0.3)
    ref = o.get_state()
    o.close()
    assert np.abs(out - ref).max() > 1e-6


def test_F2_fixed_ghosts_hold_the_set_state_edge_values(oracle_mod):
    """What is frozen is the nearest interior cell at set_state (np.pad 'edge'), per interior row on x-sides and
    over the full padded width on y-sides -- checked after the run, when the interior edge has long moved on."""
    nx, ny = 30, 26
    w, gamma = _pulse(nx, ny)
    o = oracle_mod.Oracle(nx, ny, gamma, (2, 2, 2, 2))
    o.set_state(w)
    o.step(40, 0.3)
    out = o.get_state()
    for f in range(6):
        ref0 = np.pad(np.pad(w[f], ((0, 0), (3, 3)), mode="edge"), ((3, 3), (0, 0)), mode="edge")
        p = o.padded(f)
        assert np.array_equal(p[3:-3, 3:-3], out[f])
        ghost = np.ones_like(p, dtype=bool)
        ghost[3:-3, 3:-3] = False
        assert np.array_equal(p[ghost], ref0[ghost])
        assert not np.array_equal(out[f][:, -1], w[f][:, -1]) or f == 4          # the edge itself moved (bx may not)
    o.close()


# ----------------------------------------------------------------------------- rhs() against PAPER.md:35, analytically
class Jet:
    """value and first partial derivatives of a scalar field on the grid: sums and products by the rules of calculus."""

    def __init__(self, v, dx, dy):
        self.v, self.dx, self.dy = v, dx, dy

    def __add__(self, o):
        o = _jet(o)
        return Jet(self.v + o.v, self.dx + o.dx, self.dy + o.dy)

    __radd__ = __add__

    def __sub__(self, o):
        o = _jet(o)
        return Jet(self.v - o.v, self.dx - o.dx, self.dy - o.dy)

    def __mul__(self, o):
        o = _jet(o)
        return Jet(self.v * o.v, self.dx * o.v + self.v * o.dx, self.dy * o.v + self.v * o.dy)

    __rmul__ = __mul__


def _jet(o):
    return o if isinstance(o, Jet) else Jet(o, 0.0, 0.0)


def _div(fx, fy):
    return fx.dx + fy.dy


def _manufactured(n):
    """Smooth periodic primitive fields with their analytic gradients; B = curl(A z) is solenoidal."""
    x = si.centres(n)[None, :] * np.ones((n, 1))
    y = si.centres(n)[:, None] * np.ones((1, n))
    k = 2 * np.pi
    s, c = np.sin, np.cos
    rho = Jet(1.0 + 0.2 * s(k * x) * c(k * y), 0.2 * k * c(k * x) * c(k * y), -0.2 * k * s(k * x) * s(k * y))
    vx = Jet(0.5 + 0.3 * c(k * (x + y)), -0.3 * k * s(k * (x + y)), -0.3 * k * s(k * (x + y)))
    vy = Jet(-0.2 + 0.25 * s(k * (x - 2 * y)), 0.25 * k * c(k * (x - 2 * y)), -0.5 * k * c(k * (x - 2 * y)))
    p = Jet(0.7 + 0.1 * c(k * x) * s(2 * k * y), -0.1 * k * s(k * x) * s(2 * k * y), 0.2 * k * c(k * x) * c(2 * k * y))
    # A = 0.3 y - 0.2 x + 0.05 sin(kx) sin(ky) / k  ->  Bx = dA/dy, By = -dA/dx
    bx = Jet(0.3 + 0.05 * s(k * x) * c(k * y), 0.05 * k * c(k * x) * c(k * y), -0.05 * k * s(k * x) * s(k * y))
    by = Jet(0.2 - 0.05 * c(k * x) * s(k * y), 0.05 * k * s(k * x) * s(k * y), -0.05 * k * c(k * x) * c(k * y))
    return rho, vx, vy, p, bx, by


def _paper_rhs(rho, vx, vy, p, bx, by, gamma):
    """PAPER.md:35-43 (mu0 = 1, g = 0; stray grad p_t of the energy line dropped, DESIGN.md c-1), term by term in
    the paper's vector form:  d rho/dt = -div(v rho);  d(rho v)/dt = -div(v rho v - B B) - grad p_t;
    de/dt = -div(v e - B (B.v) + v p_t);  dB/dt = -div(v B - B v);  p_t = p_k + B^2/2,
    e = p_k/(gamma-1) + rho v^2/2 + B^2/2."""
    v, B = (vx, vy), (bx, by)
    b2h = 0.5 * (bx * bx + by * by)
    pt = p + b2h
    e = (1.0 / (gamma - 1.0)) * p + 0.5 * (rho * (vx * vx + vy * vy)) + b2h
    Bv = bx * vx + by * vy
    out = [None] * 6
    out[0] = -_div(vx * rho, vy * rho)
    for l in range(2):
        t = [v[d] * rho * v[l] - B[d] * B[l] for d in range(2)]
        out[1 + l] = -_div(t[0], t[1]) - (pt.dx, pt.dy)[l]
        ind = [v[d] * B[l] - B[d] * v[l] for d in range(2)]
        out[4 + l] = -_div(ind[0], ind[1])
    en = [v[d] * e - B[d] * Bv + v[d] * pt for d in range(2)]
    out[3] = -_div(en[0], en[1])
    return np.stack(out)


def test_R1_rhs_of_a_nonlinear_state_matches_the_papers_equations_to_fourth_order(oracle_mod):
    """Fails on any dropped / mis-signed / mis-indexed term of `flux` (seeded: m_l v_d dropped), on a wrong
    pressure closure, and on a wrong stencil coefficient (the order would drop)."""
    gamma, errs = 5.0 / 3.0, []
    for n in (32, 96):
        J = _manufactured(n)
        exact = _paper_rhs(*J, gamma)
        prim = dict(zip(("rho", "vx", "vy", "p", "bx", "by"), (j.v for j in J)))
        r = _rhs(oracle_mod, prim, gamma, hd_on=0)
        errs.append([np.abs(r[f] - exact[f]).max() / np.abs(exact[f]).max() for f in range(6)])
    errs = np.array(errs)
    assert (errs[0] < 5e-3).all() and (errs[1] < 6e-5).all(), errs
    assert (errs[0] / errs[1] > 60).all(), errs[0] / errs[1]            # 3^4 = 81 asymptotically
