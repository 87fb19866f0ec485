"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types a formula of oracle/smaug_oracle.cpp and compares it with itself: the expected
values are closed forms, hand-worked examples (tests/golden/), invariants of the scheme, textbook linear
MHD (primitive-variable wave matrix + the RK4 stability polynomial), numpy library routines (np.pad),
or brute force.  All CPU, `-m "not gpu"`.
"""
import math
import os

import numpy as np
import pytest

import smaug_inputs as si

GOLD = os.path.join(os.path.dirname(__file__), "golden")
PER = (0, 0, 0, 0)


def run(oracle_mod, w, bc, gamma, steps, cfl=0.3, bg=None, **params):
    ny, nx = w.shape[1:]
    o = oracle_mod.Oracle(nx, ny, gamma, bc, bg=bg, **params)
    o.set_state(w)
    o.step(steps, cfl)
    out = o.get_state()
    t = o.time()
    o.close()
    return out, t


# ----------------------------------------------------------------------------- ghost fill (c-8)
@pytest.mark.parametrize("nx,ny", [(7, 5), (2, 1), (1, 4)])
def test_ghost_fill_matches_numpy_pad(oracle_mod, nx, ny):
    rng = np.random.default_rng(3)
    w = rng.normal(size=(6, ny, nx))
    for bc, modes in [((0, 0, 0, 0), ("wrap", "wrap")), ((1, 1, 1, 1), ("edge", "edge")),
                      ((1, 1, 0, 0), ("edge", "wrap")), ((0, 0, 2, 2), ("wrap", "edge"))]:
        o = oracle_mod.Oracle(nx, ny, 1.4, bc)
        o.set_state(w)       # fixed sides are frozen at the nearest interior value at set_state
        for f in range(6):
            ref = np.pad(w[f], ((0, 0), (3, 3)), mode=modes[0])     # x first ...
            ref = np.pad(ref, ((3, 3), (0, 0)), mode=modes[1])      # ... then y over the padded width
            assert np.array_equal(o.padded(f), ref)
        o.close()


# ----------------------------------------------------------------------------- central difference (c-3)
def test_central_difference_exact_on_quartics_and_kstar(oracle_mod):
    h = 0.37
    x = (np.arange(-2, 22)) * h
    f = 0.3 - 1.1 * x + 0.7 * x**2 - 0.2 * x**3 + 0.05 * x**4
    d = oracle_mod.central_diff_1d(f, h)
    exact = (-1.1 + 1.4 * x - 0.6 * x**2 + 0.2 * x**3)[2:-2]
    assert np.allclose(d, exact, rtol=1e-12, atol=1e-12)
    # modified wavenumber k* = [8 sin(k h) - sin(2 k h)] / (6 h)   (0.988215 at 8 ppw ...)
    for ppw, ratio in [(8, 0.988215), (16, 0.999222), (32, 0.999951)]:
        k = 2 * math.pi / (ppw * h)
        xs = np.arange(-2, ppw + 2) * h
        d = oracle_mod.central_diff_1d(np.sin(k * xs), h)
        kstar = d[0] / math.cos(k * xs[2])
        assert abs(kstar / k - ratio) < 1e-6
        assert np.allclose(d, kstar * np.cos(k * xs[2:-2]), atol=1e-12)


# ----------------------------------------------------------------------------- hyperviscosity (c-5)
def test_P8_nu_unit_step_worked_example(oracle_mod):
    gold = np.loadtxt(os.path.join(GOLD, "nu_unit_step.txt"))
    n = 20
    u = np.zeros(n + 6)
    u[3 + 10:] = 1.0                       # step between cells 9 | 10
    nu = oracle_mod.hyper_nu_1d(u, coef=1.0, delta=1.0, vt=1.0)   # interfaces -1/2 .. n-1/2
    assert np.array_equal(nu[1:], gold)    # gold[k] = interface k+1/2, k = 0..n-1
    c, d, vt = 0.02, 0.125, 3.5
    assert np.allclose(oracle_mod.hyper_nu_1d(u, c, d, vt)[1:], c * d * vt * gold, rtol=1e-15)
    # reflection symmetry of the windows
    assert np.array_equal(oracle_mod.hyper_nu_1d((1 - u)[::-1].copy(), 1, 1, 1), nu[::-1])


def test_P9_nu_on_a_sine_closed_form(oracle_mod):
    for n in (16, 32, 64):
        i = np.arange(-3, n + 3)
        u = np.sin(2 * np.pi * (i + 0.5) / n)
        nu = oracle_mod.hyper_nu_1d(u, 1.0, 1.0, 1.0)
        assert abs(nu.max() - (2 * math.sin(math.pi / n)) ** 2) < 1e-12
    assert abs((2 * math.sin(math.pi / 32)) ** 2 - 3.842944e-2) < 1e-8


def test_P10_nu_bounds(oracle_mod):
    rng = np.random.default_rng(11)
    for _ in range(20):
        u = rng.normal(size=70) * 10.0 ** rng.integers(-8, 8)
        nu = oracle_mod.hyper_nu_1d(u, 1.0, 1.0, 1.0)
        assert (nu >= 0).all() and (nu <= 4.0 + 1e-12).all()
    saw = (-1.0) ** np.arange(40)
    assert np.allclose(oracle_mod.hyper_nu_1d(saw, 1.0, 1.0, 1.0), 4.0, rtol=1e-15)
    assert np.array_equal(oracle_mod.hyper_nu_1d(np.full(30, 2.5), 1.0, 1.0, 1.0), np.zeros(25))


# ----------------------------------------------------------------------------- P1 uniform state
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 1, 1, 1), (2, 2, 0, 0), (1, 1, 2, 2)])
def test_P1_uniform_state_is_preserved_bitwise(oracle_mod, bc):
    nx, ny, gamma = 12, 9, 5.0 / 3.0
    w = si.prim_to_cons(0.3, 0.7, -0.4, 0.2, 0.5, -0.25, gamma)[:, None, None] * np.ones((1, ny, nx))
    for bg in (None, si.uniform_background(nx, ny, 1.3, 2.1, 0.4, 0.3)):
        o = oracle_mod.Oracle(nx, ny, gamma, bc, bg=bg)
        o.set_state(w)
        assert np.array_equal(o.rhs(), np.zeros_like(w))       # every RHS term exactly 0
        o.step(5, 0.3)
        assert np.array_equal(o.get_state(), w)
        o.close()


# ----------------------------------------------------------------------------- P2 conservation
@pytest.mark.parametrize("with_bg", [False, True])
def test_P2_conservation_periodic(oracle_mod, with_bg):
    nx, ny = 40, 32
    w, bc, gamma = si.smooth_random(nx, ny, seed=1710, amp=1e-3)
    bg = si.uniform_background(nx, ny, 0.9, 1.7, 0.3, -0.2) if with_bg else None
    out, _ = run(oracle_mod, w, bc, gamma, 50, bg=bg)
    assert np.abs(out - w).max() > 1e-6                        # it did evolve
    scale = np.abs(w).reshape(6, -1).sum(1) + (np.abs(bg).sum() if with_bg else 0.0)
    drift = np.abs(out.reshape(6, -1).sum(1) - w.reshape(6, -1).sum(1))
    assert (drift / scale < 2e-13).all(), drift / scale
    # the RHS itself sums to zero (all terms are flux differences; uniform-background sources telescope)
    o = oracle_mod.Oracle(nx, ny, gamma, bc, bg=bg)
    o.set_state(w)
    r = o.rhs()
    assert (np.abs(r.reshape(6, -1).sum(1)) / np.abs(r).reshape(6, -1).sum(1).clip(1e-300) < 1e-12).all()
    o.close()


# ----------------------------------------------------------------------------- P3 Orszag-Tang symmetry
def test_P3_orszag_tang_point_symmetry(oracle_mod):
    n = 48
    w, bc, gamma = si.orszag_tang(n, symmetrise=True)
    out, _ = run(oracle_mod, w, bc, gamma, 30)
    sign = np.array([1, -1, -1, 1, -1, -1.0])[:, None, None]
    mirrored = sign * out[:, ::-1, ::-1]
    assert np.abs(out - mirrored).max() <= 1e-12 * np.abs(out).max()
    assert np.abs(out - w).max() > 1e-3


# ----------------------------------------------------------------------------- P5 Brio-Wu 1-D == 2-D, x <-> y
def test_P5_brio_wu_y_invariant_and_transposed(oracle_mod):
    nx, steps = 128, 60
    w1, bc, gamma = si.brio_wu(nx, 1)
    w8, _, _ = si.brio_wu(nx, 8)
    o1, t1 = run(oracle_mod, w1, bc, gamma, steps)
    o8, t8 = run(oracle_mod, w8, bc, gamma, steps)
    assert t1 == t8
    for j in range(8):
        assert np.array_equal(o8[:, j, :], o1[:, 0, :])        # cell for cell
    wt, bct, _ = si.brio_wu(nx, 8, transpose=True)
    ot, tt = run(oracle_mod, wt, bct, gamma, steps)
    assert abs(tt[0] - t8[0]) <= 1e-15
    assert np.abs(si.transpose_state(ot) - o8).max() <= 1e-13
    assert np.abs(o1 - w1).max() > 0.1


def test_P13_brio_wu_structure(oracle_mod):
    """800 points; Bx stays 0.75 exactly; left to right: fast rarefaction, slow compound
    wave, contact discontinuity, slow shock, fast rarefaction.  1000 steps at CFL 0.3 reach t ~ 0.1."""
    w, bc, gamma = si.brio_wu(800, 1)
    out, (t, _) = run(oracle_mod, w, bc, gamma, 1000)
    assert 0.095 < t < 0.105
    assert np.array_equal(out[4], np.full_like(out[4], 0.75))
    rho, x = out[0, 0], si.centres(800)
    assert rho[0] == 1.0 and rho[-1] == 0.125                   # waves have not reached the open ends
    assert np.isfinite(out).all() and rho.min() > 0.1
    by = out[5, 0]
    assert by[0] == 1.0 and by[-1] == -1.0
    # plateaus between the waves (density): post-rarefaction ~0.67, behind the contact ~0.23-0.27, ahead of the slow shock ~0.12
    assert 0.64 < rho[(x > 0.40) & (x < 0.45)].mean() < 0.70
    assert 0.20 < rho[(x > 0.57) & (x < 0.60)].mean() < 0.30
    assert 0.11 < rho[(x > 0.70) & (x < 0.80)].mean() < 0.125
    # the compound wave is a local density peak between the rarefaction plateau and the contact
    seg = rho[(x > 0.45) & (x < 0.55)]
    assert seg.max() > 0.72
    # normal velocity is positive in the fan and transverse velocity negative behind the compound wave
    vx, vy = out[1, 0] / rho, out[2, 0] / rho
    assert vx[(x > 0.4) & (x < 0.6)].min() > 0.3 and vy[(x > 0.5) & (x < 0.6)].max() < -1.0


# ----------------------------------------------------------------------------- P7 div B
def test_P7_divB_preserved_without_hd(oracle_mod):
    n = 32
    w, bc, gamma = si.orszag_tang(n)

    def divb(s):
        def c(f, ax):
            return (8 * (np.roll(f, -1, ax) - np.roll(f, 1, ax)) - (np.roll(f, -2, ax) - np.roll(f, 2, ax))) * n / 12
        return c(s[4], 1) + c(s[5], 0)

    d0 = divb(w)
    out, _ = run(oracle_mod, w, bc, gamma, 40, hd_on=0)
    assert np.abs(divb(out) - d0).max() < 1e-11 * n
    out_hd, _ = run(oracle_mod, w, bc, gamma, 40, hd_on=1)
    # with HD on the mixed resistive terms do not commute discretely: drift at truncation level (documented)
    assert np.abs(divb(out_hd) - d0).max() < 0.05 * n * np.abs(w[4:6]).max()


# ----------------------------------------------------------------------------- P11 closed-form maxima / dt0
def test_P11_closed_form_reductions(oracle_mod):
    # Brio-Wu right state: a^2 = gamma p/rho = 1.6, b^2 = (0.75^2+1)/0.125 = 12.5 (SURVEY c-7 values)
    w, bc, gamma = si.brio_wu(800, 1)
    o = oracle_mod.Oracle(800, 1, gamma, bc)
    o.set_state(w)
    ws = o.wavespeeds()
    s = 1.6 + 12.5
    cf = math.sqrt(0.5 * (s + math.sqrt(s * s - 4 * 1.6 * 0.5625 / 0.125)))
    assert abs(cf - 3.6836658566746) < 1e-12 and abs(ws[0] - 3.6836658566746) < 1e-12
    assert abs(ws[2] - 2.0) < 1e-14 and abs(ws[3] - 12.5) < 1e-14       # left a^2 = 2; right b^2
    o.step(1, 0.3)
    assert abs(o.time()[1] - 1.01800764399e-4) < 1e-15
    o.close()
    # Orszag-Tang: gamma p / rho = 1 exactly by construction; dt0 values of SURVEY c-7
    for n, dt0, thr in [(1000, 1.35443666296e-4, 8)]:
        w, bc, gamma = si.orszag_tang(n)
        o = oracle_mod.Oracle(n, n, gamma, bc, threads=thr)
        o.set_state(w)
        ws = o.wavespeeds()
        assert abs(ws[0] - 2.21494299589) < 1e-10 and abs(ws[1] - 2.16618553376) < 1e-10
        assert abs(ws[2] - 1.0) < 1e-13 and abs(math.sqrt(ws[3]) - 0.848517) < 2e-6 and ws[3] < 0.72
        assert abs(0.3 / n / max(ws[0], ws[1]) - dt0) < 1e-14
        o.close()
    assert abs(w[3].mean() - 0.349256680674) < 1e-11                     # p/(g-1) + rho/2 + 1/(8 pi)


# ----------------------------------------------------------------------------- P12 restart
def test_P12_restart_is_bitwise(oracle_mod):
    w, bc, gamma = si.orszag_tang(24)
    a, _ = run(oracle_mod, w, bc, gamma, 10)
    half, _ = run(oracle_mod, w, bc, gamma, 5)
    b, _ = run(oracle_mod, half, bc, gamma, 5)
    assert np.array_equal(a, b)


# ----------------------------------------------------------------------------- closed-form HD operators
def _uniform(nx, ny, rho0=0.8, p0=0.5, gamma=1.4):
    one = np.ones((ny, nx))
    return dict(rho=rho0 * one, vx=0 * one, vy=0 * one, p=p0 * one, bx=0 * one, by=0 * one), gamma


def _rhs(oracle_mod, prim, gamma, **params):
    w = si.prim_to_cons(prim["rho"], prim["vx"], prim["vy"], prim["p"], prim["bx"], prim["by"], gamma)
    ny, nx = w.shape[1:]
    o = oracle_mod.Oracle(nx, ny, gamma, PER, **params)
    o.set_state(w)
    r = o.rhs()
    o.close()
    return r


def test_hd_sawtooth_closed_forms(oracle_mod):
    """A +-A sawtooth is annihilated by the 4th-order central difference and has M3/M1 = 4 (P10), so the
    RHS is the interface operator alone: R = nu (u_{i+1} - 2 u_i + u_{i-1}) / Delta^2 = -16 c v_t A (-1)^i / Delta."""
    nx, ny, A = 16, 8, 1e-2
    c_rho, c_mom, c_b = 0.03, 0.5, 0.07
    par = dict(c_rho=c_rho, c_mom=c_mom, c_b=c_b, c_e=0.011)
    sx = ((-1.0) ** np.arange(nx))[None, :] * np.ones((ny, 1))
    sy = ((-1.0) ** np.arange(ny))[:, None] * np.ones((1, nx))
    dx, dy = 1.0 / nx, 1.0 / ny
    # (a) density sawtooth along x
    prim, g = _uniform(nx, ny)
    rho0, p0 = 0.8, 0.5
    prim["rho"] = rho0 + A * sx
    r = _rhs(oracle_mod, prim, g, **par)
    vt = math.sqrt(g * p0 / (rho0 - A))
    assert np.allclose(r[0], -16 * c_rho * vt * A * sx / dx, rtol=1e-11)
    assert np.abs(r[1:]).max() < 1e-11
    # (b) vx sawtooth along x: rho-bar weighting, no viscous work because the interface average of v is 0
    prim, g = _uniform(nx, ny)
    prim["vx"] = A * sx
    r = _rhs(oracle_mod, prim, g, **par)
    vt = math.sqrt(g * p0 / rho0)
    assert np.allclose(r[1], -16 * c_mom * rho0 * vt * A * sx / dx, rtol=1e-11)
    assert max(np.abs(r[f]).max() for f in (0, 2, 3, 4, 5)) < 1e-11
    # (c) vx sawtooth along y: the off-diagonal stress carries the factor 1/2
    prim, g = _uniform(nx, ny)
    prim["vx"] = A * sy
    r = _rhs(oracle_mod, prim, g, **par)
    assert np.allclose(r[1], -8 * c_mom * rho0 * vt * A * sy / dy, rtol=1e-11)
    assert max(np.abs(r[f]).max() for f in (0, 2, 3, 4, 5)) < 1e-11
    # (d) bx sawtooth along y about B0: resistive flux, and ohmic coupling B-bar_x * flux in the energy
    prim, g = _uniform(nx, ny)
    B0 = 0.3
    prim["bx"] = B0 + A * sy
    r = _rhs(oracle_mod, prim, g, **par)
    vt = math.sqrt(g * p0 / rho0) + math.sqrt((B0 + A) ** 2 / rho0)
    expect = -16 * c_b * vt * A * sy / dy
    assert np.allclose(r[4], expect, rtol=1e-11)
    assert np.allclose(r[3], B0 * expect, rtol=1e-10)
    assert max(np.abs(r[f]).max() for f in (0, 1, 2, 5)) < 1e-10
    # (e) thermal-energy sawtooth along x (pressure sawtooth, everything else uniform)
    prim, g = _uniform(nx, ny)
    prim["p"] = p0 + A * sx
    r = _rhs(oracle_mod, prim, g, **par)
    vt = math.sqrt(g * (p0 + A) / rho0)
    assert np.allclose(r[3], -16 * 0.011 * vt * (A / (g - 1)) * sx / dx, rtol=1e-10)


def _kstar(n):
    kh = 2 * math.pi / n
    return (8 * math.sin(kh) - math.sin(2 * kh)) / 6 * n      # Lx = 1


def test_hd_mixed_terms_closed_form(oracle_mod):
    """v_y (or b_y) = sin(2 pi x) g(y), everything else uniform and at rest: the only non-zero term of
    R_mx (R_bx) is the mixed term d^c_y{ fac * nubar_x * d^c_x(.) }.  The ratio M3/M1 is scale invariant, so
    nubar_x is the 1-D ratio of sin(2 pi x) (pinned by P8-P10); d^c of a sine is k* cos (pinned above)."""
    nx, ny = 32, 16
    c_mom, c_b = 0.4, 0.02
    x, y = si.centres(nx)[None, :], si.centres(ny)[:, None]
    a, gy = np.sin(2 * np.pi * x), 1 + 0.3 * np.cos(2 * np.pi * y)
    line = np.sin(2 * np.pi * (np.arange(-3, nx + 3) + 0.5) / nx)
    ratio = oracle_mod.hyper_nu_1d(line, 1.0, 1.0, 1.0)             # interfaces -1/2 .. nx-1/2
    rbar = 0.5 * (ratio[:-1] + ratio[1:])[None, :]
    dcx = _kstar(nx) * np.cos(2 * np.pi * x)
    dcy_g = -0.3 * _kstar(ny) * np.sin(2 * np.pi * y)
    rho0, p0 = 0.8, 0.5
    prim, g = _uniform(nx, ny)
    prim["vy"] = a * gy
    r = _rhs(oracle_mod, prim, g)
    vt = math.sqrt(g * p0 / rho0)
    expect = 0.5 * rho0 * c_mom * (1.0 / nx) * vt * rbar * dcx * dcy_g
    assert np.abs(r[1] - expect).max() < 1e-11 * np.abs(expect).max() + 1e-15
    assert np.abs(expect).max() > 1e-6
    # magnetic: R_bx = -d^c_y{ nubar_x(by) d^c_x by };  R_e (v = 0) = ohmic part of the by x-flux only
    prim, g = _uniform(nx, ny)
    prim["by"] = a * gy
    r = _rhs(oracle_mod, prim, g)
    vt = math.sqrt(g * p0 / rho0) + math.sqrt((prim["by"] ** 2).max() / rho0)
    expect = -c_b * (1.0 / nx) * vt * rbar * dcx * dcy_g
    assert np.abs(r[4] - expect).max() < 1e-11 * np.abs(expect).max()
    by = prim["by"]
    nu_r = c_b * (1.0 / nx) * vt * ratio[1:][None, :]               # interface i+1/2, i = 0..nx-1
    phi_r = nu_r * (np.roll(by, -1, 1) - by) * nx
    e_r = 0.5 * (np.roll(by, -1, 1) + by) * phi_r
    expect_e = (e_r - np.roll(e_r, 1, 1)) * nx
    assert np.abs(r[3] - expect_e).max() < 1e-10 * np.abs(expect_e).max()


# ----------------------------------------------------------------------------- background split (c-2)
def test_split_equals_unsplit_for_uniform_background(oracle_mod):
    nx, ny = 24, 20
    W, bc, gamma = si.smooth_random(nx, ny, seed=5, amp=5e-2)
    W[1] += 0.2 * W[0]
    rho_b, e_b, bx_b, by_b = 0.15, 0.2, 0.12, 0.05
    bg = si.uniform_background(nx, ny, rho_b, e_b, bx_b, by_b)
    wt = W.copy()
    wt[0] -= rho_b; wt[3] -= e_b; wt[4] -= bx_b; wt[5] -= by_b
    o_full = oracle_mod.Oracle(nx, ny, gamma, bc)
    o_split = oracle_mod.Oracle(nx, ny, gamma, bc, bg=bg)
    o_full.set_state(W); o_split.set_state(wt)
    rf, rs = o_full.rhs(), o_split.rhs()
    assert np.abs(rf - rs).max() < 1e-12 * np.abs(rf).max()
    o_full.step(10, 0.3); o_split.step(10, 0.3)
    a, b = o_full.get_state(), o_split.get_state()
    b[0] += rho_b; b[3] += e_b; b[4] += bx_b; b[5] += by_b
    assert np.abs(a - b).max() < 1e-12
    assert abs(o_full.time()[0] - o_split.time()[0]) < 1e-15


def test_split_consistent_with_paper_equations_on_pinch_background(oracle_mod):
    """Non-uniform background in equilibrium WITH tension: azimuthal field B_phi = B0 (r/a) exp(-r^2/a^2)
    confined by the pressure p(r) = p_c - B0^2 [exp(-2s)(s/2 - 1/4) + 1/4], s = r^2/a^2 (integrates
    dp/dr = -(B_phi/r) d(r B_phi)/dr).  Then grad p_tb = (B_b.grad)B_b and div B_b = 0, so the split RHS
    equals the RHS of PAPER.md:35 for the total fields up to truncation error, O(h^4)."""
    gamma, errs = 5.0 / 3.0, []
    a, B0, p_c = 0.12, 0.5, 0.6
    for n in (40, 120):
        x = si.centres(n)[None, :] * np.ones((n, 1)) - 0.5
        y = x.T
        s_ = (x * x + y * y) / a ** 2
        bphi_over_r = B0 / a * np.exp(-s_)
        Bx_b, By_b = -y * bphi_over_r, x * bphi_over_r
        p_b = p_c - B0 ** 2 * (np.exp(-2 * s_) * (0.5 * s_ - 0.25) + 0.25)
        rho_b = 1 + 0.2 * np.exp(-s_)
        bg = np.stack([rho_b, p_b / (gamma - 1) + 0.5 * (Bx_b ** 2 + By_b ** 2), Bx_b, By_b])
        xx, yy = x + 0.5, y + 0.5
        wt = np.zeros((6, n, n))
        wt[0] = 1e-2 * np.sin(2 * np.pi * (xx + yy))
        wt[1] = 5e-2 * np.cos(2 * np.pi * (xx - yy))
        wt[2] = 3e-2 * np.sin(2 * np.pi * (2 * xx + yy))
        wt[3] = 2e-2 * np.cos(2 * np.pi * (xx - 2 * yy))
        wt[4] = 1e-2 * np.sin(2 * np.pi * yy)
        wt[5] = 1e-2 * np.sin(2 * np.pi * xx)
        W = wt.copy()
        W[0] += bg[0]; W[3] += bg[1]; W[4] += bg[2]; W[5] += bg[3]
        o_full = oracle_mod.Oracle(n, n, gamma, PER, hd_on=0)
        o_split = oracle_mod.Oracle(n, n, gamma, PER, bg=bg, hd_on=0)
        o_full.set_state(W); o_split.set_state(wt)
        rf, rs = o_full.rhs(), o_split.rhs()
        errs.append(np.abs(rf - rs).max() / np.abs(rf).max())
    assert 1e-7 < errs[0] < 1e-2 and errs[0] / errs[1] > 40, errs     # 3^4 = 81 asymptotically


# ----------------------------------------------------------------------------- P4 linear waves
def _rk4_factor(z):
    return 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24


def _wave_matrix(rho, vx, p, bx, by, gamma):
    """Textbook primitive-variable matrix of 1-D ideal MHD along x for (rho, vx, vy, p, By), mu0 = 1."""
    return np.array([[vx, rho, 0, 0, 0],
                     [0, vx, 0, 1 / rho, by / rho],
                     [0, 0, vx, 0, -bx / rho],
                     [0, gamma * p, 0, vx, 0],
                     [0, by, -bx, 0, vx]], dtype=float)


@pytest.mark.parametrize("ppw", [8, 16])
@pytest.mark.parametrize("kind", ["sound", "alfven", "fast", "slow"])
@pytest.mark.parametrize("transpose", [False, True])
def test_P4_linear_wave_phase_and_amplitude(oracle_mod, ppw, kind, transpose):
    """Amplitude 1e-8 eigenmode of the textbook wave matrix, HD off, periodic, one wavelength of `ppw`
    points: after n RK4 steps the Fourier coefficient is multiplied by G(z)^n, z = -i lambda k* dt, with
    lambda the ANALYTIC wave speed, k* the modified wavenumber of the 4th-order difference and G the RK4
    stability polynomial."""
    gamma, rho0, p0, amp, nsteps = 5.0 / 3.0, 1.2, 0.7, 1e-8, 10
    bx0, by0 = dict(sound=(0.0, 0.0), alfven=(0.6, 0.0), fast=(0.5, 0.4), slow=(0.5, 0.4))[kind]
    a2, b2 = gamma * p0 / rho0, (bx0 ** 2 + by0 ** 2) / rho0
    disc = math.sqrt((a2 + b2) ** 2 - 4 * a2 * bx0 ** 2 / rho0)
    lam = dict(sound=math.sqrt(a2), alfven=bx0 / math.sqrt(rho0),
               fast=math.sqrt(0.5 * (a2 + b2 + disc)), slow=math.sqrt(0.5 * (a2 + b2 - disc)))[kind]
    vals, vecs = np.linalg.eig(_wave_matrix(rho0, 0.0, p0, bx0, by0, gamma))
    if kind == "alfven":      # By = 0: the (vy, By) pair decouples and travels at Bx/sqrt(rho)
        r = np.array([0, 0, -1 / math.sqrt(rho0), 0, 1.0])
    elif kind == "sound":
        r = np.array([rho0, math.sqrt(a2), 0, rho0 * a2, 0])
    else:
        j = int(np.argmin(np.abs(vals - lam)))
        assert abs(vals[j] - lam) < 1e-12          # eigenvalue of the textbook matrix == c-4 formula
        r = np.real(vecs[:, j])
    nx, ny = ppw, 4
    th = 2 * np.pi * si.centres(nx)[None, :] * np.ones((ny, 1))
    c = np.cos(th)
    w = si.prim_to_cons(rho0 + amp * r[0] * c, amp * r[1] * c, amp * r[2] * c, p0 + amp * r[3] * c,
                        bx0 + 0 * c, by0 + amp * r[4] * c, gamma)
    w_eq = si.prim_to_cons(rho0, 0.0, 0.0, p0, bx0, by0, gamma)[:, None, None]
    bc = PER
    if transpose:
        w, (nx, ny) = si.transpose_state(w), (ny, nx)
        w_eq = w_eq[[0, 2, 1, 3, 5, 4]]
    dt = 0.3 / ppw / (lam + 0.3)
    o = oracle_mod.Oracle(nx, ny, gamma, bc, hd_on=0, fixed_dt=dt)
    o.set_state(w)
    o.step(nsteps, 0.3)
    out = o.get_state()
    o.close()
    if transpose:
        out, w, w_eq = si.transpose_state(out), si.transpose_state(w), w_eq[[0, 2, 1, 3, 5, 4]]
    comp = 0 if abs(r[0]) > 0.1 * np.abs(r).max() else 5       # density, else By
    proj = lambda s: ((s[comp] - w_eq[comp]) * np.exp(-1j * th)).mean()
    kstar = _kstar(ppw)
    expect = _rk4_factor(-1j * lam * kstar * dt) ** nsteps
    got = proj(out) / proj(w)
    assert abs(got - expect) < 2e-6, (got, expect)
    # numerical phase speed = analytic * k*/k up to the O(z^5) RK4 phase error
    speed = -np.angle(got) / (2 * np.pi * nsteps * dt)
    assert abs(speed / lam - kstar / (2 * np.pi)) < 2e-4


def test_P4_oblique_sound_wave(oracle_mod):
    n, gamma, rho0, p0, amp, nsteps = 16, 1.4, 1.0, 1.0 / 1.4, 1e-8, 20
    cs = 1.0
    x, y = si.centres(n)[None, :], si.centres(n)[:, None]
    th = 2 * np.pi * (x + y)
    c = np.cos(th)
    w = si.prim_to_cons(rho0 * (1 + amp * c), amp * cs * c / math.sqrt(2), amp * cs * c / math.sqrt(2),
                        p0 * (1 + gamma * amp * c), 0 * c, 0 * c, gamma)
    dt = 0.2 / n
    o = oracle_mod.Oracle(n, n, gamma, PER, hd_on=0, fixed_dt=dt)
    o.set_state(w)
    o.step(nsteps, 0.3)
    out = o.get_state()
    proj = lambda s: ((s[0] - rho0) * np.exp(-1j * th)).mean()
    expect = _rk4_factor(-1j * cs * math.sqrt(2) * _kstar(n) * dt) ** nsteps
    assert abs(proj(out) / proj(w) - expect) < 2e-6


# ----------------------------------------------------------------------------- P6 convergence orders
def test_P6_fourth_order_in_space_and_time(oracle_mod):
    gamma, T = 5.0 / 3.0, 0.04
    sols = []
    for n in (16, 48, 144):          # cell centres of grid n coincide with centres 3i+1 of grid 3n
        w, bc, _ = si.smooth_random(n, n, seed=2, kmax=1, amp=0.2, gamma=gamma)
        steps = n // 4
        out, _ = run(oracle_mod, w, bc, gamma, steps, hd_on=0, fixed_dt=T / steps)
        sols.append(out)
    e1 = np.abs(sols[0] - sols[1][:, 1::3, 1::3]).max()
    e2 = np.abs(sols[1] - sols[2][:, 1::3, 1::3]).max()
    order = math.log(e1 / e2) / math.log(3)
    assert 3.6 < order < 4.6, (e1, e2, order)
    # time: fixed grid, dt halved twice
    n, T = 24, 0.08
    w, bc, _ = si.smooth_random(n, n, seed=2, kmax=2, amp=0.2, gamma=gamma)
    outs = [run(oracle_mod, w, bc, gamma, s, hd_on=0, fixed_dt=T / s)[0] for s in (4, 8, 16)]
    d1, d2 = np.abs(outs[0] - outs[1]).max(), np.abs(outs[1] - outs[2]).max()
    order_t = math.log2(d1 / d2)
    assert 3.6 < order_t < 4.6, (d1, d2, order_t)
    # rk_order 2 (midpoint) is second order, rk_order 1 first order
    for rk, lo, hi in [(2, 1.7, 2.4), (1, 0.8, 1.3)]:
        outs = [run(oracle_mod, w, bc, gamma, s, hd_on=0, fixed_dt=0.25 * T / s, rk_order=rk)[0]
                for s in (8, 16, 32)]
        d1, d2 = np.abs(outs[0] - outs[1]).max(), np.abs(outs[1] - outs[2]).max()
        assert lo < math.log2(d1 / d2) < hi


# ----------------------------------------------------------------------------- API errors (section 8(b))
def test_api_argument_errors(oracle_mod):
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(0, 4, 1.4, PER)
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(4, 4, 1.0, PER)
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(4, 4, 1.4, (0, 1, 0, 0))      # periodic on one side only
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(4, 4, 1.4, (0, 0, 3, 3))
    o = oracle_mod.Oracle(4, 4, 1.4, PER)
    with pytest.raises(oracle_mod.OracleError):
        o.set_param(99, 1.0)
    o.set_state(np.zeros((6, 4, 4)))                    # rho = 0 -> non-finite dt
    with pytest.raises(oracle_mod.OracleError) as ei:
        o.step(1, 0.3)
    assert ei.value.code == oracle_mod.ENONFINITE


def test_hd_viscous_work_differential_pin(oracle_mod):
    """R(c_mom) - R(c_mom = 0) isolates the viscous terms: for a 1-D flow vx(x), rho(x) they are
    d(Phi)/dx in the momentum and d(vbar * Phi)/dx in the energy, Phi = rho-bar nu (vx_{i+1}-vx_i)/dx."""
    nx, ny, gamma, c_mom = 32, 4, 1.4, 0.4
    x = si.centres(nx)[None, :] * np.ones((ny, 1))
    prim = dict(rho=0.8 * (1 + 0.1 * np.cos(2 * np.pi * x)), vx=0.3 + 0.2 * np.sin(2 * np.pi * x),
                vy=0 * x, p=0.5 + 0 * x, bx=0 * x, by=0 * x)
    r1 = _rhs(oracle_mod, prim, gamma, c_mom=c_mom)
    r0 = _rhs(oracle_mod, prim, gamma, c_mom=0.0)
    vline = 0.3 + 0.2 * np.sin(2 * np.pi * (np.arange(-3, nx + 3) + 0.5) / nx)
    vt = math.sqrt((gamma * prim["p"] / prim["rho"]).max())
    nu = oracle_mod.hyper_nu_1d(vline, c_mom, 1.0 / nx, vt)[1:][None, :]        # interface i+1/2
    rho, vx = prim["rho"], prim["vx"]
    phi = 0.5 * (rho + np.roll(rho, -1, 1)) * nu * (np.roll(vx, -1, 1) - vx) * nx
    work = 0.5 * (vx + np.roll(vx, -1, 1)) * phi
    assert np.allclose(r1[1] - r0[1], (phi - np.roll(phi, 1, 1)) * nx, rtol=1e-9, atol=1e-13)
    assert np.allclose(r1[3] - r0[3], (work - np.roll(work, 1, 1)) * nx, rtol=1e-9, atol=1e-13)
    assert np.abs(r1[3] - r0[3]).max() > 1e-5
    for f in (0, 2, 4, 5):
        assert np.array_equal(r1[f], r0[f])
