"""Pins of the 3-D oracle (oracle/smaug3d_oracle.cpp, reading c-11 of DESIGN.md section 3).

None of these re-types a formula of the oracle.  The two load-bearing ones:
  D1  on z-invariant data the 3-D oracle must reproduce the 2-D oracle (a different program, itself pinned by ~55
      closed-form / invariant pins) cell for cell -- this fixes every x/y term of the 3-D code;
  D2  exchanging two axes (and the matching vector components, lengths, boundary kinds, gravity) of a fully 3-D state
      must exchange the result -- so every z term is the image of an x or y term that D1 fixes.
A mistake that survives both would have to sit in a term that is symmetric under every axis exchange AND vanishes
for z-invariant data; the MHD fluxes have no such term (none is a product of three different components).  The
seeded mistakes listed in DESIGN.md section 3 (each run once against these tests with a mutated copy of the oracle)
all fail at least one pin.
"""
import numpy as np
import pytest

import oracle
import smaug_inputs as si

P, O, F = si.BC_PERIODIC, si.BC_OPEN, si.BC_FIXED
MAP23 = ((0, 0), (1, 1), (2, 2), (4, 3), (5, 4), (6, 5))      # (3-D field, 2-D field)


def run3(w, bc, gamma, steps=0, cfl=0.3, lengths=(1.0, 1.0, 1.0), g=(0.0, 0.0, 0.0), want="state", **params):
    _, nz, ny, nx = w.shape
    o = oracle.Oracle3D(nx, ny, nz, gamma, bc, lx=lengths[0], ly=lengths[1], lz=lengths[2], gx=g[0], gy=g[1], gz=g[2], **params)
    o.set_state(w)
    if want == "rhs":
        out = o.rhs()
    else:
        o.step(steps, cfl)
        out = o.get_state()
    t = o.time()
    ws = o.wavespeeds()
    o.close()
    return out, t, ws


# ------------------------------------------------------------------------------------------------ D1
@pytest.mark.parametrize("nz", [1, 5])
@pytest.mark.parametrize("case", ["periodic", "brio_wu_open_x", "fixed_y", "hd_off", "rk2", "gravity"])
def test_D1_z_invariant_data_reproduce_the_2d_oracle(case, nz):
    params, g = {}, (0.0, 0.0, 0.0)
    if case == "brio_wu_open_x":
        w2, bc2, gamma = si.brio_wu(48, 3)
    elif case == "fixed_y":
        w2, _, gamma = si.smooth_random(20, 14, seed=5, amp=5e-2)
        bc2 = (O, O, F, F)
    else:
        w2, bc2, gamma = si.smooth_random(18, 13, seed=11, amp=5e-2)
        if case == "hd_off":
            params["hd_on"] = 0
        if case == "rk2":
            params["rk_order"] = 2
        if case == "gravity":
            g = (0.3, -0.7, 0.0)
    ny, nx = w2.shape[1:]
    w3 = si.extrude_2d(w2, nz)
    bc3 = tuple(bc2) + (P, P)
    o2 = oracle.Oracle(nx, ny, gamma, bc2, gx=g[0], gy=g[1], **params)
    o2.set_state(w2)
    R2 = o2.rhs()
    R3, _, ws3 = run3(w3, bc3, gamma, want="rhs", g=g, **params)
    ws2 = o2.wavespeeds()
    assert (ws3[[0, 1, 3, 4]] == ws2).all() and ws3[2] >= 0.0
    for f3, f2 in MAP23:
        assert np.array_equal(R3[f3], np.broadcast_to(R2[f2], R3[f3].shape)), (case, f3)
    assert not R3[3].any() and not R3[7].any()
    o2.step(6, 0.3)
    S3, t3, _ = run3(w3, bc3, gamma, steps=6, g=g, **params)
    assert t3 == o2.time()
    S2 = o2.get_state()
    for f3, f2 in MAP23:
        assert np.array_equal(S3[f3], np.broadcast_to(S2[f2], S3[f3].shape)), (case, f3)
    assert not S3[3].any() and not S3[7].any()
    o2.close()


# ------------------------------------------------------------------------------------------------ D2
def full3d_case(bc=(P, P, P, P, P, P)):
    lengths = (1.0, 0.8, 0.6)
    w, _, gamma = si.smooth_random_3d(12, 10, 8, seed=23, amp=4e-2, lengths=lengths)
    return w, bc, gamma, lengths, (0.11, -0.23, 0.31)


@pytest.mark.parametrize("which", ["xy", "xz", "yz"])
@pytest.mark.parametrize("bc", [(P, P, P, P, P, P), (P, P, O, O, F, F), (O, F, P, P, O, O)])
def test_D2_axis_exchange_of_a_3d_state_exchanges_the_result(which, bc):
    w, bc, gamma, L, g = full3d_case(bc)
    R, _, ws = run3(w, bc, gamma, want="rhs", lengths=L, g=g)
    wp, bcp, Lp, gp = si.swap_axes_3d(w, which), si.swap_triple(bc, which), si.swap_triple(L, which), si.swap_triple(g, which)
    Rp, _, wsp = run3(wp, bcp, gamma, want="rhs", lengths=Lp, g=gp)
    back = si.swap_axes_3d(Rp, which)
    scale = np.abs(R).reshape(8, -1).max(1)[:, None, None, None]
    assert (scale > 0).all()                      # every field's R is exercised
    assert np.abs(back - R).max() / 1.0 <= 1e-12 * scale.max()
    assert (np.abs(back - R) <= 2e-12 * scale).all()
    assert np.allclose(si.swap_triple(tuple(wsp[:3]), which), ws[:3], rtol=1e-14) and np.allclose(wsp[3:], ws[3:], rtol=1e-14)
    # two full steps (CFL dt: the time step must agree as well)
    S, t, _ = run3(w, bc, gamma, steps=2, lengths=L, g=g)
    Sp, tp, _ = run3(wp, bcp, gamma, steps=2, lengths=Lp, g=gp)
    assert np.allclose(tp, t, rtol=1e-13)
    assert si.rel_l2(si.swap_axes_3d(Sp, which), S).max() <= 1e-11


def test_D2b_one_dimensional_brio_wu_along_each_axis():
    """The Brio-Wu tube along x (2-D oracle, pinned by P13), along y and along z: the same profile."""
    w2, bc2, gamma = si.brio_wu(64, 1)
    o2 = oracle.Oracle(64, 1, gamma, bc2)
    o2.set_state(w2)
    o2.step(25, 0.3)
    ref = o2.get_state()[:, 0, :]
    o2.close()
    w3 = si.extrude_2d(w2, 1)                                   # tube along x: [8, 1, 1, 64]
    bcx = (O, O, P, P, P, P)
    Sx, _, _ = run3(w3, bcx, gamma, steps=25)
    for f3, f2 in MAP23:
        assert np.array_equal(Sx[f3, 0, 0], ref[f2])
    for which in ("xz", "xy"):
        Sw, _, _ = run3(si.swap_axes_3d(w3, which), si.swap_triple(bcx, which), gamma, steps=25)
        assert si.rel_l2(si.swap_axes_3d(Sw, which), Sx).max() <= 1e-10


# ------------------------------------------------------------------------------------------------ D3
@pytest.mark.parametrize("bc", [(P,) * 6, (O, O, F, F, P, P), (F, O, O, F, O, O), (F,) * 6])
def test_D3_uniform_state_is_a_fixed_point_bitwise(bc):
    w = si.prim_to_cons3(1.3 * np.ones((5, 6, 7)), (0.3, -0.2, 0.5), 0.7, (0.4, 0.1, -0.6), 1.4)
    S, _, _ = run3(w, bc, 1.4, steps=4, g=(0.0, 0.0, 0.0))
    assert np.array_equal(S, w)
    R, _, _ = run3(w, bc, 1.4, want="rhs")
    assert not R.any()


# ------------------------------------------------------------------------------------------------ D4
def test_D4_conservation_on_a_periodic_box_with_hyperdiffusion():
    w, bc, gamma = si.smooth_random_3d(10, 9, 8, seed=3, amp=5e-2)
    S, _, _ = run3(w, bc, gamma, steps=12)
    assert np.abs(S - w).max() > 1e-5
    s0, s1 = w.reshape(8, -1).sum(1), S.reshape(8, -1).sum(1)
    scale = np.abs(w).reshape(8, -1).sum(1).max()
    assert np.abs(s1 - s0).max() <= 1e-13 * scale


# ------------------------------------------------------------------------------------------------ D5
def pad_like_c8(a, bc):
    """numpy.pad axis by axis in the order x, y, z (c-8): periodic -> wrap, open / fixed-at-set_state -> edge."""
    for axis, (lo, hi) in ((2, bc[0:2]), (1, bc[2:4]), (0, bc[4:6])):
        pw = [(0, 0)] * 3
        pw[axis] = (3, 3)
        a = np.pad(a, pw, mode="wrap" if lo == P else "edge")
    return a


@pytest.mark.parametrize("bc", [(P,) * 6, (O, O, P, P, F, F), (F, F, O, O, P, P), (P, P, F, O, O, F)])
@pytest.mark.parametrize("shape", [(4, 5, 6), (1, 2, 7), (2, 1, 1)])
def test_D5_ghost_fill_equals_numpy_pad_and_fixed_ghosts_stay_frozen(bc, shape):
    nz, ny, nx = shape
    rng = np.random.default_rng(9)
    w = si.prim_to_cons3(1.0 + 0.1 * rng.random(shape), 0.05 * rng.standard_normal((3,) + shape), 1.0 + 0.1 * rng.random(shape),
                         0.1 * rng.standard_normal((3,) + shape), 1.5)
    o = oracle.Oracle3D(nx, ny, nz, 1.5, bc)
    o.set_state(w)
    for f in range(8):
        assert np.array_equal(o.padded(f), pad_like_c8(w[f], bc)), f
    first = [o.padded(f) for f in range(8)]
    o.step(3, 0.2)
    S = o.get_state()
    assert np.abs(S - w).max() > 0
    for f in range(8):
        now = o.padded(f)
        # a fixed side keeps its whole ghost slab, as far as no later (periodic / open) fill owns the cell
        if bc[4] == F:
            assert np.array_equal(now[:3], first[f][:3])
        if bc[5] == F:
            assert np.array_equal(now[-3:], first[f][-3:])
        if bc[2] == F:
            assert np.array_equal(now[3:-3, :3], first[f][3:-3, :3])
        if bc[3] == F:
            assert np.array_equal(now[3:-3, -3:], first[f][3:-3, -3:])
        if bc[0] == F:
            assert np.array_equal(now[3:-3, 3:-3, :3], first[f][3:-3, 3:-3, :3])
        if bc[1] == F:
            assert np.array_equal(now[3:-3, 3:-3, -3:], first[f][3:-3, 3:-3, -3:])
        # periodic / open sides are refilled from the new interior
        if F not in bc:
            assert np.array_equal(now, pad_like_c8(S[f], bc))
    o.close()


# ------------------------------------------------------------------------------------------------ D6
def test_D6_closed_form_maxima_and_dt_of_a_uniform_flow():
    rho, v, p, B, gamma = 1.3, (0.3, -0.2, 0.5), 0.7, (0.4, 0.1, -0.6), 1.4
    # the one-cell axes are SHORT, so that they would decide dt if the n = 1 rule of c-7 did not leave them out
    for shape, L in (((6, 5, 4), (1.0, 2.0, 0.5)), ((1, 5, 4), (1.0, 2.0, 1e-3)), ((6, 1, 1), (1e-3, 1e-3, 3.0))):
        nz, ny, nx = shape
        w = si.prim_to_cons3(rho * np.ones(shape), v, p, B, gamma)
        o = oracle.Oracle3D(nx, ny, nz, gamma, (P,) * 6, lx=L[0], ly=L[1], lz=L[2])
        o.set_state(w)
        ws = o.wavespeeds()
        a2, b2 = gamma * p / rho, sum(b * b for b in B) / rho          # textbook sound / Alfven speeds squared
        want = [abs(v[d]) + np.sqrt(0.5 * (a2 + b2 + np.sqrt((a2 + b2) ** 2 - 4 * a2 * B[d] ** 2 / rho))) for d in range(3)]
        assert np.allclose(ws, want + [a2, b2], rtol=1e-13)
        o.step(1, 0.4)
        n = (nx, ny, nz)
        dt = 0.4 * min(L[d] / n[d] / want[d] for d in range(3) if n[d] > 1)
        assert np.isclose(o.time()[1], dt, rtol=1e-13)
        o.close()


# ------------------------------------------------------------------------------------------------ D7
def central_div(b, L):
    """fourth-order central divergence on a periodic box, numpy (np.roll), b = (bx, by, bz) as [nz, ny, nx]"""
    out = 0.0
    for comp, axis, length in ((b[0], 2, L[0]), (b[1], 1, L[1]), (b[2], 0, L[2])):
        h = length / comp.shape[axis]
        out = out + (8 * (np.roll(comp, -1, axis) - np.roll(comp, 1, axis)) - (np.roll(comp, -2, axis) - np.roll(comp, 2, axis))) / (12 * h)
    return out


def test_D7_central_div_b_is_preserved_without_hyperdiffusion():
    L = (1.0, 0.8, 0.6)
    w, bc, gamma = si.smooth_random_3d(12, 10, 8, seed=8, amp=5e-2, lengths=L)
    S, _, _ = run3(w, bc, gamma, steps=10, lengths=L, hd_on=0)
    d0, d1 = central_div(w[5:8], L), central_div(S[5:8], L)
    assert np.abs(S[5:8] - w[5:8]).max() > 1e-4
    assert np.abs(d1 - d0).max() <= 1e-11 * np.abs(w[5:8]).max() * 12 / min(L)


# ------------------------------------------------------------------------------------------------ D8
def test_D8_temporal_and_spatial_order_four_on_an_oblique_smooth_problem():
    gamma = 5.0 / 3.0

    def state(n):
        x, y, z = si.grid3(n, n, n)
        ph = 2 * np.pi * (x + y + z)
        one = np.ones((n, n, n))
        rho = 1.0 + 0.05 * np.sin(ph)
        v = (0.05 * np.sin(ph) * one, -0.03 * np.cos(ph) * one, 0.02 * np.sin(ph + 0.4) * one)
        b = (0.3 + 0.02 * np.cos(ph), 0.2 - 0.02 * np.cos(ph) * one, 0.1 * one)
        return si.prim_to_cons3(rho, v, 0.6 + 0.03 * np.sin(ph), b, gamma)

    # temporal: fixed 12^3 grid, T = 0.08 with dt, dt/2, dt/4 against dt/16
    def run_dt(nsteps):
        S, _, _ = run3(state(12), (P,) * 6, gamma, steps=nsteps, hd_on=0, fixed_dt=0.08 / nsteps)
        return S
    ref = run_dt(32)
    e = [np.abs(run_dt(k) - ref).max() for k in (2, 4, 8)]
    assert 12.0 < e[0] / e[1] < 20.0 and 11.0 < e[1] / e[2] < 20.0, e
    # spatial: R(w) at n = 8, 16 against n = 32 sampled at common cell centres is awkward on a cell-centred grid;
    # use the modified-wavenumber identity instead: for a single oblique Fourier mode every central derivative is the
    # exact one times k*/k, k* h = (8 sin kh - sin 2kh)/6, so R_rho of a state with uniform v is -(v.k*) d(rho)
    for n in (8, 16):
        x, y, z = si.grid3(n, n, n)
        ph = 2 * np.pi * (x + y + z) * np.ones((n, n, n))
        vel = (0.3, -0.2, 0.5)
        w = si.prim_to_cons3(1.0 + 0.1 * np.sin(ph), vel, 0.6, (0.0, 0.0, 0.0), gamma)
        R, _, _ = run3(w, (P,) * 6, gamma, want="rhs", hd_on=0)
        kh = 2 * np.pi / n
        kstar = (8 * np.sin(kh) - np.sin(2 * kh)) / 6 * n
        want = -sum(vel) * kstar * 0.1 * np.cos(ph)
        assert np.abs(R[0] - want).max() <= 1e-12
