"""Domain decomposition on the GPU: a px x py group of contexts -- halos pulled
through peer pointers, one shared wave-speed reduction, lockstep stages -- must be BIT-IDENTICAL to the unsplit GPU run
and to the oracle (which has no such feature: it always computes the global problem).  All members live on one device
here (peer pointers are then ordinary device pointers; each member has its own stream, ordered by events)."""
import numpy as np
import pytest

import smaug_inputs as si

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need a B200")
    import paper_1710_06423_b200 as pkg
    pkg.lib()
    return pkg


def unsplit(pkg, w, bc, gamma, steps, bg=None, **params):
    import torch
    ny, nx = w.shape[1:]
    s = pkg.Smaug(nx, ny, gamma, bc, bg=None if bg is None else torch.from_numpy(bg), **params)
    s.set_state(torch.from_numpy(w))
    s.step(steps, 0.3)
    out = s.get_state().cpu().numpy(), s.time(), s.wavespeeds()
    s.close()
    return out


def split(pkg, px, py, w, bc, gamma, steps, bg=None, chunks=1, **params):
    import torch
    ny, nx = w.shape[1:]
    g = pkg.SmaugGroup(px, py, nx, ny, gamma, bc, bg=None if bg is None else torch.from_numpy(bg), **params)
    g.set_state(torch.from_numpy(w))
    for _ in range(chunks):
        g.step(steps // chunks, 0.3)
    out = g.get_state(torch.empty((6, ny, nx), dtype=torch.float64)).numpy(), g.time(), g.wavespeeds()
    launches = g.launch_count()
    g.close()
    return out, launches


def oracle_run(oracle_mod, w, bc, gamma, steps, bg=None, **params):
    ny, nx = w.shape[1:]
    o = oracle_mod.Oracle(nx, ny, gamma, bc, bg=bg, threads=8, **params)
    o.set_state(w)
    o.step(steps, 0.3)
    out = o.get_state(), o.time(), o.wavespeeds()
    o.close()
    return out


def same(a, b):
    assert np.array_equal(a[0], b[0]), np.abs(a[0] - b[0]).max()
    assert tuple(a[1]) == tuple(b[1]) and list(a[2]) == list(b[2])


@pytest.mark.parametrize("px,py", [(2, 1), (1, 2), (2, 2), (3, 2)])
def test_orszag_tang_1000_split_equals_unsplit_and_oracle(gpu, oracle_mod, px, py):
    """BASELINE config 2's grid, 20 steps (the shapes of the paper's Table 1: 2 x 2 sub-domains of a 1000^2 grid)."""
    w, bc, gamma = si.orszag_tang(1000)
    ref = oracle_run(oracle_mod, w, bc, gamma, 20)
    one = unsplit(gpu, w, bc, gamma, 20)
    grp, (n_stage, n_exch) = split(gpu, px, py, w, bc, gamma, 20)
    same(one, ref)
    same(grp, ref)
    assert n_exch == px * py * (1 + 20 * 4)            # one pull per member at set_state and per RK stage
    assert n_stage >= px * py * 20 * 4


@pytest.mark.parametrize("px,py", [(2, 1), (1, 2), (2, 2)])
def test_stratified_background_gravity_split(gpu, oracle_mod, px, py):
    """Non-uniform background + gravity, periodic in x, open in y: the background blocks get their ghosts through the
    same exchange (once), the split kernel's BG form runs per member."""
    w, bc, gamma, bg, (gx, gy) = si.stratified_atmosphere(420, 380)
    ref = oracle_run(oracle_mod, w, bc, gamma, 20, bg=bg, gx=gx, gy=gy)
    grp, _ = split(gpu, px, py, w, bc, gamma, 20, bg=bg, gx=gx, gy=gy)
    same(grp, ref)


@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (2, 2, 0, 0), (0, 0, 2, 1), (2, 1, 1, 2)])
def test_boundary_kinds_through_the_group(gpu, oracle_mod, bc):
    """Open and fixed global sides with the blocks' internal sides exchanged; ragged blocks (101 = 33 + 34 + 34)."""
    nx, ny = 101, 67
    w, _, gamma = si.smooth_random(nx, ny, seed=11, amp=5e-2)
    w[1] += 0.3 * w[0]
    ref = oracle_run(oracle_mod, w, bc, gamma, 25)
    grp, _ = split(gpu, 3, 2, w, bc, gamma, 25, chunks=5)
    same(grp, ref)


@pytest.mark.parametrize("params", [dict(hd_on=0), dict(rk_order=2), dict(rk_order=1), dict(fixed_dt=2e-4, c_mom=0.2)])
def test_parameters_through_the_group(gpu, oracle_mod, params):
    w, bc, gamma = si.orszag_tang(150, 90)
    ref = oracle_run(oracle_mod, w, bc, gamma, 12, **params)
    grp, _ = split(gpu, 2, 2, w, bc, gamma, 12, **params)
    same(grp, ref)


def test_brio_wu_1d_over_four_members(gpu, oracle_mod):
    """The paper's other multi-GPU workload (Brio-Wu on up to 10 GPUs): 800 x 1 over 4 x 1 blocks,
    200 steps; blocks narrower than the ghost width along y (ny = 1, periodic wrap inside one member)."""
    w, bc, gamma = si.brio_wu(800, 1)
    ref = oracle_run(oracle_mod, w, bc, gamma, 200)
    grp, _ = split(gpu, 4, 1, w, bc, gamma, 200)
    same(grp, ref)


def test_group_leaves_a_short_one_cell_axis_out_of_dt(gpu, oracle_mod):
    """the n = 1 rule of c-7 through the group: the leader's dt_kernel gets the GLOBAL cell counts, and the collapsed y axis
    is short (L_y = 1e-3), so it would decide dt if it were counted"""
    w, bc, gamma = si.brio_wu(400, 1)
    ref = oracle_run(oracle_mod, w, bc, gamma, 30, ly=1e-3)
    grp, _ = split(gpu, 3, 1, w, bc, gamma, 30, ly=1e-3)
    same(grp, ref)


def test_tiny_blocks_narrower_than_the_halo(gpu, oracle_mod):
    """Blocks of 2 cells: a ghost cell's source lies two members away."""
    w, bc, gamma = si.orszag_tang(8, 6)
    ref = oracle_run(oracle_mod, w, bc, gamma, 6)
    grp, _ = split(gpu, 4, 3, w, bc, gamma, 6)
    same(grp, ref)


def test_member_cannot_be_stepped_alone_and_devices_are_validated(gpu):
    import ctypes as C
    L = gpu.lib()
    h = C.c_void_p()
    bc = (C.c_int * 4)(0, 0, 0, 0)
    assert L.smaug_group_create(2, 1, 64, 64, 1.4, bc, None, (C.c_int * 2)(0, 99), C.byref(h)) == gpu.EINVAL


def test_tau_terms_add_up_to_the_step_time(gpu):
    """smaug_group_get_tau: with timing on, the three terms of every member cover its stream's time
    gap-free, so their sum is the device time of the steps (checked against CUDA events around the call, loosely: the
    marks sit inside the call), each term is positive, tau is their log ratio, and the state is unchanged by timing."""
    import math
    import torch
    w, bc, gamma = si.orszag_tang(600, 400)
    g = gpu.SmaugGroup(2, 2, 600, 400, gamma, bc)
    g.set_state(torch.from_numpy(w))
    g.step(4, 0.3)
    g.set_timing(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    g.step(10, 0.3)
    e1.record()
    torch.cuda.synchronize()
    tau = g.tau()
    timed = g.get_state(torch.empty((6, 400, 600), dtype=torch.float64)).numpy(), g.time()
    g.close()
    total = tau["t_comp"] + tau["t_comm"] + tau["t_idle"]
    assert tau["t_comp"] > 0 and tau["t_comm"] > 0 and tau["t_idle"] >= 0
    assert 0.5 * e0.elapsed_time(e1) < total < 1.05 * e0.elapsed_time(e1), (tau, e0.elapsed_time(e1))
    assert math.isclose(tau["tau"], math.log(tau["t_comp"] / (tau["t_comm"] + tau["t_idle"])), rel_tol=1e-12)
    plain, _ = split(gpu, 2, 2, w, bc, gamma, 14)
    assert np.array_equal(timed[0], plain[0]) and tuple(timed[1]) == tuple(plain[1])


def _visible_gpus():
    try:
        import torch
        return torch.cuda.device_count()
    except Exception:  # noqa: BLE001
        return 0


# Defined -- hence collected -- only where two GPUs are visible: a skip on the one-GPU boxes would read as coverage.
if _visible_gpus() >= 2:
    def test_group_across_two_devices_equals_unsplit(gpu, oracle_mod):
        """The several-GPU form (peer pointers over NVLink, system-scope atomic maxima into the leader's slots, events
        across devices): members on devices 0 and 1 against the unsplit run and the oracle, bit for bit."""
        w, bc, gamma = si.orszag_tang(200, 120)
        ref = oracle_run(oracle_mod, w, bc, gamma, 12)
        same(unsplit(gpu, w, bc, gamma, 12), ref)
        import torch
        g = gpu.SmaugGroup(2, 1, 200, 120, gamma, bc, devices=[0, 1])
        g.set_state(torch.from_numpy(w))
        g.step(12, 0.3)
        out = g.get_state(torch.empty((6, 120, 200), dtype=torch.float64)).numpy(), g.time(), g.wavespeeds()
        g.close()
        same(out, ref)
