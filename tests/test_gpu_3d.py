"""GPU parity of the 3-D path (include/smaug3d.h, through the thin binding) against the 3-D oracle, element by element
on the same seeded / analytic inputs.  Bar: relative L2 <= 1e-10 per field (north_star);
both sides implement one IEEE operation sequence, so equality is asserted too."""
import numpy as np
import pytest

import smaug_inputs as si

pytestmark = pytest.mark.gpu
TOL = 1e-10
P, O, F = si.BC_PERIODIC, si.BC_OPEN, si.BC_FIXED


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need a B200")
    import paper_1710_06423_b200 as pkg
    pkg.lib()
    return pkg


def gpu_run(pkg, w, bc, gamma, steps, cfl=0.3, host=True, chunks=1, **params):
    import torch
    _, nz, ny, nx = w.shape
    s = pkg.Smaug3D(nx, ny, nz, gamma, bc, **params)
    s.set_state(torch.from_numpy(w) if host else torch.from_numpy(w).cuda())
    for _ in range(chunks):
        s.step(steps // chunks, cfl)
    out = s.get_state(torch.empty(w.shape, dtype=torch.float64) if host else None)
    t, ws = s.time(), s.wavespeeds()
    s.close()
    return out.cpu().numpy(), t, ws


def cpu_run(oracle_mod, w, bc, gamma, steps, cfl=0.3, threads=8, **params):
    _, nz, ny, nx = w.shape
    o = oracle_mod.Oracle3D(nx, ny, nz, gamma, bc, threads=threads, **params)
    o.set_state(w)
    o.step(steps, cfl)
    out, t, ws = o.get_state(), o.time(), o.wavespeeds()
    o.close()
    return out, t, ws


def check(a, ta, wsa, b, tb, wsb):
    err = si.rel_l2(a, b)
    assert np.isfinite(a).all()
    assert (err <= TOL).all(), err
    assert np.array_equal(a, b), (err, np.abs(a - b).max())
    assert ta == tb, (ta, tb)
    assert list(wsa) == list(wsb), (wsa, wsb)


@pytest.mark.parametrize("shape,steps", [((24, 20, 150), 6), ((9, 130, 33), 5), ((40, 7, 5), 5), ((64, 64, 64), 10)])
def test_orszag_tang_3d_parity(gpu, oracle_mod, shape, steps):
    """several thread blocks / tiles along every axis plus ragged tails; thin and thick axes; both kernel forms"""
    nz, ny, nx = shape
    w, bc, gamma = si.orszag_tang_3d(nx, ny, nz)
    ref = cpu_run(oracle_mod, w, bc, gamma, steps)
    check(*gpu_run(gpu, w, bc, gamma, steps), *ref)
    check(*gpu_run(gpu, w, bc, gamma, steps, kernel=0), *ref)


@pytest.mark.parametrize("kernel", [1, 0])
@pytest.mark.parametrize("bc", [(P, P, O, O, F, F), (O, F, P, P, O, O), (F, F, F, F, F, F), (O, O, O, O, P, P)])
def test_boundary_kinds_3d(gpu, oracle_mod, bc, kernel):
    """open / fixed / periodic mixes on six sides, edges and corners included (a smooth state is not periodic-compatible
    with them, so the boundaries are active from the first step)"""
    L = (1.0, 0.8, 0.6)
    w, _, gamma = si.smooth_random_3d(37, 22, 14, seed=5, amp=4e-2, lengths=L)
    kw = dict(lx=L[0], ly=L[1], lz=L[2])
    check(*gpu_run(gpu, w, bc, gamma, 8, kernel=kernel, **kw), *cpu_run(oracle_mod, w, bc, gamma, 8, **kw))


@pytest.mark.parametrize("params", [dict(hd_on=0), dict(rk_order=2), dict(rk_order=1), dict(gx=0.3, gy=-0.2, gz=0.5),
                                    dict(c_rho=0.05, c_mom=0.2, c_e=0.01, c_b=0.08), dict(fixed_dt=2e-4),
                                    dict(hd_on=0, rk_order=2, gz=-1.0)])
def test_parameters_3d(gpu, oracle_mod, params):
    """every parameter in both kernel forms (SMAUG3_PARAM_KERNEL: 1 = fused tile kernel, 0 = C_d volumes in HBM)"""
    w, bc, gamma = si.smooth_random_3d(30, 18, 12, seed=17, amp=5e-2)
    bc = (P, P, O, O, P, P) if "gz" in params else bc
    ref = cpu_run(oracle_mod, w, bc, gamma, 7, **params)
    for kernel in (1, 0):
        check(*gpu_run(gpu, w, bc, gamma, 7, kernel=kernel, **params), *ref)


@pytest.mark.parametrize("shape", [(1, 40, 60), (1, 1, 200), (3, 1, 50), (50, 1, 1), (2, 2, 2)])
def test_degenerate_axes_3d(gpu, oracle_mod, shape):
    """axes with one or two cells (fewer than the ghost width): the wrap map and the n = 1 rule of the CFL step"""
    nz, ny, nx = shape
    w, bc, gamma = si.smooth_random_3d(nx, ny, nz, seed=3, amp=5e-2)
    check(*gpu_run(gpu, w, bc, gamma, 6), *cpu_run(oracle_mod, w, bc, gamma, 6))


@pytest.mark.parametrize("shape,lens", [((1, 40, 60), dict(lz=1e-3)), ((50, 1, 1), dict(lx=1e-3, ly=1e-3)), ((20, 1, 30), dict(ly=1e-3))])
def test_one_cell_axes_are_left_out_of_dt_3d(gpu, oracle_mod, shape, lens):
    """the n = 1 rule of c-7 where it decides dt: the one-cell axes are SHORT, so counting them would shrink dt 10x or more
    (dt3_kernel against the oracle rule that tests/test_oracle_dt_pins.py pins)"""
    nz, ny, nx = shape
    w, bc, gamma = si.smooth_random_3d(nx, ny, nz, seed=5, amp=5e-2)
    a = gpu_run(gpu, w, bc, gamma, 6, **lens)
    check(*a, *cpu_run(oracle_mod, w, bc, gamma, 6, **lens))
    assert a[1][1] > 0.3 * 2e-3                  # far above any cfl * 1e-3 / cmax a counted short axis would give


def test_z_invariant_3d_equals_the_2d_cuda_path(gpu, oracle_mod):
    """the 3-D kernels on a z-invariant state against the 2-D CUDA path (and both against their oracles)"""
    import torch
    w2, bc2, gamma = si.orszag_tang(96, 80)
    w3 = si.extrude_2d(w2, 3)
    a3, t3, ws3 = gpu_run(gpu, w3, tuple(bc2) + (P, P), gamma, 12)
    s = gpu.Smaug(96, 80, gamma, bc2)
    s.set_state(torch.from_numpy(w2))
    s.step(12, 0.3)
    a2 = s.get_state().cpu().numpy()
    assert s.time() == t3
    s.close()
    for f3, f2 in ((0, 0), (1, 1), (2, 2), (4, 3), (5, 4), (6, 5)):
        assert np.array_equal(a3[f3], np.broadcast_to(a2[f2], a3[f3].shape))
    assert not a3[3].any() and not a3[7].any()


def test_device_buffers_chunked_calls_and_restart_3d(gpu, oracle_mod):
    """device-resident state pointers; 8 steps as 4 + 4; get / set / continue equals the uninterrupted run (periodic)"""
    import torch
    w, bc, gamma = si.orszag_tang_3d(48, 20, 16)
    ref = cpu_run(oracle_mod, w, bc, gamma, 8)
    check(*gpu_run(gpu, w, bc, gamma, 8, host=False, chunks=2), *ref)
    s = gpu.Smaug3D(48, 20, 16, gamma, bc)
    s.set_state(torch.from_numpy(w))
    s.step(4, 0.3)
    mid = s.get_state()
    t_mid = s.time()[0]
    s2 = gpu.Smaug3D(48, 20, 16, gamma, bc)
    s2.set_state(mid)
    s2.step(4, 0.3)
    assert np.array_equal(s2.get_state().cpu().numpy(), ref[0])
    assert abs(t_mid + s2.time()[0] - ref[1][0]) < 1e-15
    assert s.launch_count() > 0
    s.close(); s2.close()


def test_bench_configuration_3d(gpu, oracle_mod):
    """the bench workload (Orszag-Tang 3-D, 256^3) in the launch configuration bench.py times: one full step against the
    oracle on EVERY cell (the 16-thread oracle needs about a minute and 16 GB at that size), then a second step checked
    for finiteness, conservation and positive maxima"""
    import torch
    w, bc, gamma = si.orszag_tang_3d(256)
    s = gpu.Smaug3D(256, 256, 256, gamma, bc)
    wt = torch.from_numpy(w).cuda()
    s.set_state(wt)
    s.step(1, 0.3)
    a, ta, wsa = s.get_state().cpu().numpy(), s.time(), s.wavespeeds()
    check(a, ta, wsa, *cpu_run(oracle_mod, w, bc, gamma, 1, threads=16))
    s.step(1, 0.3)
    out = s.get_state()
    assert torch.isfinite(out).all()
    s0, s1 = wt.reshape(8, -1).sum(1), out.reshape(8, -1).sum(1)
    assert (s1 - s0).abs().max().item() <= 1e-12 * wt.abs().reshape(8, -1).sum(1).max().item()
    assert all(v > 0 for v in s.wavespeeds())
    s.close()
