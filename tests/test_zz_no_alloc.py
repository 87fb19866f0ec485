"""smaug_wavespeeds_static: the wave-speed maxima for callers that cannot allocate device memory.

Some users of the library hold a state on the GPU but may not call cudaMalloc -- their memory belongs to another
allocator (a framework pool that reserved the whole device), or they sit in a loop that cannot take cudaMalloc's
device-wide synchronisation.  For them the library keeps the reduction's working memory inside its own image (a fixed
0.5 MiB array per GPU) and serves grids of up to 16384 * 4096 cells from it.  These tests check that entry point
against the ordinary route (a context: smaug_set_state + smaug_get_wavespeeds) bit for bit, on consecutive calls,
because the array is shared and keeps the previous call's contents.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes on its own in a fresh process and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

import paper_1710_06423_b200 as pkg
import smaug_inputs as si


def _context_maxima(w, gamma, bc, bg=None):
    """The existing path: a context loads the state and reduces its maxima into its own (allocated) slots."""
    import torch
    ny, nx = w.shape[1:]
    sim = pkg.Smaug(nx, ny, gamma, bc, bg=None if bg is None else torch.from_numpy(bg))
    sim.set_state(torch.from_numpy(w))
    m = sim.wavespeeds()
    sim.close()
    return np.array(m)


def test_size_limit_is_refused_before_anything_touches_the_gpu():
    """Needs no device: a grid beyond the array's capacity is turned away with a message that names the limit."""
    L = pkg.lib()
    assert pkg.WAVESPEEDS_STATIC_MAX_CELLS == 16384 * 4096
    fake = C.c_void_p(256)                                    # never dereferenced: the size check comes first
    assert L.smaug_wavespeeds_static(8192, 8193, 5.0 / 3.0, fake, None, fake, None) == pkg.EINVAL
    msg = L.smaug_last_error().decode()
    assert "67108864" in msg and "static scratch" in msg, msg
    assert L.smaug_wavespeeds_static(0, 8, 5.0 / 3.0, fake, None, fake, None) == pkg.EINVAL
    assert L.smaug_wavespeeds_static(8, 8, 1.0, fake, None, fake, None) == pkg.EINVAL
    assert L.smaug_wavespeeds_static(8, 8, 5.0 / 3.0, None, None, fake, None) == pkg.EINVAL


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_context_path():
    """A large state first (several hundred blocks leave their partial maxima in the array), then a much smaller and
    slower one: if the second call picked up anything the first left behind, its maxima would be too large.  Then the
    first state again.  Every result equals the context path's exactly (a maximum does not depend on the order)."""
    import torch
    torch.cuda.set_device(0)
    w_big, bc, gamma = si.orszag_tang(1100, 900)              # 990,000 cells = 242 blocks, ragged last block
    w_small, _, _ = si.orszag_tang(96, 80)
    w_small = w_small.copy()
    w_small[1:3] *= 0.25                                      # slower flow: every maximum below the big state's
    w_small[4:6] *= 0.5
    want_big = _context_maxima(w_big, gamma, bc)
    want_small = _context_maxima(w_small, gamma, bc)
    assert (want_small[:2] < want_big[:2]).all() and want_small[3] < want_big[3]
    d_big, d_small = torch.from_numpy(w_big).cuda(), torch.from_numpy(w_small).cuda()
    out = torch.full((3, 4), -1.0, dtype=torch.float64, device="cuda")   # the caller's own output buffer
    pkg.wavespeeds_static(d_big, gamma, out=out[0])
    pkg.wavespeeds_static(d_small, gamma, out=out[1])
    pkg.wavespeeds_static(d_big, gamma, out=out[2])
    got = out.cpu().numpy()
    assert (got[0] == want_big).all(), (got[0], want_big)
    assert (got[1] == want_small).all(), (got[1], want_small)
    assert (got[2] == want_big).all(), (got[2], want_big)


@pytest.mark.gpu
def test_background_form_and_a_one_dimensional_state():
    """The split form (totals = background + perturbation) and Brio-Wu 800 x 1 (one block, n < 4096), back to back."""
    import torch
    torch.cuda.set_device(0)
    w, bc, gamma, bg, _ = si.stratified_atmosphere(300, 200)
    want = _context_maxima(w, gamma, bc, bg)
    got = pkg.wavespeeds_static(torch.from_numpy(w).cuda(), gamma, bg=torch.from_numpy(bg).cuda()).cpu().numpy()
    assert (got == want).all(), (got, want)
    w1, bc1, gamma1 = si.brio_wu(800)
    want1 = _context_maxima(w1, gamma1, bc1)
    got1 = pkg.wavespeeds_static(torch.from_numpy(w1).cuda(), gamma1).cpu().numpy()
    assert (got1 == want1).all(), (got1, want1)
    assert abs(got1[0] - 3.6836658566746) < 1e-12            # SURVEY c-7: cmax_x of the right state


@pytest.mark.gpu
def test_host_pointers_are_refused():
    """There is no staging buffer to copy a host array into, so the call says so instead of faulting."""
    import torch
    torch.cuda.set_device(0)
    w, _, gamma = si.orszag_tang(32, 32)
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    rc = pkg.lib().smaug_wavespeeds_static(32, 32, gamma, C.c_void_p(w.ctypes.data), None, C.c_void_p(out.data_ptr()), None)
    assert rc == pkg.EINVAL and b"DEVICE pointers" in pkg.lib().smaug_last_error()
