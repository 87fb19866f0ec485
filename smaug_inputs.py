"""Seeded / analytic input generators shared by the tests, bench.py and smoke() for BOTH the oracle and
the CUDA path.  numpy only.  Holds none of the method's arithmetic: it only tabulates initial conditions
(BASELINE.json "configs"; PAPER.md:99-112 Orszag-Tang, PAPER.md:130 Brio-Wu) on the cell-centred grid
x_i = (i + 1/2) Lx / nx and converts primitive (rho, v, p, B) to the stored variables
w = (rho, mx, my, e, bx, by), e = p/(gamma-1) + rho v^2/2 + B^2/2 (PAPER.md:39-43 solved for e).

The workloads are analytic, so they stand in for no external dataset (the paper uses none).
"""
from __future__ import annotations

import numpy as np

BC_PERIODIC, BC_OPEN, BC_FIXED = 0, 1, 2
FIELDS = ("rho", "mx", "my", "e", "bx", "by")


def centres(n: int, length: float = 1.0) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) + 0.5) * (length / n)


def prim_to_cons(rho, vx, vy, p, bx, by, gamma: float) -> np.ndarray:
    rho, vx, vy, p, bx, by = np.broadcast_arrays(rho, vx, vy, p, bx, by)
    e = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy) + 0.5 * (bx * bx + by * by)
    return np.ascontiguousarray(np.stack([rho, rho * vx, rho * vy, e, bx, by]).astype(np.float64))


def orszag_tang(nx: int, ny: int | None = None, gamma: float = 5.0 / 3.0, symmetrise: bool = False):
    """BASELINE.json configs 2-5: rho=25/(36 pi), p=5/(12 pi), vx=-sin 2 pi y, vy=sin 2 pi x,
    Bx=-sin(2 pi y)/sqrt(4 pi), By=sin(4 pi x)/sqrt(4 pi) on [0,1]^2, periodic.
    Returns (w[6,ny,nx], bc, gamma).  symmetrise=True makes the 180-degree point symmetry exact in fp."""
    ny = nx if ny is None else ny
    x = centres(nx)[None, :]
    y = centres(ny)[:, None]
    rho = 25.0 / (36.0 * np.pi)
    p = 5.0 / (12.0 * np.pi)
    b0 = 1.0 / np.sqrt(4.0 * np.pi)
    one = np.ones((ny, nx))
    w = prim_to_cons(rho * one, -np.sin(2 * np.pi * y) * one, np.sin(2 * np.pi * x) * one, p * one,
                     -b0 * np.sin(2 * np.pi * y) * one, b0 * np.sin(4 * np.pi * x) * one, gamma)
    if symmetrise:
        sign = np.array([1, -1, -1, 1, -1, -1], dtype=np.float64)[:, None, None]
        w = 0.5 * (w + sign * w[:, ::-1, ::-1])
    return np.ascontiguousarray(w), (BC_PERIODIC,) * 4, gamma


def brio_wu(nx: int = 800, ny: int = 1, gamma: float = 2.0, transpose: bool = False):
    """BASELINE.json config 1: left (x<0.5) rho=1,p=1,By=1; right rho=0.125,p=0.1,By=-1; Bx=0.75, v=0;
    open in x, periodic in y (y-invariant).  transpose=True swaps the roles of x and y.
    Returns (w, bc, gamma)."""
    x = centres(nx)[None, :] * np.ones((ny, 1))
    left = x < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    by = np.where(left, 1.0, -1.0)
    bx = 0.75 * np.ones_like(x)
    zero = np.zeros_like(x)
    w = prim_to_cons(rho, zero, zero, p, bx, by, gamma)
    bc = (BC_OPEN, BC_OPEN, BC_PERIODIC, BC_PERIODIC)
    if transpose:
        w = transpose_state(w)
        bc = (BC_PERIODIC, BC_PERIODIC, BC_OPEN, BC_OPEN)
    return w, bc, gamma


def transpose_state(w: np.ndarray) -> np.ndarray:
    """The x<->y mirrored problem: swap axes and swap the x/y components."""
    wt = np.transpose(w, (0, 2, 1))
    return np.ascontiguousarray(wt[[0, 2, 1, 3, 5, 4]])


def smooth_random(nx: int, ny: int, seed: int = 1710, kmax: int = 4, amp: float = 1e-3,
                  gamma: float = 5.0 / 3.0, mean=None):
    """Periodic random smooth state: Orszag-Tang mean state (rho, p) with v=0, B=mean B, plus a sum of
    Fourier modes |k| <= kmax of relative amplitude `amp` on each primitive variable (SURVEY P2 recipe).
    Returns (w, bc, gamma)."""
    rng = np.random.default_rng(seed)
    x = centres(nx)[None, :]
    y = centres(ny)[:, None]
    if mean is None:
        mean = dict(rho=25.0 / (36.0 * np.pi), p=5.0 / (12.0 * np.pi), vx=0.0, vy=0.0, bx=0.2, by=0.1)

    def field(scale):
        f = np.zeros((ny, nx))
        norm = 0.0
        for kx in range(-kmax, kmax + 1):
            for ky in range(0, kmax + 1):
                if kx * kx + ky * ky > kmax * kmax or (kx == 0 and ky == 0):
                    continue
                a, ph = rng.normal(), rng.uniform(0, 2 * np.pi)
                f += a * np.cos(2 * np.pi * (kx * x + ky * y) + ph)
                norm += abs(a)
        return scale * amp * f / norm          # grid-independent normalisation: |field| <= scale*amp

    rho = mean["rho"] + field(mean["rho"])
    p = mean["p"] + field(mean["p"])
    vx = mean["vx"] + field(1.0)
    vy = mean["vy"] + field(1.0)
    bx = mean["bx"] + field(1.0)
    by = mean["by"] + field(1.0)
    return prim_to_cons(rho, vx, vy, p, bx, by, gamma), (BC_PERIODIC,) * 4, gamma


def uniform_background(nx: int, ny: int, rho_b: float, e_b: float, bx_b: float, by_b: float) -> np.ndarray:
    bg = np.empty((4, ny, nx))
    bg[0], bg[1], bg[2], bg[3] = rho_b, e_b, bx_b, by_b
    return bg


def stratified_atmosphere(nx: int, ny: int, gamma: float = 5.0 / 3.0, g: float = 1.0, scale_height: float = 0.25,
                          rho0: float = 1.0, by0: float = 0.3, pulse: float = 1e-2, split: bool = True):
    """A gravitationally stratified, magnetised atmosphere with a wave-driving pulse (the use the paper
    states for the code): isothermal hydrostatic column rho_b = rho0 exp(-y/H),
    p_b = rho_b g H under g = (0, -g), uniform vertical field B_b = (0, by0) (force-free, so the balance
    grad p_tb - (B_b.grad)B_b = rho_b g holds analytically), e_b = p_b/(gamma-1) + by0^2/2; on top a
    Gaussian velocity/pressure pulse of relative amplitude `pulse` centred at (0.5, 0.3).  Periodic in x,
    open in y.  split=True: returns the perturbation w on the background bg; split=False: the same total
    state as a perturbation on a zero background (bg = None).
    Returns (w, bc, gamma, bg, (gx, gy))."""
    x = centres(nx)[None, :] * np.ones((ny, 1))
    y = centres(ny)[:, None] * np.ones((1, nx))
    H = scale_height
    rho_b = rho0 * np.exp(-y / H)
    p_b = rho_b * g * H
    e_b = p_b / (gamma - 1.0) + 0.5 * by0 * by0
    bump = np.exp(-((x - 0.5) ** 2 + (y - 0.3) ** 2) / (2 * 0.05 ** 2))
    vy = pulse * bump
    vx = 0.5 * pulse * bump * np.sin(2 * np.pi * x)
    p = p_b * (1.0 + pulse * bump)
    rho = rho_b * (1.0 + 0.5 * pulse * bump)
    tot = prim_to_cons(rho, vx, vy, p, np.zeros_like(x), by0 * np.ones_like(x), gamma)
    bc = (BC_PERIODIC, BC_PERIODIC, BC_OPEN, BC_OPEN)
    if not split:
        return tot, bc, gamma, None, (0.0, -g)
    bg = np.ascontiguousarray(np.stack([rho_b, e_b, np.zeros_like(x), by0 * np.ones_like(x)]))
    w = tot.copy()
    w[0] -= rho_b
    w[3] -= e_b
    w[5] -= by0
    return np.ascontiguousarray(w), bc, gamma, bg, (0.0, -g)


def rel_l2(a: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """c-9 error metric per field: ||a_f - ref_f||_2 / ||ref_f||_2; where the denominator is 0 the
    numerator is divided by max_f ||ref_f||_2 instead."""
    num = np.sqrt(((a - ref) ** 2).reshape(a.shape[0], -1).sum(1))
    den = np.sqrt((ref ** 2).reshape(ref.shape[0], -1).sum(1))
    fallback = den.max() if den.max() > 0 else 1.0
    return num / np.where(den > 0, den, fallback)


# ------------------------------------------------------------------------------------------------ three dimensions
# State [8, nz, ny, nx] = (rho, mx, my, mz, e, bx, by, bz); bc = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi).
FIELDS3 = ("rho", "mx", "my", "mz", "e", "bx", "by", "bz")


def prim_to_cons3(rho, v, p, b, gamma: float) -> np.ndarray:
    rho, vx, vy, vz, p, bx, by, bz = np.broadcast_arrays(rho, v[0], v[1], v[2], p, b[0], b[1], b[2])
    e = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bx * bx + by * by + bz * bz)
    return np.ascontiguousarray(np.stack([rho, rho * vx, rho * vy, rho * vz, e, bx, by, bz]).astype(np.float64))


def grid3(nx: int, ny: int, nz: int, lengths=(1.0, 1.0, 1.0)):
    x = centres(nx, lengths[0])[None, None, :]
    y = centres(ny, lengths[1])[None, :, None]
    z = centres(nz, lengths[2])[:, None, None]
    return x, y, z


def orszag_tang_3d(nx: int, ny: int | None = None, nz: int | None = None, gamma: float = 5.0 / 3.0, eps: float = 0.2):
    """A three-dimensional Orszag-Tang-like vortex (the paper prints no 3-D configuration; this recipe is ours, DESIGN.md
    section 9): the BASELINE.json Orszag-Tang state modulated along z, plus a z-flow and a z-field,
      rho = 25/(36 pi), p = 5/(12 pi), m(z) = 1 + eps sin 2 pi z,
      v = (-m sin 2 pi y, m sin 2 pi x, eps sin 2 pi z),  B = (-m sin 2 pi y, m sin 4 pi x, eps sin 2 pi x) / sqrt(4 pi)
    (every component of B is independent of its own coordinate: div B = 0), periodic.  Returns (w[8,nz,ny,nx], bc, gamma)."""
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    x, y, z = grid3(nx, ny, nz)
    one = np.ones((nz, ny, nx))
    rho = 25.0 / (36.0 * np.pi) * one
    p = 5.0 / (12.0 * np.pi) * one
    b0 = 1.0 / np.sqrt(4.0 * np.pi)
    m = 1.0 + eps * np.sin(2 * np.pi * z)
    v = (-m * np.sin(2 * np.pi * y) * one, m * np.sin(2 * np.pi * x) * one, eps * np.sin(2 * np.pi * z) * one)
    b = (-b0 * m * np.sin(2 * np.pi * y) * one, b0 * m * np.sin(4 * np.pi * x) * one, b0 * eps * np.sin(2 * np.pi * x) * one)
    return prim_to_cons3(rho, v, p, b, gamma), (BC_PERIODIC,) * 6, gamma


def smooth_random_3d(nx: int, ny: int, nz: int, seed: int = 1710, kmax: int = 2, amp: float = 1e-2,
                     gamma: float = 5.0 / 3.0, lengths=(1.0, 1.0, 1.0)):
    """Periodic random smooth 3-D state: the Orszag-Tang mean (rho, p), mean field (0.2, 0.1, -0.15), plus Fourier modes
    |k| <= kmax of relative amplitude `amp` on each of the eight primitive variables.  Returns (w, bc, gamma)."""
    rng = np.random.default_rng(seed)
    x, y, z = grid3(nx, ny, nz, lengths)

    def field(scale):
        f = np.zeros((nz, ny, nx))
        norm = 0.0
        for kx in range(-kmax, kmax + 1):
            for ky in range(-kmax, kmax + 1):
                for kz in range(0, kmax + 1):
                    if kx * kx + ky * ky + kz * kz > kmax * kmax or (kx == 0 and ky == 0 and kz == 0):
                        continue
                    a, ph = rng.normal(), rng.uniform(0, 2 * np.pi)
                    f += a * np.cos(2 * np.pi * (kx * x / lengths[0] + ky * y / lengths[1] + kz * z / lengths[2]) + ph)
                    norm += abs(a)
        return scale * amp * f / norm

    rho0, p0 = 25.0 / (36.0 * np.pi), 5.0 / (12.0 * np.pi)
    rho = rho0 + field(rho0)
    p = p0 + field(p0)
    v = (field(1.0), field(1.0), field(1.0))
    b = (0.2 + field(1.0), 0.1 + field(1.0), -0.15 + field(1.0))
    return prim_to_cons3(rho, v, p, b, gamma), (BC_PERIODIC,) * 6, gamma


def extrude_2d(w2: np.ndarray, nz: int) -> np.ndarray:
    """A 2-D state [6, ny, nx] as the z-invariant 3-D state [8, nz, ny, nx] with mz = bz = 0."""
    _, ny, nx = w2.shape
    w3 = np.zeros((8, nz, ny, nx))
    for f3, f2 in ((0, 0), (1, 1), (2, 2), (4, 3), (5, 4), (6, 5)):
        w3[f3] = w2[f2][None, :, :]
    return w3


_SWAPS = {      # axis swap -> (transpose of [f, z, y, x], field order)
    "xy": ((0, 1, 3, 2), (0, 2, 1, 3, 4, 6, 5, 7)),
    "xz": ((0, 3, 2, 1), (0, 3, 2, 1, 4, 7, 6, 5)),
    "yz": ((0, 2, 1, 3), (0, 1, 3, 2, 4, 5, 7, 6)),
}


def swap_axes_3d(w: np.ndarray, which: str) -> np.ndarray:
    """The mirrored problem with two axes (and the matching vector components) exchanged; which = 'xy', 'xz' or 'yz'."""
    tr, order = _SWAPS[which]
    return np.ascontiguousarray(np.transpose(w, tr)[list(order)])


def swap_triple(t, which: str):
    """Exchange the entries of a per-axis triple (x, y, z) -- or of the six per-side boundary kinds -- the same way."""
    a, b = "xyz".index(which[0]), "xyz".index(which[1])
    t = list(t)
    if len(t) == 3:
        t[a], t[b] = t[b], t[a]
    else:
        t[2 * a:2 * a + 2], t[2 * b:2 * b + 2] = t[2 * b:2 * b + 2], t[2 * a:2 * a + 2]
    return tuple(t)
