"""Seeded synthetic input generators (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: it only builds bathymetry H, initial
(h, qx, qy, w, p) arrays and the parameter dictionaries of the five BASELINE.json configs
(restated in SURVEY.md 8(d) / DESIGN.md "Input recipe").  No public dataset is used: the
configs stand in for the paper's workloads (1D solitary channel PAPER.md L552-560,
Synolakis-type beach L623-635, 2D basin L669-677, dam-break grids L700-720); `conical_island` is the
geometry of the paper's section 7.6 (L669-677) as a second synthetic workload.

Arrays are NumPy float64, cell fields (ny, nx), node fields (ny+1, nx+1), C order (x fastest).
Every generator takes the grid size so tests can run the same recipe on smaller grids.
"""
from __future__ import annotations

import numpy as np

BC_PERIODIC, BC_WALL, BC_OUTFLOW = 0, 1, 2

SEEDS = {1: 1001, 2: 1002, 3: 1003, 4: 1004, 5: 1005}


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _pack(name, nx, ny, dx, dy, H, h, qx, qy, params, h0, steps, w=None, p=None):
    H = np.ascontiguousarray(H, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float64)
    z = np.zeros((ny, nx))
    return dict(
        name=name, nx=int(nx), ny=int(ny), dx=float(dx), dy=float(dy), H=H, h=h,
        qx=np.ascontiguousarray(z + qx), qy=np.ascontiguousarray(z + qy),
        w=np.zeros((ny + 1, nx + 1)) if w is None else w,
        p=np.zeros((ny + 1, nx + 1)) if p is None else p,
        params=params, h0=float(h0), steps=int(steps),
    )


def config1_channel(nx=512, ny=8, dx=0.1, steps=200):
    """Solitary wave in a flat channel (configs[0]): x walls, y periodic, h0 = 1."""
    g, A, H0, xc = 9.81, 0.1, 1.0, 15.0 * (nx * dx) / 51.2
    x = (np.arange(nx) + 0.5) * dx
    eta = A / np.cosh(np.sqrt(3.0 * A / (4.0 * H0 ** 3)) * (x - xc)) ** 2
    c = np.sqrt(g * (H0 + A))
    H = np.full((ny, nx), H0)
    h = H + eta[None, :]
    qx = np.broadcast_to(c * eta[None, :], (ny, nx))
    params = dict(g=g, cfl=0.5, nonhydro=1, breaking=0, time_order=2,
                  bc_xlo=BC_WALL, bc_xhi=BC_WALL, bc_ylo=BC_PERIODIC, bc_yhi=BC_PERIODIC)
    return _pack("channel_solitary", nx, ny, dx, dx, H, h, qx, 0.0, params, H0, steps)


def config2_lake(nx=512, ny=512, dx=1.0, steps=1000, nbumps=20, seed=SEEDS[2]):
    """Lake at rest over 20 seeded Gaussian bumps, some emerging as dry islands (configs[1])."""
    rng = _rng(seed)
    Lx, Ly = nx * dx, ny * dx
    scale = Lx / 512.0                       # keep bump widths proportional on smaller test grids
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dx
    X, Y = np.meshgrid(x, y)
    H = np.full((ny, nx), 5.0)
    for _ in range(nbumps):
        cx, cy = rng.uniform(0, Lx), rng.uniform(0, Ly)
        s = rng.uniform(10.0, 60.0) * scale
        a = rng.uniform(1.0, 7.0)
        H -= a * np.exp(-((X - cx) ** 2 + (Y - cy) ** 2) / (2.0 * s * s))
    h = np.maximum(H, 0.0)
    params = dict(g=9.81, cfl=0.5, nonhydro=1, breaking=0, time_order=2,
                  bc_xlo=BC_WALL, bc_xhi=BC_WALL, bc_ylo=BC_WALL, bc_yhi=BC_WALL)
    return _pack("lake_at_rest", nx, ny, dx, dx, H, h, 0.0, 0.0, params, 5.0, steps)


def config3_radial(nx=2048, ny=2048, dx=0.05, steps=500):
    """Radial dispersive spreading of a Gaussian hump on a flat bottom (configs[2])."""
    H0 = 0.5
    x = (np.arange(nx) + 0.5) * dx - 0.5 * nx * dx
    y = (np.arange(ny) + 0.5) * dx - 0.5 * ny * dx
    X, Y = np.meshgrid(x, y)
    eta = 0.05 * np.exp(-(X * X + Y * Y) / 0.5 ** 2)
    H = np.full((ny, nx), H0)
    params = dict(g=9.81, cfl=0.5, nonhydro=1, breaking=0, time_order=2,
                  bc_xlo=BC_OUTFLOW, bc_xhi=BC_OUTFLOW, bc_ylo=BC_OUTFLOW, bc_yhi=BC_OUTFLOW)
    return _pack("radial_hump", nx, ny, dx, dx, H, H + eta, 0.0, 0.0, params, H0, steps)


def config4_beach(nx=4096, ny=256, dx=0.05, steps=2000, seed=SEEDS[4]):
    """Solitary wave breaking and running up a 1:30 plane beach (configs[3]).

    Bed: -0.4 m offshore, 1:30 slope from x_toe = 12 m up to +0.2 m, dry plateau beyond;
    multiplied by (1 + 0.01 n(y)) with n a sum of 4 y-periodic Fourier modes, |n| <= 1.
    Wave: generating relaxation zone at x-lo (A = 0.12, h0 = 0.4, L_rel = 6 m, crest at -4 m).
    CFL 0.9, the value of the paper's run-up experiments (BASELINE.json gives none for
    this config): with the two-direction time step of eq. (23) (R20) the 2000 configured
    steps then span about 19 s -- generation, shoaling, breaking, run-up over the dry slope and
    backwash all fall inside the run (at CFL 0.5 the run ends while the wave is still shoaling).
    """
    rng = _rng(seed)
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dx
    Ly = ny * dx
    x_toe, slope, ztop, zoff = 12.0, 1.0 / 30.0, 0.2, -0.4
    zb = np.minimum(np.maximum(zoff + (x - x_toe) * slope, zoff), ztop)
    amp = rng.uniform(0.5, 1.0, 4)
    amp /= amp.sum()
    ph = rng.uniform(0, 2 * np.pi, 4)
    n = sum(amp[k] * np.sin(2 * np.pi * (k + 1) * y / Ly + ph[k]) for k in range(4))
    ZB = zb[None, :] * (1.0 + 0.01 * n[:, None])
    H = -ZB
    h = np.maximum(H, 0.0)
    params = dict(g=9.81, cfl=0.9, nonhydro=1, breaking=1, B1=0.15, B2=0.5, time_order=2,
                  bc_xlo=BC_OUTFLOW, bc_xhi=BC_WALL, bc_ylo=BC_PERIODIC, bc_yhi=BC_PERIODIC,
                  gen_on=1, gen_A=0.12, gen_h0=0.4, gen_x0=-4.0, gen_Lrel=6.0)
    return _pack("breaking_beach", nx, ny, dx, dx, H, h, 0.0, 0.0, params, 0.4, steps)


def config5_tsunami(nx=8192, ny=8192, dx=100.0, steps=200, seed=SEEDS[5], nmodes=48,
                    window="source"):
    """Tsunami-scale basin (configs[4]): 4000 m abyssal plain + smooth fractal noise (std 300 m,
    wavelengths 40-400 km, scaled by local depth) + shelf ramp to 50 m + emerged coast (+20 m),
    elliptical Gaussian uplift of 2 m (axes 100 x 40 km, rotated 20 degrees).

    The geometry is fixed in ABSOLUTE coordinates on the full 819.2 km x 819.2 km basin; a
    smaller grid is a CROP (window) of it with the same dx, depths and slopes (so the same
    conditioning h/dx = 40 and the same diagonal-dominance margin): window="source" is centred on
    the uplift, window="coast" ends at the emerged coast (x = 819.2 km) and contains the
    shoreline.  nx = ny = 8192 is the whole basin."""
    rng = _rng(seed)
    LX = 8192 * 100.0                                 # full basin, metres
    nfx, nfy = int(round(LX / dx)), int(round(LX / dx))
    xc, yc = 0.305 * LX, 0.5 * LX                     # uplift centre (250 km, 410 km)
    if window == "source":
        i0 = int(np.clip(round(xc / dx) - nx // 2, 0, max(nfx - nx, 0)))
    elif window == "coast":
        i0 = max(nfx - nx, 0)
    else:
        raise ValueError(window)
    j0 = int(np.clip(round(yc / dx) - ny // 2, 0, max(nfy - ny, 0)))
    x = (i0 + np.arange(nx) + 0.5) * dx
    y = (j0 + np.arange(ny) + 0.5) * dx

    def sstep(t):
        t = np.clip(t, 0.0, 1.0)
        return t * t * (3.0 - 2.0 * t)

    s = x / LX
    depth = 4000.0 - 3800.0 * sstep((s - 0.61) / 0.12) - 150.0 * sstep((s - 0.73) / 0.22) \
        - 70.0 * sstep((s - 0.95) / 0.05)             # 4000 -> 200 -> 50 -> -20 (emerged)
    # fractal noise: plane waves, amplitude ~ wavelength^1 (red spectrum), separable evaluation
    lam = np.exp(rng.uniform(np.log(40e3), np.log(400e3), nmodes))
    th = rng.uniform(0, 2 * np.pi, nmodes)
    ph = rng.uniform(0, 2 * np.pi, nmodes)
    a = lam / lam.max() * rng.uniform(0.5, 1.0, nmodes)
    kx, ky = 2 * np.pi / lam * np.cos(th), 2 * np.pi / lam * np.sin(th)
    # cos(kx x + ky y + ph) = cos(kx x + ph) cos(ky y) - sin(kx x + ph) sin(ky y)
    Cx = np.cos(np.outer(x, kx) + ph[None, :]) * a[None, :]
    Sx = np.sin(np.outer(x, kx) + ph[None, :]) * a[None, :]
    Cy, Sy = np.cos(np.outer(y, ky)), np.sin(np.outer(y, ky))
    noise = Cy @ Cx.T - Sy @ Sx.T                     # (ny, nx)
    noise *= 300.0 / np.sqrt(0.5 * np.sum(a * a))     # std 300 m (analytic, size independent)
    H = depth[None, :] + noise * (np.maximum(depth, 0.0) / 4000.0)[None, :]
    del noise
    ax, ay = 50e3, 20e3
    c20, s20 = np.cos(np.deg2rad(20.0)), np.sin(np.deg2rad(20.0))
    X = x[None, :] - xc
    Y = y[:, None] - yc
    xr, yr = c20 * X + s20 * Y, -s20 * X + c20 * Y
    eta = 2.0 * np.exp(-(xr * xr / ax ** 2 + yr * yr / ay ** 2))
    h = np.maximum(H + eta, 0.0)
    h[H <= 0.0] = 0.0
    params = dict(g=9.81, cfl=0.5, nonhydro=1, breaking=0, time_order=2,
                  bc_xlo=BC_OUTFLOW, bc_xhi=BC_OUTFLOW, bc_ylo=BC_OUTFLOW, bc_yhi=BC_OUTFLOW)
    return _pack("tsunami_basin", nx, ny, dx, dx, H, h, 0.0, 0.0, params, 4000.0, steps)


def paper_dam_break(n=250):
    """The paper's own timing workload (section 7.7, Table 2): circular dam break
    on [-5,5]^2, H = 1 - 0.25 exp(-x^2 - y^2), h0 = H inside r <= 0.5 and H + 0.25 outside, q = 0,
    CFL 0.9, open boundaries, run to t = 1; n x n cells (the paper: 250 ... 1500).  The initial
    condition is the paper's formula, not a dataset.  `steps` is a rough count (the run is to t=1)."""
    dx = 10.0 / n
    x = (np.arange(n) + 0.5) * dx - 5.0
    X, Y = np.meshgrid(x, x)
    r2 = X * X + Y * Y
    H = 1.0 - 0.25 * np.exp(-r2)
    h = np.where(np.sqrt(r2) <= 0.5, H, H + 0.25)
    params = dict(g=9.81, cfl=0.9, nonhydro=1, breaking=0, time_order=2,
                  bc_xlo=BC_OUTFLOW, bc_xhi=BC_OUTFLOW, bc_ylo=BC_OUTFLOW, bc_yhi=BC_OUTFLOW)
    return _pack("paper_dam_break", n, n, dx, dx, H, h, 0.0, 0.0, params, 1.25, int(0.8 * n))


def conical_island(n=1400, w_advect=0):
    """The geometry of the paper's second 2D workload (section 7.6): basin
    [-5, 23] x [0, 28] m at still-water depth 0.32 m with a conical island (base diameter 7.2 m, top
    diameter 2.2 m, 0.625 m high, side slope 1:4) whose top emerges; solitary wave (33) of amplitude
    0.06 m centred at x = 0 for eta and u; Manning n = 0.015, breaking with B1 = 0.15, B2 = 0.5,
    CFL 0.9, free outflow on all sides.  n x n cells (the paper: dx = 2 cm, n = 1400); the island
    sits at the centre of the numerical domain (the text says "near the center"; the gauge positions
    and the laboratory records are not used).  Geometry and formulas only -- a synthetic stand-in,
    compared between the oracle and the CUDA path, never against the measurements.  `steps` is the
    step count to t = 30 s at the paper's resolution, scaled with n."""
    g, H0, A = 9.81, 0.32, 0.06
    dx = 28.0 / n
    x = (np.arange(n) + 0.5) * dx - 5.0
    y = (np.arange(n) + 0.5) * dx
    X, Y = np.meshgrid(x, y)
    r = np.sqrt((X - 9.0) ** 2 + (Y - 14.0) ** 2)
    zb = np.clip(0.25 * (3.6 - r), 0.0, 0.625)          # bed above the basin floor: cone frustum
    H = H0 - zb
    eta = A / np.cosh(np.sqrt(3.0 * A / (4.0 * H0 ** 3)) * X) ** 2
    h = np.maximum(H + eta, 0.0)
    c = np.sqrt(g * (H0 + A))
    qx = np.where(h > 0.0, c * eta, 0.0)
    params = dict(g=g, cfl=0.9, nonhydro=1, breaking=1, B1=0.15, B2=0.5, manning_n=0.015, time_order=2,
                  w_advect=int(w_advect),
                  bc_xlo=BC_OUTFLOW, bc_xhi=BC_OUTFLOW, bc_ylo=BC_OUTFLOW, bc_yhi=BC_OUTFLOW)
    return _pack("conical_island", n, n, dx, dx, H, h, qx, 0.0, params, H0, int(7.0 * n))


CONFIGS = {1: config1_channel, 2: config2_lake, 3: config3_radial, 4: config4_beach,
           5: config5_tsunami}


def make_config(idx: int, **kw):
    """idx = 1..5 (BASELINE.json configs[idx-1]); kw overrides grid size / steps."""
    return CONFIGS[idx](**kw)


def random_smooth_state(nx, ny, dx, dy, seed=7, depth=1.0, rough=0.3, dry_fraction=0.0):
    """Seeded smooth random (H, h, qx, qy, w, p) for operator / kernel level parity tests.

    Low-order trigonometric fields, periodic over the domain; `rough` scales their amplitude
    relative to `depth`; dry_fraction > 0 lowers the water level so that part of the bed
    emerges (wet/dry cells)."""
    rng = _rng(seed)
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    xn = np.arange(nx + 1) / nx
    yn = np.arange(ny + 1) / ny

    def field(xs, ys, nm=3):
        f = np.zeros((len(ys), len(xs)))
        for _ in range(nm):
            kx, ky = rng.integers(0, 3), rng.integers(0, 3)
            a = rng.uniform(-1, 1)
            px, py = rng.uniform(0, 2 * np.pi, 2)
            f += a * np.outer(np.cos(2 * np.pi * ky * ys + py), np.cos(2 * np.pi * kx * xs + px))
        return f / nm

    H = depth * (1.0 + rough * field(x, y))
    eta = 0.2 * rough * depth * field(x, y)
    if dry_fraction > 0.0:
        level = np.quantile(H, dry_fraction)
        H = H - level - 0.05 * depth          # part of the bed above still water
    h = np.maximum(H + eta, 0.0)
    vel = np.sqrt(9.81 * depth)
    qx = 0.3 * vel * h * field(x, y)
    qy = 0.3 * vel * h * field(x, y)
    w = 0.1 * vel * field(xn, yn)
    p = 0.1 * 9.81 * depth * field(xn, yn)
    return dict(nx=nx, ny=ny, dx=dx, dy=dy, H=H, h=h, qx=qx, qy=qy, w=w, p=p)
