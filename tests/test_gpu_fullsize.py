"""Parity of the CUDA path at BASELINE.json's FULL sizes, in the launch configuration bench.py
times (one context per problem, nh_step on a stream, state resident in HBM)  (-m gpu).

The oracle needs ~10 minutes per step at 8192 x 8192, so at full size the comparison is
  (a) on SAMPLED OUTPUTS the oracle can compute one by one: every kernel outside the Krylov solver
      is a local stencil, so its output on a window of the full grid equals the oracle's output
      on the same window cut out of the full-size input (window sides that are not domain
      boundaries get a margin wider than the stencil).  Bit-exact, as in test_gpu_parity.py;
  (b) via properties that hold at any size: the solver's true residual (with the operator apply
      that (a) verifies), commutation of a whole step with x<->y transposition (oracle pin P4),
      lake at rest (P1), mass conservation (P2);
  (c) against the oracle outright, for as many full-size steps as it finishes in about a minute
      (configs 1-4).
"""
import numpy as np
import pytest

from paper_1706_04551_b200 import inputs

from test_gpu_parity import assert_parity, parity  # noqa: F401  (same bars)

pytestmark = pytest.mark.gpu

PER, WALL, OUT = inputs.BC_PERIODIC, inputs.BC_WALL, inputs.BC_OUTFLOW
MARGIN = 4   # > stencil radius of every local kernel (predictor: 2 cells + slopes of neighbours = 3)


@pytest.fixture(scope="module")
def G():
    from paper_1706_04551_b200 import nh
    nh.lib()
    return nh


def _windows(nx, ny, n, seed, extra=()):
    """(i0, j0) of n x n cell windows: the four corners, the middle of each side, `extra`, and
    seeded random positions."""
    rng = np.random.Generator(np.random.PCG64(seed))
    w = [(0, 0), (nx - n, 0), (0, ny - n), (nx - n, ny - n), (nx // 2, 0), (nx // 2, ny - n),
         (0, ny // 2), (nx - n, ny // 2)]
    w += list(extra)
    w += [(int(rng.integers(0, nx - n)), int(rng.integers(0, ny - n))) for _ in range(6)]
    return w


def _crop_state(s, H, i0, j0, n):
    c = {k: np.ascontiguousarray(s[k][j0:j0 + n, i0:i0 + n]) for k in ("h", "qx", "qy")}
    c.update({k: np.ascontiguousarray(s[k][j0:j0 + n + 1, i0:i0 + n + 1]) for k in ("w", "p")})
    c["H"] = np.ascontiguousarray(H[j0:j0 + n, i0:i0 + n])
    return c


def _interior(i0, j0, n, nx, ny, node):
    """Slices of the window (local indices) that are comparable: margin off every window side that
    is not a side of the full domain (there the oracle window applies the domain's own BC)."""
    lo_i = 0 if i0 == 0 else MARGIN
    lo_j = 0 if j0 == 0 else MARGIN
    hi_i = (n if i0 + n == nx else n - MARGIN) + (1 if node else 0)
    hi_j = (n if j0 + n == ny else n - MARGIN) + (1 if node else 0)
    if node:
        if i0 + n != nx:
            hi_i -= 1
        if j0 + n != ny:
            hi_j -= 1
    return slice(lo_j, hi_j), slice(lo_i, hi_i)


def test_config5_full_size_local_kernels_on_windows_and_solver_residual(O, G):
    cfg = inputs.make_config(5)
    nx, ny = cfg["nx"], cfg["ny"]
    assert (nx, ny) == (8192, 8192)
    prm = cfg["params"]
    g = G.NH(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], **prm)
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    g.step(1)                       # a state with non-trivial q, w, p everywhere the wave has reached
    assert g.sync() == 0
    i1 = g.info()
    assert i1.steps == 1 and i1.solves == 2 and i1.clamps == 0
    assert i1.res_last <= 1e-12 and 100 < i1.iters_last < 2000
    s0 = g.get_state()
    dt = g.compute_dt()
    assert 0.1 < dt < 0.2           # CFL 0.5 * 100 m / (2 sqrt(g 4300 m)) ~ 0.12 s

    n = 96
    src = (int(0.305 * nx) - n // 2, ny // 2 - n // 2)                 # the uplift
    shore = []                                                         # shoreline (wet/dry) windows
    for f in (0.2, 0.7):
        j = int(f * ny)
        ish = int(np.argmax(cfg["H"][j] <= 0.0))                       # first emerged cell of row j
        assert 0 < ish < nx
        shore.append((min(ish - n // 2, nx - n), j - n // 2))
    wins = _windows(nx, ny, n, seed=55, extra=[src] + shore)

    # --- local kernels of the pressure step on the state s0: coefficients, rhs, operator apply
    rng = np.random.Generator(np.random.PCG64(56))
    x = rng.standard_normal((ny + 1, nx + 1))
    cg_, bg, yg = g.coeffs(), g.rhs(dt), g.apply_A(x)
    for (i0, j0) in wins:
        c = _crop_state(s0, cfg["H"], i0, j0, n)
        o = O.Oracle(n, n, cfg["dx"], cfg["dy"], c["H"], **prm)
        o.set_state(c["h"], c["qx"], c["qy"], c["w"], c["p"])
        sj, si = _interior(i0, j0, n, nx, ny, node=True)
        gj, gi = slice(j0 + sj.start, j0 + sj.stop), slice(i0 + si.start, i0 + si.stop)
        co = o.coeffs()
        for k in co:
            assert np.array_equal(co[k][sj, si], cg_[k][gj, gi]), (k, i0, j0)
        assert np.array_equal(o.rhs(dt)[sj, si], bg[gj, gi]), ("rhs", i0, j0)
        xo = np.ascontiguousarray(x[j0:j0 + n + 1, i0:i0 + n + 1])
        assert np.array_equal(o.apply_A(xo)[sj, si], yg[gj, gi]), ("apply_A", i0, j0)
    del cg_, yg

    # --- the solve at full size: true residual with the operator verified above
    p, iters, relres = g.solve(bg, x0=s0["p"])
    r = bg - g.apply_A(p)
    true_rel = np.sqrt(np.sum(r * r)) / np.sqrt(np.sum(bg * bg))
    assert true_rel <= 1.05e-12, true_rel       # one polish iteration after ||r|| <= 1e-12 ||b||
    assert relres <= 1e-12
    del r, p, bg, x

    # --- predictor at full size (state s0 -> U*), windows bit-exact
    g.hydrostatic_step(dt)
    assert g.sync() == 0
    s1 = g.get_state()
    wet_dry_windows = 0
    for (i0, j0) in wins:
        c = _crop_state(s0, cfg["H"], i0, j0, n)
        o = O.Oracle(n, n, cfg["dx"], cfg["dy"], c["H"], **prm)
        o.set_state(c["h"], c["qx"], c["qy"], c["w"], c["p"])
        o.hydrostatic_step(dt)
        so = o.get_state()
        sj, si = _interior(i0, j0, n, nx, ny, node=False)
        gj, gi = slice(j0 + sj.start, j0 + sj.stop), slice(i0 + si.start, i0 + si.stop)
        for k in ("h", "qx", "qy"):
            assert np.array_equal(so[k][sj, si], s1[k][gj, gi]), (k, i0, j0)
        hh = c["h"]
        wet_dry_windows += int(hh.min() == 0.0 and hh.max() > 0.0)
    assert wet_dry_windows >= 2     # the sample contains shoreline windows


def test_config5_full_size_step_commutes_with_transposition(G):
    """Oracle pin P4 at full size: step(transpose(U)) == transpose(step(U)) (dx = dy), within the
    north_star tolerances (two solves of the same system at 1e-12)."""
    cfg = inputs.make_config(5)
    nx, ny = cfg["nx"], cfg["ny"]
    prm = dict(cfg["params"])
    g = G.NH(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], **prm)
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    g.step(2)
    assert g.sync() == 0
    a = g.get_state()
    ia = g.info()
    g.close()
    T = lambda f: np.ascontiguousarray(f.T)
    prmT = dict(prm, bc_xlo=prm["bc_ylo"], bc_xhi=prm["bc_yhi"], bc_ylo=prm["bc_xlo"], bc_yhi=prm["bc_xhi"])
    gt = G.NH(ny, nx, cfg["dy"], cfg["dx"], T(cfg["H"]), **prmT)
    gt.set_state(T(cfg["h"]), T(cfg["qy"]), T(cfg["qx"]), T(cfg["w"]), T(cfg["p"]))
    gt.step(2)
    assert gt.sync() == 0
    b = gt.get_state()
    ib = gt.info()
    gt.close()
    # the max-reduction is order independent; the second step's state carries solver-level differences
    assert abs(ia.dt_last - ib.dt_last) <= 1e-12 * ia.dt_last and abs(ia.t - ib.t) <= 1e-12 * ia.t
    bt = dict(h=b["h"].T, qx=b["qy"].T, qy=b["qx"].T, w=b["w"].T, p=b["p"].T)
    assert_parity(a, bt, cfg["H"], cfg["h0"])
    assert abs(ia.iters_total - ib.iters_total) <= 0.1 * ia.iters_total
    # closed-basin-like bookkeeping: nothing has reached the open boundaries after 2 steps
    m0 = float(np.sum(cfg["h"], dtype=np.longdouble))
    m1 = float(np.sum(a["h"], dtype=np.longdouble))
    assert abs(m1 - m0) <= 1e-12 * m0


def test_config3_full_size_two_steps_against_oracle(O, G):
    cfg = inputs.make_config(3)
    assert (cfg["nx"], cfg["ny"]) == (2048, 2048)
    o = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    for k in (o, g):
        k.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    o.step(2)
    g.step(2)
    assert g.sync() == 0
    sg, so = g.get_state(), o.get_state()
    assert_parity(sg, so, cfg["H"], cfg["h0"])
    # the second step's dt comes from a state that already carries the 1e-12-level difference of two
    # valid solves: equal to rounding, not necessarily bitwise
    assert abs(g.info().dt_last - o.info().dt_last) <= 1e-12 * o.info().dt_last and g.info().clamps == 0
    # the hump sits at the domain centre: four-fold mirror symmetry survives the step
    eta = sg["h"] - cfg["H"]
    assert np.max(np.abs(eta - eta[::-1, :])) <= 1e-9 * cfg["h0"]
    assert np.max(np.abs(eta - eta[:, ::-1])) <= 1e-9 * cfg["h0"]
    assert np.max(np.abs(eta - eta.T)) <= 1e-9 * cfg["h0"]


def test_config3_full_size_run_properties(G):
    """Config 3 for 60 of its 500 steps at full size: mass is conserved to round-off while the
    ring is inside the domain, the state keeps its symmetry, every solve converges."""
    cfg = inputs.make_config(3)
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    g.step(60)
    assert g.sync() == 0
    i = g.info()
    assert i.steps == 60 and i.solves == 120 and i.clamps == 0 and i.res_last <= 1e-12
    s = g.get_state()
    m0 = float(np.sum(cfg["h"], dtype=np.longdouble))
    m1 = float(np.sum(s["h"], dtype=np.longdouble))
    assert abs(m1 - m0) <= 1e-12 * m0
    eta = s["h"] - cfg["H"]
    assert np.max(np.abs(eta - eta[::-1, ::-1])) <= 1e-9 * cfg["h0"]
    assert np.max(np.abs(s["qx"] - s["qy"].T)) <= 1e-9 * max(np.max(np.abs(s["qx"])), 1e-3)
    assert 0.0 < eta.max() < 0.05     # the hump has started to collapse and radiate


def test_config4_full_size_steps_against_oracle(O, G):
    cfg = inputs.make_config(4)
    assert (cfg["nx"], cfg["ny"]) == (4096, 256)
    o = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    for k in (o, g):
        k.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    for _ in range(2):
        o.step(3)
        g.step(3)
        assert g.sync() == 0
        assert_parity(g.get_state(), o.get_state(), cfg["H"], cfg["h0"])
    assert abs(g.info().dt_last - o.info().dt_last) <= 1e-12 * o.info().dt_last


def test_config2_full_size_lake_at_rest_1000_steps(O, G):
    cfg = inputs.make_config(2)
    assert (cfg["nx"], cfg["ny"]) == (512, 512) and cfg["steps"] == 1000
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    o = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    o.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    o.step(20)
    g.step(20)
    assert g.sync() == 0
    sg, so = g.get_state(), o.get_state()
    for k in sg:
        assert np.array_equal(sg[k], so[k]), k          # no solver iterations: bit-exact
    g.step(980)
    assert g.sync() == 0
    s = g.get_state()
    assert (cfg["H"] < 0).any() and (cfg["H"] > 0).any()   # islands emerge
    assert np.max(np.abs(s["qx"])) == 0.0 and np.max(np.abs(s["qy"])) == 0.0
    assert np.max(np.abs(s["h"] - cfg["h"])) <= 1e-13 * cfg["h0"]
    assert np.all(s["w"] == 0.0) and np.all(s["p"] == 0.0)
    i = g.info()
    assert i.steps == 1000 and i.iters_total == 0 and i.clamps == 0
