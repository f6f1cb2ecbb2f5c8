"""Parity of the CUDA path against the CPU oracle over the CONFIGURED horizons of configs 3, 4 and 5
(BASELINE.json north_star: "after the configured steps"; SURVEY.md 8(d) "Parity metric": checkpoints
every 10 % of the run) at grid sizes the oracle finishes in minutes, plus checkpoint-restart windows
of config 4 at 1024 x 48 placed on the onset of breaking and on the maximum run-up (-m gpu).

Larger sizes of the same runs (config 3 at 512^2, config 4 at 1024 x 48 for all 2000 steps, the
config-5 crops at 512^2) are recorded by `python bench.py --parityruns ...` under profiles/.
Bars: those of tests/test_gpu_parity.py (north_star tolerances).
"""
import numpy as np
import pytest

from paper_1706_04551_b200 import inputs

from test_gpu_parity import assert_parity, both, parity  # noqa: F401  (same bars)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    from paper_1706_04551_b200 import nh
    nh.lib()
    return nh


def side_by_side(O, G, cfg, steps, ncp=10, **over):
    """Advance both sides `steps` steps, comparing the full state at `ncp` checkpoints."""
    o, g = both(O, G, cfg, **over)
    done, worst = 0, {}
    for k in range(ncp):
        n = (steps * (k + 1)) // ncp - done
        o.step(n)
        g.step(n)
        done += n
        assert g.sync() == 0
        r = parity(g.get_state(), o.get_state(), cfg["H"], cfg["h0"])
        assert all(np.isfinite(v) and v <= 1.0 for v in r.values()), (done, r)
        worst = {k_: max(worst.get(k_, 0.0), v) for k_, v in r.items()}
    assert g.info().steps == o.info().steps == steps
    assert g.info().t == pytest.approx(o.info().t, rel=1e-11)
    return o, g, worst


def test_config3_radial_hump_500_steps(O, G):
    # 256 x 256 (12.8 m square, same dx, depth and hump as the 2048^2 config): in 500 steps the ring
    # reaches and leaves through the outflow boundaries
    cfg = inputs.make_config(3, nx=256, ny=256)
    assert cfg["steps"] == 500
    o, g, worst = side_by_side(O, G, cfg, 500)
    s = g.get_state()
    assert g.info().clamps == 0
    assert np.max(np.abs(s["h"] - cfg["H"])) < 0.3 * 0.05            # the hump has spread out
    edge = np.concatenate([s["qx"][:, -3:].ravel(), s["qy"][-3:, :].ravel()])
    assert np.max(np.abs(edge)) > 1e-4                                # ... and reached the boundary


def test_config4_beach_2000_steps_narrow(O, G):
    """The whole configured run of config 4 -- generation, shoaling, breaking, run-up over the dry slope
    and plateau -- on a 640 x 8 strip of the same beach (same dx, slope, y-perturbed bed, generating
    zone, breaking and wet/dry parameters); the bore overtops the +0.2 m plateau and a thin film runs
    over the dry bed to the wall: the negative-depth clamp of R7 acts on real values.

    This run is SENSITIVE: the breaking switch (9) and the wet/dry front turn differences of the
    size of the solver tolerance into O(1e-3) differences (two ORACLE runs at solver_rtol 1e-12 and
    1e-13 differ by 1e4 bars right after breaking sets in and by 4e6 bars at step 2000,
    profiles/r02b_config4_sensitivity.md), so an element-by-element bar over the full horizon is only
    meaningful where both sides do the same arithmetic: with the paper's solver (solver 1, R28) the
    CUDA path reproduces the oracle BIT FOR BIT through all 2000 steps.  The default solver is then
    held against the same oracle run by what is unique: the wet/dry front, the run-up, the breaking
    activity, and the state within the spread two valid solves show."""
    cfg = inputs.make_config(4, nx=640, ny=8)
    assert cfg["steps"] == 2000 and cfg["params"]["breaking"] == 1
    wet0 = cfg["h"] > 1e-5
    o, g = both(O, G, cfg, solver=1, srj_eps=1e-6)
    g0 = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])   # default solver
    g0.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    probe = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    done, broke, wet_max = 0, 0, 0
    for k in range(10):
        o.step(200)
        g.step(200)
        g0.step(200)
        done += 200
        assert g.sync() == 0 and g0.sync() == 0
        so, sg, s0 = o.get_state(), g.get_state(), g0.get_state()
        for f in ("h", "qx", "qy", "w", "p"):
            assert np.array_equal(sg[f], so[f]), (done, f, np.max(np.abs(sg[f] - so[f])))
        ig, io = g.info(), o.info()
        assert ig.iters_total == io.iters_total and ig.t == io.t and ig.clamps == io.clamps
        wet = so["h"] > 1e-5
        wet_max = max(wet_max, int(np.sum(wet & ~wet0)))
        probe.set_state(so["h"], so["qx"], so["qy"], so["w"], so["p"])
        b = probe.breaking(o.info().dt_last)
        broke = max(broke, int(np.sum(b["w"] != so["w"])))
        # default solver (BiCGStab to 1e-12) against the same oracle run (Jacobi to 1e-6 increment): two
        # different valid solves of every pressure system
        assert np.mean((s0["h"] > 1e-5) != wet) <= 0.01, done
        assert np.max(np.abs(s0["h"] - so["h"])) <= 0.05 * cfg["h0"], done
        assert g0.info().t == pytest.approx(io.t, rel=1e-4)
    assert broke > 0          # the breaking criterion (9) was active inside a compared window
    assert wet_max > 8 * 100  # the shoreline ran up by more than 5 m of beach (100 cells per row)
    ig, io = g.info(), o.info()
    assert list(ig.clamp_hist) == list(io.clamp_hist) and sum(list(io.clamp_hist)[2:]) > 0
    assert ig.clamp_max == io.clamp_max
    g0.close()


def test_config4_checkpoint_restart_on_breaking_onset_and_maximum_runup(O, G):
    """Config 4 at 1024 x 48.  The CUDA path runs the whole 2000 steps alone, checkpointing every 25
    steps; from the checkpoint before breaking first fires and from the one before the maximum
    run-up both sides are restarted (nh_set_state + nh_set_time: the checkpoint of SURVEY section 5)
    and advanced 50 steps side by side.  Valid because B1 < B2 makes the breaking flag stateless
    (R11) and p~ (the solver's start vector) is part of the checkpoint."""
    cfg = inputs.make_config(4, nx=1024, ny=48)
    prm = cfg["params"]
    assert prm["B1"] < prm["B2"]
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    wet0 = cfg["h"] > 1e-5
    cps = []
    for k in range(80):
        s = g.get_state()
        i = g.info()
        nbreak = 0
        if i.dt_last > 0.0:
            b = g.breaking(i.dt_last)
            nbreak = int(np.sum(b["w"] != s["w"]))
        cps.append(dict(state=s, t=i.t, nbreak=nbreak, runup=int(np.sum((s["h"] > 1e-5) & ~wet0))))
        g.step(25)
        assert g.sync() == 0
    cps.append(dict(state=g.get_state(), t=g.info().t, nbreak=0, runup=0))   # the end of the run
    first_break = next(k for k, c in enumerate(cps) if c["nbreak"] > 0)
    top = min(int(np.argmax([c["runup"] for c in cps])), len(cps) - 2)
    assert first_break >= 2 and cps[top]["runup"] > 48 * 20
    for name, k0 in (("breaking onset", first_break - 1), ("maximum run-up", max(top - 1, 0))):
        c = cps[k0]
        s = c["state"]
        o = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
        g2 = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
        for a in (o, g2):
            a.set_state(s["h"], s["qx"], s["qy"], s["w"], s["p"])
            a.set_time(c["t"])
        for _ in range(2):
            o.step(25)
            g2.step(25)
            assert g2.sync() == 0
            so, sg = o.get_state(), g2.get_state()
            r = parity(sg, so, cfg["H"], cfg["h0"])
            assert all(np.isfinite(v) and v <= 1.0 for v in r.values()), (name, r)
            assert np.array_equal(sg["h"] > 1e-5, so["h"] > 1e-5), name
        assert g2.info().t == pytest.approx(o.info().t, rel=1e-12)
        # the restarted run retraces the uninterrupted one (same kernels, same start vector)
        ref = cps[k0 + 2]["state"]
        assert_parity(sg, ref, cfg["H"], cfg["h0"])
        if name == "breaking onset":
            probe = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
            probe.set_state(so["h"], so["qx"], so["qy"], so["w"], so["p"])
            assert np.sum(probe.breaking(o.info().dt_last)["w"] != so["w"]) > 0
        g2.close()
    g.close()


@pytest.mark.parametrize("window", ["source", "coast"])
def test_config5_tsunami_crops_200_steps(O, G, window):
    # crops of the 819.2 km basin with the same dx = 100 m, depths and slopes (h/dx = 40, the
    # conditioning of the full grid): the uplift region, and the shelf with the emerged coast
    cfg = inputs.make_config(5, nx=256, ny=256, window=window)
    assert cfg["steps"] == 200
    o, g, worst = side_by_side(O, G, cfg, 200)
    assert g.info().clamps == o.info().clamps
    if window == "coast":
        assert np.any(cfg["h"] == 0.0) and np.any(cfg["h"] > 0.0)     # the shoreline is inside


def test_config5_source_crop_1024_twenty_steps(O, G):
    # a crop of the tsunami basin large enough for the marching warps to run in their full-size shape
    # (18 strips of 60 columns, bands of many rows, several CTAs per SM busy) and for the Krylov solve to
    # need hundreds of iterations: 20 whole steps against the oracle at 4 checkpoints, every field at the
    # north_star bars, qx and qy each against its own maximum
    cfg = inputs.make_config(5, nx=1024, ny=1024, window="source")
    o, g, worst = side_by_side(O, G, cfg, 20, ncp=4)
    assert g.info().clamps == o.info().clamps == 0
    assert g.info().iters_total > 20 * 2 * 100
    # the iteration counts of two valid solves of the same systems stay close
    assert abs(g.info().iters_total - o.info().iters_total) <= 0.05 * o.info().iters_total
