"""The optional fp32 variant (nh_params.precision = 32; north_star "optional fp32 variant")
against the fp64 CPU oracle (-m gpu).

All field planes and their arithmetic are fp32 (eta = h - H stored beside h), dt / clock / dot products
fp64, solver_rtol 1e-4.  Tolerances (derived from u32 = 6e-8 and the solver
tolerance, measured margins >= 8 in profiles/r02d_fp32.md), against the oracle state `o`:
    max|d eta| <= 1e-4 max|eta_o|;   max|d q| <= 1e-4 max|q_o| (q one vector);
    max|d w| <= 1e-3 max|w_o|;       max|d p| <= 1e-2 max|p_o|
with the floors of the fp64 bars (1e-3 of the natural scales); eta: floor 1e-2 h0, i.e. never below
1e-6 h0 = 17 u32 h0 -- the fluxes are formed from h = H + eta, which fp32 resolves to u32 h0.
"""
import numpy as np
import pytest

from paper_1706_04551_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    from paper_1706_04551_b200 import nh
    nh.lib()
    return nh


def fp32_ratios(sg, so, H, h0, g=9.81):
    c0 = np.sqrt(g * h0)
    wet = so["h"] > 1e-5
    eta_o, eta_g = so["h"] - H, sg["h"] - H
    esc = max(np.max(np.abs(eta_o[wet])) if wet.any() else 0.0, 1e-2 * h0)
    out = {"eta": np.max(np.abs(eta_g - eta_o)) / (1e-4 * esc)}
    qs = max(np.max(np.abs(so["qx"])), np.max(np.abs(so["qy"])), 1e-3 * h0 * c0)
    out["q"] = max(np.max(np.abs(sg["qx"] - so["qx"])), np.max(np.abs(sg["qy"] - so["qy"]))) / (1e-4 * qs)
    out["w"] = np.max(np.abs(sg["w"] - so["w"])) / (1e-3 * max(np.max(np.abs(so["w"])), 1e-3 * c0))
    out["p"] = np.max(np.abs(sg["p"] - so["p"])) / (1e-2 * max(np.max(np.abs(so["p"])), 1e-3 * g * h0))
    return out


def run32(O, G, cfg, checkpoints, **over):
    prm = dict(cfg["params"])
    prm.update(over)
    o = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **dict(prm, precision=32, solver_rtol=1e-4))
    for a in (o, g):
        a.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    done, worst = 0, {}
    for n in checkpoints:
        o.step(n - done)
        g.step(n - done)
        done = n
        assert g.sync() == 0
        r = fp32_ratios(g.get_state(), o.get_state(), cfg["H"], cfg["h0"])
        assert all(np.isfinite(v) and v <= 1.0 for v in r.values()), (n, r)
        worst = {k: max(worst.get(k, 0.0), v) for k, v in r.items()}
    assert g.info().t == pytest.approx(o.info().t, rel=1e-5) and g.info().steps == o.info().steps
    return o, g, worst


def test_fp32_rejects_nothing_silently_and_reports_precision(G):
    H = np.ones((8, 8))
    with pytest.raises(G.NHError) as e:
        G.NH(8, 8, 1.0, 1.0, H, precision=16)
    assert e.value.code == G.EINVAL
    g = G.NH(8, 8, 1.0, 1.0, H, precision=32)
    assert g.sync() == 0


def test_fp32_state_round_trip_keeps_eta_on_deep_water(G):
    # 4000 m of depth, 2 m of signal: eta = h - H is formed in fp64 and stored in fp32, so the surface
    # elevation survives to fp32 relative accuracy of ETA (an fp32 h alone would quantise it to 2.4e-4 m)
    rng = np.random.default_rng(3)
    H = 4000.0 + 300.0 * rng.standard_normal((40, 56))
    H[:4, :] = -20.0                                          # emerged land
    eta = 2.0 * rng.standard_normal((40, 56))
    h = np.maximum(H + eta, 0.0)
    q = 400.0 * rng.standard_normal((40, 56))
    g = G.NH(56, 40, 100.0, 100.0, H, precision=32)
    g.set_state(h, q, -q, None, None)
    s = g.get_state()
    wet = h > 0
    assert np.all(s["h"][~wet] == 0.0)
    assert np.max(np.abs((s["h"] - H)[wet] - eta[wet])) <= 2.0 ** -23 * np.max(np.abs(eta))
    assert np.max(np.abs(s["qx"] - q)) <= 2.0 ** -23 * np.max(np.abs(q))


def test_fp32_lake_at_rest_stays_exactly_at_rest(O, G):
    cfg = inputs.make_config(2, nx=128, ny=128)
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **dict(cfg["params"], precision=32))
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    g.step(200)
    assert g.sync() == 0
    s = g.get_state()
    assert np.all(s["qx"] == 0.0) and np.all(s["qy"] == 0.0) and np.all(s["w"] == 0.0) and np.all(s["p"] == 0.0)
    assert np.max(np.abs(s["h"] - cfg["h"])) <= 1e-6 and g.info().iters_total == 0


def test_fp32_config1_channel_full(O, G):
    cfg = inputs.make_config(1)
    o, g, worst = run32(O, G, cfg, [50, 100, 150, 200])
    assert 0 < g.info().iters_total < o.info().iters_total      # fewer iterations: tolerance 1e-4, not 1e-12


def test_fp32_config3_radial_hump_500_steps(O, G):
    cfg = inputs.make_config(3, nx=256, ny=256)
    run32(O, G, cfg, [100, 250, 500])


@pytest.mark.parametrize("window", ["source", "coast"])
def test_fp32_config5_tsunami_crops_200_steps(O, G, window):
    cfg = inputs.make_config(5, nx=256, ny=256, window=window)
    run32(O, G, cfg, [20, 100, 200])


def test_fp32_config4_beach_reduced(O, G):
    # generating zone, breaking and wet/dry bed in fp32 (before the breaking switch makes the run
    # sensitive to any perturbation, profiles/r02b_config4_sensitivity.md)
    cfg = inputs.make_config(4, nx=640, ny=8)
    run32(O, G, cfg, [100, 200])


def test_fp32_both_solvers_and_w_advection(O, G):
    from test_gpu_parity import BCS, rnd_cfg
    cfg = rnd_cfg(150, 77, BCS[2], seed=43, dry=0.2, dx=0.2, dy=0.25, w_advect=1)
    run32(O, G, cfg, [4])
    prm = dict(cfg["params"], solver=1, srj_eps=1e-5)
    o = O.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **dict(prm, precision=32))
    for a in (o, g):
        a.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
        a.step(4)
    assert g.sync() == 0
    r = fp32_ratios(g.get_state(), o.get_state(), cfg["H"], cfg["h0"])
    assert all(v <= 1.0 for v in r.values()), r


def test_fp32_effective_tolerance_and_stagnation_flag(G):
    """nh_info tells what the solver really stopped at: the effective tolerance (requests below 1e-4 are
    raised to 1e-4 in fp32, never in fp64), and -- bit 3 of flags -- whether any solve was accepted on a
    stalled true residual ABOVE that tolerance, so that a stall cannot pass for a converged solve."""
    from test_gpu_parity import BCS, rnd_cfg
    cfg = rnd_cfg(150, 77, BCS[1], seed=7, dry=0.2, dx=0.2, dy=0.25)
    prm = dict(cfg["params"], solver_rtol=1e-9)
    g64 = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **prm)
    assert g64.info().solver_rtol_effective == 1e-9
    g64.close()
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **dict(prm, precision=32))
    assert g.info().solver_rtol_effective == 1e-4
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    for _ in range(6):          # one step at a time: res_last is the residual of the step's last solve
        g.step(1)
        assert g.sync() == 0
        i = g.info()
        if not (i.flags & G.FLAG_STAGNATED):
            assert i.res_last <= i.solver_rtol_effective, (i.res_last, i.flags)
    g.close()
    # a tolerance fp32 cannot reach on a stiff operator (h / dx = 40, the config-5 conditioning): forced
    # through the solve hook with a right-hand side of full range; either the tolerance is met or the
    # acceptance is flagged -- never a silent pass above it
    cfg = inputs.make_config(5, nx=256, ny=256, window="source")
    g = G.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **dict(cfg["params"], precision=32, solver_rtol=1e-4))
    g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    b = inputs.random_smooth_state(256, 256, 1.0, 1.0, seed=3)["p"]
    x, it, rr = g.solve(b, allow=(G.ENOCONV,))
    g.step(1)                   # the hook clears the bits it set; a step's own solves set them again
    assert g.sync() == 0
    i = g.info()
    assert (i.flags & G.FLAG_STAGNATED) or i.res_last <= 1e-4
    g.close()
