#!/usr/bin/env python
"""bench.py -- throughput of the full non-hydrostatic time step on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--config 1..5]

A "step" is one full two-stage Runge-Kutta non-hydrostatic step (CFL dt, then per stage:
predictor, breaking sources, pressure assembly + BiCGStab solve to 1e-12, correction; RK
combine) of BASELINE.json's headline workload: configs[4], the 8192 x 8192 tsunami grid, fp64,
on seeded synthetic input (paper_1706_04551_b200/inputs.py).  `metric` = cell-updates/s =
nx*ny*K / device time of the K timed steps (CUDA events on the context's stream, state resident
in HBM).  `e2e` = the same through the C ABI with HOST buffers: every step copies the state in
from pinned host memory (nh_set_state), steps (nh_step), and copies it out (nh_get_state).

N > 1 (torchrun): the path is single-GPU (replicas only), so every rank
runs an independent replica of the workload; value = cells updated by all ranks / max-over-ranks
time; no data-path collective.

--impl reference: the CPU oracle (oracle/, as it stands) timed on the host cores on a bounded
crop of the same workload (rank 0 only).

Other modes (records for profiles/, not the driver's line): --solver srj (the paper's own solver),
--precision 32 (the labelled fp32 variant), --hydrostatic (SWE mode: alu-bound predictor roofline
against the fp64 rate measured live), --onesolve (one isolated solve for the ncu capture behind
profiles/traffic.json), --table2 (the paper's timing experiment), --fullruns (every config at full
size and length), --parityruns [--spread] [--solver srj] [--precision 32] [--param k=v] (the CUDA
path beside the oracle over a configured horizon, ratios at the parity bars every 10 %).
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/s per full NH step (fp64)"
UNIT = "cell-updates/s"
# Algorithmic bytes of the dominant kernel:
# one Jacobi-preconditioned BiCGStab iteration moves >= 20 doubles per node.
BYTES_PER_NODE_ITER = 160.0
ORACLE_CROP = 640          # cpu_baseline / reference sample: crop of the config-5 basin (cells per side);
                           # --oracle-crop changes it and the line says so (config.oracle_crop)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); mx.append(float(f[1]))
                except ValueError:
                    continue
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            os.unlink(self.path)
        except Exception:
            pass
        if not sm:   # timed region shorter than one sampling period: one reading right after it
            try:
                r = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                    "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=20)
                f = [x.strip() for x in r.stdout.strip().splitlines()[0].split(",")]
                sm.append(float(f[0])); mx.append(float(f[1]))
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
                out["note"] = "timed region < 200 ms: sampled once right after it"
            except Exception:
                pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def _oracle_sample(steps, warmup, crop):
    """Time the CPU oracle (as it stands) on a crop of the config-5 basin: same dx, depths,
    conditioning (h/dx = 40); `steps` full RK2 NH steps after `warmup`.  ONE protocol for the
    cpu_baseline leg of the B200 arm and for `--impl reference`: both pass --steps / --warmup /
    --oracle-crop as given, so the same flags time the same oracle work."""
    from oracle import nh_oracle
    from paper_1706_04551_b200 import inputs
    cfg = inputs.make_config(5, nx=crop, ny=crop)
    o = nh_oracle.Oracle(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], **cfg["params"])
    o.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    info = o.info()
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return dict(value=crop * crop * steps / dt, seconds=dt, cores=cores, cells=crop * crop,
                iters_per_solve=info.iters_total / max(info.solves, 1),
                sample=f"config 5 'source' crop {crop}x{crop} cells (same dx, depth, h/dx=40), "
                       f"{steps} full RK2 step(s) after {warmup} warm-up")


def max_over_ranks(x, world, device=None):
    """MAX over the ranks of a process group (any backend; world 1: identity)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cells_per_replica, steps, world, seconds_max):
    """Replicas only: every rank advances its own copy of the workload, so the job
    updates world * cells * steps cells in the max-over-ranks time."""
    return world * cells_per_replica * steps / seconds_max


def _predictor_roofline(nh, prof, nc, args, hbm_peak, hbm_src):
    """SWE mode: the dominant kernel is the fused predictor, bounded by the plain fp64 ALUs.
    achieved = fp64-pipe warp instructions per second = (instructions per cell, ncu sm__inst_executed_pipe_fp64
    of this kernel on this workload, profiles/traffic.json) x cells x launches / CUDA-event time of the launches;
    peak = the fp64 FMA rate measured live by nh_fp64_rate (/ 32: warp instructions).  The HBM side (56 B per
    cell) is reported beside it; the bound is the slower of the two."""
    pm, pn = prof["predictor"]
    rate = nh.fp64_rate() / 32.0
    per_cell = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        try:
            per_cell = json.load(open(tp)).get("predictor_fp64_pipe_warp_inst_per_cell", {}).get(
                "f32" if args.precision == 32 else "f64")
        except Exception:
            pass
    t = pm * 1e-3
    hbm = 56.0 * (0.5 if args.precision == 32 else 1.0) * nc * pn / t / 1e9 if t > 0 else 0.0
    out = {"bound": "alu", "kernel": "k_predictor (one launch per Runge-Kutta stage)", "unit": "fp64 warp-instructions/s",
           "peak": rate, "peak_source": "measured live: nh_fp64_rate (DFMA chains), / 32",
           "achieved": None, "frac": None, "traffic": None,
           "fp64_pipe_warp_inst_per_cell": per_cell, "launches": pn, "avg_launch_ms": pm / max(pn, 1),
           "cells_per_s_per_launch": nc * pn / t if t > 0 else None,
           "hbm_side": {"bytes_per_cell": 56.0 * (0.5 if args.precision == 32 else 1.0), "achieved_GBs": hbm,
                        "peak_GBs": hbm_peak, "frac": hbm / hbm_peak, "peak_source": hbm_src},
           "phase_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()}}
    if per_cell and t > 0:
        out["achieved"] = per_cell * nc * pn / t
        out["frac"] = out["achieved"] / rate
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    r = _oracle_sample(args.steps, args.warmup, args.oracle_crop)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * r["seconds"] / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "configs[4] tsunami 8192x8192 (timed on a bounded crop, see cpu_baseline.sample)",
                   "solver": "Jacobi-BiCGStab rtol 1e-12", "iters_per_solve": r["iters_per_solve"],
                   "oracle_crop": args.oracle_crop},
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                         "sample": r["sample"], "iters_per_solve": r["iters_per_solve"], "seconds": r["seconds"]},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_1706_04551_b200 import inputs, nh

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    kw = {}
    if args.nx:
        kw["nx"] = args.nx
    if args.ny:
        kw["ny"] = args.ny
    cfg = inputs.make_config(args.config, **kw)
    nx, ny = cfg["nx"], cfg["ny"]
    nc, nn = nx * ny, (nx + 1) * (ny + 1)
    stream = torch.cuda.Stream(device=dev)
    prm = dict(cfg["params"])
    if args.solver == "srj":
        prm.update(solver=1, srj_eps=args.srj_eps)
    if args.precision == 32:      # the optional fp32 variant: labelled, never the headline
        prm.update(precision=32, solver_rtol=1e-4)
    if args.hydrostatic:          # SWE mode (nonhydro = 0): the step is the fused predictor alone (Table 2, column SWE)
        prm.update(nonhydro=0)
    sim = nh.NH(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], stream=stream, **prm)
    sim.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])

    # ---- device-resident leg: W warm-up steps, then exactly K timed steps
    sim.step(args.warmup)
    sim.sync()
    i0 = sim.info()
    l0 = sim.launch_count()
    sim.profile(True)
    clocks = ClockSampler(local)
    barrier()
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        sim.step(1)
    e1.record(stream)
    barrier()
    clk = clocks.stop()
    st = sim.sync()
    ms = e0.elapsed_time(e1)
    prof = sim.profile_read()
    sim.profile(False)
    i1 = sim.info()
    launches = sim.launch_count() - l0
    ms_max = max_over_ranks(ms, world, dev)
    value = whole_job_value(nc, args.steps, world, ms_max * 1e-3)
    iters = i1.iters_total - i0.iters_total
    solves = i1.solves - i0.solves

    # ---- roofline of the dominant kernel (the BiCGStab solve), timed live with CUDA events
    peak, peak_src = _peaks()
    sol_ms, sol_n = prof["solver"]
    node_iters = (iters + solves) * float(nn)          # + the polish iteration of every solve (solver 1: + the
                                                       # sweep that meets the stopping rule)
    half = 0.5 if args.precision == 32 else 1.0
    # ALGORITHMIC bytes per node-iteration of the kernel as built: the matrix-free
    # two-pass BiCGStab iteration reads / writes 18 planes (144 B in fp64); one Jacobi sweep of k_srj reads
    # x, b', 4 coefficients and writes x' (56 B).  `achieved` and `frac` are computed from THIS figure.
    # SURVEY 8(d)'s 160 B describes a solver with stored rows; the rate on that model is only the labelled
    # side field `effective_on_survey_160B_model` (it overstates the DRAM rate of this kernel by 11 %).
    bytes_unit = (56.0 if args.solver == "srj" else 144.0) * half
    survey_unit = (56.0 if args.solver == "srj" else BYTES_PER_NODE_ITER) * half
    per_s = node_iters / (sol_ms * 1e-3) / 1e9 if sol_ms > 0 else 0.0
    achieved = bytes_unit * per_s
    # measured DRAM traffic: ncu dram__bytes_read + write per node-iteration of the SAME kernel
    # (profiles/traffic.json names the capture), scaled by this run's node-iterations per launch
    traffic, traffic_unit = None, None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        try:
            tj = json.load(open(tp))
            key = ("k_srj" if args.solver == "srj" else "k_bicgstab") + ("_f32" if args.precision == 32 else "_f64")
            if key in tj.get("dram_bytes_per_node_iteration", {}) and nx * ny >= 4096 * 4096:
                traffic_unit = float(tj["dram_bytes_per_node_iteration"][key])
                traffic = traffic_unit * node_iters / max(sol_n, 1)
        except Exception:
            pass
    if args.hydrostatic:
        roofline = _predictor_roofline(nh, prof, nc, args, peak, peak_src)
    else:
      roofline = {
        "bound": "hbm", "kernel": ("k_srj" if args.solver == "srj" else "k_bicgstab") +
                                  " (one cooperative launch per pressure solve)",
        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
        "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / 8000.0,
        "bytes_per_node_iteration": bytes_unit,
        "bytes_source": "the planes this kernel must move per node-iteration (DESIGN.md section 6; fp32 variant: half)",
        "effective_on_survey_160B_model": {"bytes_per_node_iteration": survey_unit, "GB/s": survey_unit * per_s,
                                           "frac": survey_unit * per_s / peak,
                                           "note": "SURVEY.md 8(d) per-unit figure of a stored-row solver: not this "
                                                   "kernel's DRAM rate"},
        "achieved_dram": {"GB/s": traffic_unit * per_s, "frac": traffic_unit * per_s / peak}
                         if traffic_unit is not None else None,
        "traffic_per_node_iteration": traffic_unit,
        "traffic_note": "derived: ncu DRAM bytes per node-iteration of this kernel (profiles/traffic.json) x this run's "
                        "node-iterations per launch" if traffic is not None else None,
        "launches": sol_n,
        "avg_launch_ms": sol_ms / max(sol_n, 1),
        "iterations_per_launch": (iters + solves) / max(solves, 1),
        "phase_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()},
        "kernel_share_of_step": sol_ms / ms if ms > 0 else None,
      }

    # ---- end-to-end leg: host buffers in and out through the C ABI every step, on the SAME step window as the
    # device leg (steps W+1 .. W+K of the run): a fresh context is taken through the same warm-up -- its last
    # warm-up step already through the host buffers (pages them in, same code path) -- so that both legs do
    # the same solves (bit-identical states, same iteration counts) and differ only by the copies.  The state
    # comes back through nh_continue_state: the caller says that the run goes on (the solver keeps its history).
    sim.close()
    sim = nh.NH(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], stream=stream, **prm)
    sim.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    hb = [{k: torch.empty(cfg[k].shape, dtype=torch.float64).pin_memory() for k in ("h", "qx", "qy", "w", "p")}
          for _ in range(2)]

    def e2e_step():
        a, b = hb[0], hb[1]
        sim.set_state(*(a[k].numpy() for k in ("h", "qx", "qy", "w", "p")), keep_history=True)
        sim.step(1)
        sim.get_state({k: v.numpy() for k, v in b.items()})   # synchronises: the result is on the host
        hb.reverse()

    if args.warmup > 1:
        sim.step(args.warmup - 1)
    sim.get_state({k: v.numpy() for k, v in hb[0].items()})
    if args.warmup >= 1:
        e2e_step()
    ie0 = sim.info()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    ie1 = sim.info()
    e2e_max = max_over_ranks(e2e_s, world, dev)
    e2e_value = whole_job_value(nc, args.steps, world, e2e_max)
    e2e_iters = (ie1.iters_total - ie0.iters_total) / max(ie1.solves - ie0.solves, 1)
    st2 = sim.sync()
    io_bytes = 8 * (3 * nc + 2 * nn)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.precision == 32 else "f64", "data": "synthetic",
        "config": {"workload": f"configs[{args.config - 1}] {cfg['name']} {nx}x{ny} cells, dx={cfg['dx']} m"
                               + (" -- fp32 VARIANT (precision = 32, solver_rtol 1e-4), not the fp64 headline" if args.precision == 32 else "")
                               + (" -- SWE MODE (nonhydro = 0: predictor only), not the headline" if args.hydrostatic else ""),
                   "solver": (("Jacobi-BiCGStab rtol %s, device-resident convergence" % ("1e-4" if args.precision == 32 else "1e-12")) if args.solver == "bicgstab"
                              else f"scheduled-relaxation Jacobi (paper's solver), increment rule (32) eps {args.srj_eps:g}"),
                   "iters_per_solve": iters / max(solves, 1), "time_order": 2,
                   "l2": "working set >> L2 (one fp64 plane = %.0f MB); no flush needed" % (8e-6 * nc)
                         if 8 * nc > 200e6 else "working set near/below L2 size: L2-resident, not an HBM claim",
                   "parallelism": "replicas" if world > 1 else "single GPU",
                   "status": [int(st), int(st2)], "clamps": int(i1.clamps)},
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes,
                "d2h_bytes_per_step": io_bytes, "ms_per_step": 1e3 * e2e_max / args.steps,
                "iters_per_solve": e2e_iters, "window": "steps %d..%d of the run, as the device leg" % (args.warmup + 1, args.warmup + args.steps)},
        "gpu_launches": int(launches),
        "roofline": roofline,
    }
    if rank == 0 and world == 1 and not args.no_cpu:
        r = _oracle_sample(args.steps, args.warmup, args.oracle_crop)   # what --impl reference runs on these flags
        line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                "sample": r["sample"], "seconds": r["seconds"],
                                "iters_per_solve": r["iters_per_solve"]}
        line["config"]["oracle_crop"] = args.oracle_crop
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_streammix(args):
    """What HBM gives the solver's own read / write mix (nh_stream_mix_rate): planes of the node-plane size of
    --config, a plain streaming kernel per mix.  One BiCGStab iteration is one pass B (5 planes read, 1 written)
    plus one pass CA (8 read, 4 written) = 18 planes = 144 B per node: the floor per iteration is the sum of the
    two passes at the rates their mixes reach, to hold against the ms per iteration bench.py measures.  One
    JSON line; a record for profiles/, not the driver's bench line."""
    import torch
    from paper_1706_04551_b200 import inputs, nh
    torch.cuda.set_device(0)
    kw = {}
    if args.nx:
        kw["nx"] = args.nx
    if args.ny:
        kw["ny"] = args.ny
    cfg = inputs.make_config(args.config, **kw)
    nn = (cfg["nx"] + 1) * (cfg["ny"] + 1)
    n = nn + (nn & 1)
    peak, peak_src = _peaks()
    clocks = ClockSampler(0)
    clocks.start()
    rates = {}
    for rep in range(3):          # three rounds: the median per mix
        for mix in ((1, 1), (5, 1), (8, 4), (6, 1)):
            rates.setdefault(mix, []).append(nh.stream_mix_rate(mix[0], mix[1], n))
    clk = clocks.stop()
    med = {m: float(np.median(v)) for m, v in rates.items()}
    plane = 8.0 * nn
    tB, tCA = 6 * plane / (med[(5, 1)] * 1e9), 12 * plane / (med[(8, 4)] * 1e9)
    print(json.dumps({
        "streammix": f"{cfg['name']} {cfg['nx']}x{cfg['ny']}", "nodes": nn, "plane_MB": plane / 1e6,
        "GBs": {f"{m[0]}R+{m[1]}W": med[m] for m in med}, "all_GBs": {f"{m[0]}R+{m[1]}W": v for m, v in rates.items()},
        "copy_peak_GBs": peak, "peak_source": peak_src,
        "frac_of_copy_peak": {f"{m[0]}R+{m[1]}W": med[m] / peak for m in med},
        "bicgstab_floor_ms_per_iteration": 1e3 * (tB + tCA),
        "bicgstab_floor_note": "pass B (5R+1W, 6 planes) + pass CA (8R+4W, 12 planes) at the rates of their mixes; no "
                               "halo rows, no grid barrier, no arithmetic",
        "bicgstab_floor_GBs_at_144B": 144.0 * nn / (tB + tCA) / 1e9,
        "srj_floor_ms_per_sweep": 1e3 * 7 * plane / (med[(6, 1)] * 1e9), "clocks": clk}))
    return 0


def run_onesolve(args):
    """One pressure solve in isolation, for the ncu capture behind profiles/traffic.json: W warm-up
    steps, then nh_nonhydro_correct(dt_last) = exactly one launch of the solver kernel; prints its
    iteration count so that DRAM bytes per node-iteration = ncu bytes / ((iterations + 1) x nodes).
    Capture with: ncu --set full -k regex:k_bicgstab -s <2 W> -c 1 python bench.py --onesolve ..."""
    import torch
    from paper_1706_04551_b200 import inputs, nh
    torch.cuda.set_device(0)
    kw = {}
    if args.nx:
        kw["nx"] = args.nx
    if args.ny:
        kw["ny"] = args.ny
    cfg = inputs.make_config(args.config, **kw)
    prm = dict(cfg["params"])
    if args.solver == "srj":
        prm.update(solver=1, srj_eps=args.srj_eps)
    if args.precision == 32:
        prm.update(precision=32, solver_rtol=1e-4)
    stream = torch.cuda.Stream()
    sim = nh.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], stream=stream, **prm)
    sim.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
    sim.step(args.warmup)
    sim.sync()
    dt = sim.info().dt_last
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sim.profile(True)
    e0.record(stream)
    sim.nonhydro_correct(dt)
    e1.record(stream)
    st = sim.sync()
    prof = sim.profile_read()
    i = sim.info()
    nn = (cfg["nx"] + 1) * (cfg["ny"] + 1)
    print(json.dumps(dict(onesolve=cfg["name"], nx=cfg["nx"], ny=cfg["ny"], precision=args.precision, solver=args.solver,
                          iterations=int(i.iters_last), node_iterations=(int(i.iters_last) + 1) * nn,
                          solver_ms=prof["solver"][0], status=int(st), res_last=i.res_last)))
    return 0


def run_table2(args):
    """The paper's own timing experiment (Table 2) on this GPU: circular dam
    break to t = 1, CFL 0.9, SWE (nonhydro = 0) and NH with the paper's solver (solver 1) at its
    three tolerances, wall time of the whole time loop on the device (CUDA events around it; whole
    steps until t >= 1, checked on the host every 25 steps).  Context, not the headline metric."""
    import torch
    from paper_1706_04551_b200 import inputs, nh
    torch.cuda.set_device(0)
    sizes = [int(x) for x in args.table2.split(",")]
    paper = {}   # the paper's printed seconds (tests/golden/table2_seconds.txt, cited there)
    gp = os.path.join(ROOT, "tests", "golden", "table2_seconds.txt")
    if os.path.exists(gp):
        for line in open(gp):
            f = line.split()
            if f and not line.startswith("#"):
                paper[int(f[0])] = dict(zip(("swe", "nh_1e-3", "nh_1e-4", "nh_1e-5"), map(float, f[1:5])))
    rows = []
    for n in sizes:
        cfg = inputs.paper_dam_break(n)
        row = {"n": n}
        for tag, over in (("swe", dict(nonhydro=0)), ("nh_1e-3", dict(solver=1, srj_eps=1e-3)),
                          ("nh_1e-4", dict(solver=1, srj_eps=1e-4)), ("nh_1e-5", dict(solver=1, srj_eps=1e-5))):
            prm = dict(cfg["params"]); prm.update(over)
            prm["solver_maxit"] = 1000000   # plain-Jacobi phases across the initial discontinuity are long
            stream = torch.cuda.Stream()
            sim = nh.NH(n, n, cfg["dx"], cfg["dy"], cfg["H"], stream=stream, **prm)
            sim.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
            sim.step(2); sim.sync()                                   # warm-up (module load, caches)
            sim.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            i0 = sim.info()
            e0.record(stream)
            while True:
                sim.step(25)
                sim.sync()
                if sim.info().t - i0.t >= 1.0:
                    break
            e1.record(stream)
            torch.cuda.synchronize()
            i1 = sim.info()
            row[tag] = {"seconds": e0.elapsed_time(e1) * 1e-3, "steps": int(i1.steps - i0.steps),
                        "t_end": i1.t - i0.t,
                        "sweeps_per_solve": (i1.iters_total - i0.iters_total) / max(i1.solves - i0.solves, 1)}
            sim.close()
            if n in paper:
                row[tag]["paper_seconds_titan_black"] = paper[n][tag]
                row[tag]["paper_over_b200"] = paper[n][tag] / row[tag]["seconds"]
            print(f"table2 n={n} {tag}: {row[tag]}", file=sys.stderr, flush=True)
        rows.append(row)
    print(json.dumps({"table2": rows, "unit": "seconds of the whole time loop to t >= 1",
                      "note": "PAPER.md Table 2 workload; paper's numbers are on a GTX Titan Black"}))
    return 0


def run_fullruns(args):
    """Every listed BASELINE.json config at full size for its full number of steps (one nh_step call,
    CUDA events around it): status, iterations, clamps, mass.  A robustness record, not the metric."""
    import torch
    from paper_1706_04551_b200 import inputs, nh
    torch.cuda.set_device(0)
    for idx in [int(x) for x in args.fullruns.split(",")]:
        cfg = inputs.make_config(idx)
        steps = cfg["steps"]
        stream = torch.cuda.Stream()
        g = nh.NH(cfg["nx"], cfg["ny"], cfg["dx"], cfg["dy"], cfg["H"], stream=stream, **cfg["params"])
        g.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        g.step(steps)
        e1.record(stream)
        status = g.sync(allow=(nh.ENOCONV,))
        torch.cuda.synchronize()
        i, s = g.info(), g.get_state()
        sec = e0.elapsed_time(e1) * 1e-3
        m0 = float(np.sum(cfg["h"], dtype=np.longdouble))
        m1 = float(np.sum(s["h"], dtype=np.longdouble))
        print(json.dumps(dict(
            config=idx, name=cfg["name"], nx=cfg["nx"], ny=cfg["ny"], steps=int(i.steps), seconds=sec,
            cell_updates_per_s=cfg["nx"] * cfg["ny"] * steps / sec, status=int(status), t_end=i.t,
            iters_per_solve=i.iters_total / max(i.solves, 1), iters_max=int(i.iters_max), res_last=i.res_last,
            clamps=int(i.clamps), mass_rel_change=(m1 - m0) / m0,
            finite=bool(all(np.isfinite(s[k]).all() for k in s)))), flush=True)
        g.close()
    return 0


def parity_ratios(go, oo, H, h0, g=9.81, tol=1e-9):
    """error / allowed per field at the north_star bars (SURVEY 8(d) "Parity metric"): all <= 1 passes.
    max|eta_g - eta_o| <= tol h0;  max|a_g - a_o| <= tol max(max|a_o|, 1e-3 floor_a) for a in q, w, p,
    floors (h0 c0, c0, g h0), c0 = sqrt(g h0).  The discharge is reported twice: qx_own, qy_own = each component
    against its own maximum (the north_star bar), qx, qy = both against max|q| (the joint bar of DESIGN.md
    section 4, weaker where one component is small)."""
    c0 = float(np.sqrt(g * h0))
    out = {"eta": float(np.max(np.abs((go["h"] - H) - (oo["h"] - H))) / (tol * h0))}
    qscale = max(float(np.max(np.abs(oo["qx"]))), float(np.max(np.abs(oo["qy"]))), 1e-3 * h0 * c0)
    for k in ("qx", "qy"):
        out[k] = float(np.max(np.abs(go[k] - oo[k])) / (tol * qscale))
        out[k + "_own"] = float(np.max(np.abs(go[k] - oo[k])) / (tol * max(float(np.max(np.abs(oo[k]))), 1e-3 * h0 * c0)))
    for k, f in dict(w=c0, p=g * h0).items():
        scale = max(float(np.max(np.abs(oo[k]))), 1e-3 * f)
        out[k] = float(np.max(np.abs(go[k] - oo[k])) / (tol * scale))
    return out


def fp32_ratios(go, oo, H, h0, g=9.81):
    """error / allowed at the bars of the fp32 variant (tests/test_gpu_fp32.py):
    max|d eta| <= 1e-4 max|eta_o|, max|d q| <= 1e-4 max|q_o|, max|d w| <= 1e-3 max|w_o|, max|d p| <= 1e-2 max|p_o|,
    floors 1e-3 of the natural scales (eta: 1e-2 h0, i.e. never below 1e-6 h0 = 17 u32 h0)."""
    c0 = float(np.sqrt(g * h0))
    wet = oo["h"] > 1e-5
    eo = oo["h"] - H
    esc = max(float(np.max(np.abs(eo[wet]))) if wet.any() else 0.0, 1e-2 * h0)
    out = {"eta": float(np.max(np.abs(go["h"] - oo["h"])) / (1e-4 * esc))}
    qs = max(float(np.max(np.abs(oo["qx"]))), float(np.max(np.abs(oo["qy"]))), 1e-3 * h0 * c0)
    for k in ("qx", "qy"):
        out[k] = float(np.max(np.abs(go[k] - oo[k])) / (1e-4 * qs))
    out["w"] = float(np.max(np.abs(go["w"] - oo["w"])) / (1e-3 * max(float(np.max(np.abs(oo["w"]))), 1e-3 * c0)))
    out["p"] = float(np.max(np.abs(go["p"] - oo["p"])) / (1e-2 * max(float(np.max(np.abs(oo["p"]))), 1e-3 * g * h0)))
    return out


def run_parityruns(args):
    """Configured-horizon parity (north_star: "after the configured steps"): the CUDA path and the CPU
    oracle advance the same seeded config side by side; at 10 checkpoints (every 10 % of the run; after every step of a run shorter than 10) the
    full states are compared at the north_star bars.  SPEC = idx:NXxNY:steps[:window], comma-separated.
    One JSON line per run.  Slow (the oracle runs on the host cores): a record for profiles/, not the
    driver's bench line."""
    import torch
    from oracle import nh_oracle
    from paper_1706_04551_b200 import inputs, nh
    torch.cuda.set_device(0)
    for spec in args.parityruns.split(","):
        f = spec.split(":")
        idx, (nx, ny), steps = int(f[0]), map(int, f[1].lower().split("x")), int(f[2])
        kw = dict(nx=nx, ny=ny)
        if len(f) > 3:
            kw["window"] = f[3]
        cfg = inputs.make_config(idx, **kw)
        prm = dict(cfg["params"])
        if args.solver == "srj":      # the paper's solver: both sides do the same arithmetic (bit-exact)
            prm.update(solver=1, srj_eps=args.srj_eps)
        for kv in args.param:         # e.g. --param manning_n=0.01
            k_, v_ = kv.split("=")
            prm[k_] = float(v_) if "." in v_ or "e" in v_.lower() else int(v_)
        o = nh_oracle.Oracle(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], **prm)
        gprm = dict(prm)
        if args.precision == 32:      # the fp32 variant against the fp64 oracle, at ITS bars (fp32_ratios)
            gprm.update(precision=32, solver_rtol=max(1e-4, args.rtol32))
        g = nh.NH(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], **gprm)
        o2 = None
        if args.spread:               # a second, equally valid oracle run: solver tolerance 10 x tighter
            prm2 = dict(prm)
            if args.solver == "srj":
                prm2["srj_eps"] = 0.1 * args.srj_eps
            else:
                prm2["solver_rtol"] = 0.1 * prm.get("solver_rtol", 1e-12)
            o2 = nh_oracle.Oracle(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], **prm2)
        for a in (o, g, o2):
            if a is not None:
                a.set_state(cfg["h"], cfg["qx"], cfg["qy"], cfg["w"], cfg["p"])
        probe = nh_oracle.Oracle(nx, ny, cfg["dx"], cfg["dy"], cfg["H"], **prm) if prm.get("breaking") else None
        eps_dry = 1e-5
        wet0 = int(np.sum(cfg["h"] > eps_dry))
        cps, worst, worst_own, done = [], 0.0, 0.0, 0
        t_o = t_g = 0.0
        ncp = max(1, min(10, steps))
        for k in range(ncp):
            n = (steps * (k + 1)) // ncp - done
            t0 = time.perf_counter(); o.step(n, allow_noconv=True); t_o += time.perf_counter() - t0
            t0 = time.perf_counter(); g.step(n); stg = g.sync(allow=(nh.ENOCONV,)); t_g += time.perf_counter() - t0
            done += n
            so, sg = o.get_state(), g.get_state()
            io, ig = o.info(), g.info()
            r = (fp32_ratios if args.precision == 32 else parity_ratios)(sg, so, cfg["H"], cfg["h0"])
            worst = max(worst, max(v for a, v in r.items() if not a.endswith("_own")))
            worst_own = max(worst_own, max(r.values()))
            spread = None
            if o2 is not None:
                o2.step(n, allow_noconv=True)
                spread = parity_ratios(o2.get_state(), so, cfg["H"], cfg["h0"])
            wet = so["h"] > eps_dry
            cp = dict(step=done, t_oracle=io.t, t_gpu=ig.t, ratios={a: round(b, 4) for a, b in r.items()},
                      iters_total=[int(ig.iters_total), int(io.iters_total)], clamps=[int(ig.clamps), int(io.clamps)],
                      wet_cells=int(wet.sum()), wet_cells_changed_vs_start=int(np.sum(wet != (cfg["h"] > eps_dry))),
                      wet_mask_equal=bool(np.array_equal(wet, sg["h"] > eps_dry)),
                      eta_max=float(np.max(np.where(wet, so["h"] - cfg["H"], -np.inf))), gpu_status=int(stg),
                      bit_exact=bool(all(np.array_equal(sg[a], so[a]) for a in so)))
            if spread is not None:    # oracle (tolerance / 10) against oracle: what two valid solves differ by
                cp["oracle_spread_ratios"] = {a: round(b, 4) for a, b in spread.items()}
            if probe is not None:   # where is the breaking criterion of (9) active right now? (oracle S6 hook)
                probe.set_state(so["h"], so["qx"], so["qy"], so["w"], so["p"])
                b = probe.breaking(max(io.dt_last, 1e-9))
                cp["breaking_cells"] = int(np.sum((b["qx"] != so["qx"]) | (b["qy"] != so["qy"])))
                cp["breaking_nodes"] = int(np.sum(b["w"] != so["w"]))
            cps.append(cp)
            print(f"parityrun {spec} step {done}/{steps}: worst ratio {max(r.values()):.3g} "
                  f"(oracle {t_o:.0f} s, gpu {t_g:.1f} s)", file=sys.stderr, flush=True)
        io, ig = o.info(), g.info()
        print(json.dumps(dict(
            parityrun=spec, workload=cfg["name"], nx=nx, ny=ny, dx=cfg["dx"], steps=steps, h0=cfg["h0"],
            solver=("paper's Jacobi / scheduled relaxation, eps %g" % args.srj_eps) if args.solver == "srj" else "Jacobi-BiCGStab rtol 1e-12",
            precision=args.precision,
            bars="fp32 variant: 1e-4 max|eta|, 1e-4 max|q|, 1e-3 max|w|, 1e-2 max|p| (DESIGN.md section 10); ratio = error/allowed" if args.precision == 32 else"max|d eta| <= 1e-9 h0; max|d a| <= 1e-9 max(max|a|, 1e-3 floor_a), a in qx_own, qy_own, w, p (north_star, per component: worst_ratio_per_component) and with qx, qy against max|q| (joint bar: worst_ratio); ratio = error/allowed",
            worst_ratio=worst, passed=bool(worst <= 1.0), worst_ratio_per_component=worst_own,
            passed_per_component=bool(worst_own <= 1.0), checkpoints=cps, wet_cells_start=wet0,
            clamp_hist_bins_m="<1e-15,<1e-12,<1e-9,<1e-6,<1e-3,>=1e-3",
            clamp_hist_gpu=list(ig.clamp_hist), clamp_hist_oracle=list(io.clamp_hist),
            clamp_max_gpu=ig.clamp_max, clamp_max_oracle=io.clamp_max,
            mass_rel_change_oracle=float(np.sum(so["h"], dtype=np.longdouble) / np.sum(cfg["h"], dtype=np.longdouble) - 1),
            oracle_seconds=t_o, gpu_seconds=t_g, oracle_threads=int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1)))),
            flush=True)
        g.close(); o.close()
        if o2 is not None:
            o2.close()
        if probe is not None:
            probe.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=5)   # >= 4 steps fill the start-vector history (R32)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--nx", type=int, default=0)
    ap.add_argument("--ny", type=int, default=0)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--oracle-crop", type=int, default=ORACLE_CROP,
                    help="cells per side of the config-5 crop the CPU oracle is timed on (cpu_baseline, --impl reference)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32],
                    help="32: the optional fp32 variant (labelled as such; the fp64 line is the headline)")
    ap.add_argument("--solver", default="bicgstab", choices=["bicgstab", "srj"],
                    help="bicgstab: north_star solver (default); srj: the paper's scheduled-relaxation Jacobi")
    ap.add_argument("--srj-eps", type=float, default=1e-5, help="stopping tolerance of eq. (32) for --solver srj")
    ap.add_argument("--table2", default="", help="comma-separated grid sizes: run the paper's Table 2 experiment instead")
    ap.add_argument("--fullruns", default="", help="comma-separated config numbers: run each at full size for its full step count")
    ap.add_argument("--parityruns", default="", help="idx:NXxNY:steps[:window],... : oracle beside the CUDA path over the "
                    "configured horizon, parity at 10 checkpoints (slow; a record for profiles/)")
    ap.add_argument("--rtol32", type=float, default=1e-4, help="--precision 32 with --parityruns: solver_rtol of the fp32 run")
    ap.add_argument("--hydrostatic", action="store_true", help="SWE mode (nonhydro = 0): the predictor alone; alu-bound roofline")
    ap.add_argument("--streammix", action="store_true", help="DRAM rate of plain streaming kernels with the solver's "
                    "read/write plane mixes on the node-plane size of --config (the floor of an iteration)")
    ap.add_argument("--onesolve", action="store_true", help="one isolated pressure solve after --warmup steps (ncu capture)")
    ap.add_argument("--param", action="append", default=[], help="--parityruns: override a parameter, key=value (repeatable)")
    ap.add_argument("--spread", action="store_true", help="--parityruns: also run a second oracle with a 10 x tighter "
                    "solver tolerance and report oracle-vs-oracle ratios (the spread of two valid solves)")
    args = ap.parse_args()
    if args.streammix:
        return run_streammix(args)
    if args.onesolve:
        return run_onesolve(args)
    if args.parityruns:
        return run_parityruns(args)
    if args.fullruns:
        return run_fullruns(args)
    if args.table2:
        return run_table2(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
