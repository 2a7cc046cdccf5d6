#!/usr/bin/env python
"""bench.py -- throughput of the quadtree-LBM hot path on B200 (contract: one JSON line on stdout, rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--precision 64|32] [--addressing auto|list|bricks]
    python bench.py --impl reference ...          # the CPU oracle as it stands, timed on the host cores

A "step" is one pass of the whole hot path over the workload: one COARSE step = 2^depth fine steps of the
asynchronous schedule (every level sweep with its fused coalescence / explosion / boundary links), replayed
as a CUDA graph.  `value` = actual cell updates / s (MLUPS) with the state resident in HBM; `e2e` = the
same through the C-ABI calls with pinned HOST buffers (lbm_init_fields H2D + lbm_step + lbm_get_macroscopic
D2H inside the timed region, every step).  N > 1: independent replicas, one per rank (the path does not
shard: DESIGN.md "replicas only"), no data-path collective; value = sum over ranks / max time.

Workloads (synthetic, seeded, shaped like the paper's cases):
  cylinder  BASELINE configs[2]: D2Q9-RR, 6 levels, ~9.85 M cells (default: the multilevel headline)
  uniform   configs[0] scaled to 4096^2 (tree-stored uniform periodic D2Q9-BGK; the 80 %-of-HBM target)
  cylinder:mc<k> / cylinder:mf<k>  the same box with k levels merged from the coarsest / finest (the paper's Table 2 study)
  cavity    configs[1] as given (39 k cells, launch-latency-bound)    cavity8: the same x8
  cavity:uniform  the paper's uniform lid-driven cavity, L = 4096; with --addressing matrix the Eq. 14 point
  riemann   configs[3]: D2Q37 polynomial + g + sensor, 2048^2        riemann:numeq: the same box with the numerical equilibrium
  naca      configs[4]: D2Q21 numerical equilibrium + g + sensor, 7 levels, ~18 M cells
  sod:<Q>:<mesh>  Table 3 of the paper (numerical equilibrium + g + sensor, single precision there)
The default line also measures the other configs briefly (`also`), each with its own roofline block.
"""
import argparse
import csv
import hashlib
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2504_04465_b200 import workloads as W   # input generators only (no arithmetic of the method)

# Table 3a: A100-SXM4-80GB, single precision, MLUPS of Eq. 13 (all cells x finest iterations), L = 2^13
# (D2Q37 unif: 2^12).  Context for vs_baseline of `--workload sod:<lattice>:<mesh> --precision 32`.
PAPER_TABLE3 = {(13, "unif"): 1259.1, (13, "hori"): 1088.4, (13, "band"): 1244.8, (13, "sqr"): 1072.7,
                (21, "unif"): 618.5, (21, "hori"): 555.9, (21, "band"): 588.2, (21, "sqr"): 544.4,
                (37, "unif"): 286.9, (37, "hori"): 263.0, (37, "band"): 307.4, (37, "sqr"): 266.1}
REFERENCE_BUDGET_S = 180     # wall-clock cap of the timed region of --impl reference
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent
ADDRESSING = {"auto": 0, "list": 1, "bricks": 2, "matrix": 3}      # lbm_config.addressing (LBM_ADDR_*)
PIPELINE = {"auto": 0, "off": 1, "always": 2}                    # lbm_config.pipeline (LBM_PIPE_*): pipelined sweep of the wide models
# other workloads measured briefly into the default line's `also` (name[@f32|@f64][@list|@bricks])
DEFAULT_ALSO = "cavity,uniform,uniform@matrix,uniform@matrix@f32,cylinder@list,cylinder@f32,riemann,naca,sod:21:unif@f32"
KERNEL_SOURCES = ("lattice.cuh", "collide.cuh", "sweep.cuh", "sweep_pipe.cuh", "matrix.cuh")


def make_case(name, scale):
    if name == "cylinder":
        D = int(round(200 * scale))
        return W.cylinder(D=D), dict(workload="cylinder (BASELINE configs[2]): D2Q9-RR, D=%d, 64Dx64D, 6 levels" % D, steps=300)
    if name.startswith("cylinder:mc") or name.startswith("cylinder:mf"):
        # the paper's grid-hierarchy study (Sec. 7.5, Table 2, Fig. 24) at fixed finest resolution: levels merged from
        # the coarsest (mc<k>: the k+1 coarsest levels become one) or from the finest (mf<k>: the k+1 finest levels become
        # level 0); k = 5 is the uniform finest grid either way
        k = int(name[11:])
        D = int(round(200 * scale))
        coarse = name[10] == "c"
        radii = W.CYL_RADII_D[:5 - k] if coarse else W.CYL_RADII_D[k:]
        return W.cylinder(D=D, depth=5 - k, radii=radii), dict(
            workload="cylinder, %d levels merged from the %s (Sec. 7.5 study): D2Q9-RR, D=%d, %d levels" % (
                k, "coarsest" if coarse else "finest", D, 6 - k), steps=300 if k < 4 else 600)
    if name == "cylinder:sponge":     # configs[2] with the paper's far-field pressure relaxation (Eq. 10-11) switched on
        D = int(round(200 * scale))
        return W.cylinder(D=D, sponge_d=(24, 30, 0.1)), dict(
            workload="cylinder + sponge (Eq. 10-11: sigma 0 -> 0.1 between 24 D and 30 D): D2Q9-RR, D=%d, 6 levels" % D, steps=300)
    if name == "uniform":
        n = int(round(4096 * scale))
        return W.tgv(n), dict(workload="uniform periodic %dx%d tree-stored D2Q9-BGK Taylor-Green (configs[0] scaled)" % (n, n), steps=4000)
    if name in ("uniform:13", "uniform:21", "uniform:37"):      # the paper's tree-stored uniform D2Q13-RR / D2Q21-RR points (Fig. 42)
        n = int(round(4096 * scale))
        lat = int(name.split(":")[1])
        return W.tgv(n, lattice=lat, collision=W.RR), dict(
            workload="uniform periodic %dx%d tree-stored D2Q%d-RR Taylor-Green" % (n, n, lat), steps=2000 if lat == 13 else 1200 if lat == 21 else 600)
    if name == "cavity:uniform":      # the paper's uniform Cartesian benchmark (Fig. 22): lid-driven cavity, L = 4096
        n = int(round(4096 * scale))
        return W.cavity_uniform(n), dict(workload="cavity:uniform (P:520): D2Q9-RR lid-driven cavity on a uniform %dx%d box" % (n, n), steps=4000)
    if name == "cavity":
        return W.cavity(scale), dict(workload="cavity (BASELINE configs[1]): D2Q9-RR, 2 levels, coarse %d^2" % int(128 * scale), steps=100000)
    if name == "cavity8":
        return W.cavity(8 * scale), dict(workload="cavity x8: D2Q9-RR, 2 levels, coarse %d^2" % int(1024 * scale), steps=10000)
    if name == "riemann":
        n = int(round(2048 * scale))
        return W.riemann(n=n), dict(workload="riemann (BASELINE configs[3]): D2Q37 polynomial+g+sensor, %d^2, Neumann box" % n, steps=200)
    if name == "riemann:numeq":       # configs[3]'s box with the model the paper runs on D2Q37: stable for the 2000 steps
        n = int(round(2048 * scale))
        return W.riemann(n=n, collision=W.NUMEQ), dict(
            workload="riemann:numeq (BASELINE configs[3] box, 2000 steps): D2Q37 numerical eq.+g+sensor, %d^2, Neumann box" % n, steps=2000)
    if name == "naca":
        c = int(round(1024 * scale))
        return W.naca(chord=c), dict(workload="naca (BASELINE configs[4]): D2Q21 numerical eq.+g+sensor, chord %d, 7 levels" % c, steps=8, also_steps=2)
    if name.startswith("sod"):
        # sod[:lattice[:mesh]], e.g. sod:21:unif -- the paper's only absolute GPU figures (Table 3a)
        parts = name.split(":")
        lat = int(parts[1]) if len(parts) > 1 else 21
        mesh = parts[2] if len(parts) > 2 else "unif"
        L = int(round((4096 if (lat == 37 and mesh == "unif") else 8192) * scale))
        return W.sod(L=L, lattice=lat, mesh=mesh), dict(
            workload="sod shock tube (Table 3, P:656): D2Q%d numerical eq.+g+sensor, mesh %s, L=%d, periodic box" % (lat, mesh, L),
            steps=100, paper_mlups=PAPER_TABLE3.get((lat, mesh)))
    raise SystemExit("unknown workload %r" % name)


def label_for(info, addressing):
    """The workload string of a line; the uniform boxes say which storage they ran in."""
    w = info["workload"]
    if addressing == "matrix":
        w = w.replace("tree-stored", "matrix-like").replace("on a uniform", "on a matrix-like uniform") + " [Cartesian index, AA pattern, one population copy]"
    return w


def npop_of(case):
    return case.lattice * (2 if case.ddf else 1) + (8 if case.collision == W.NUMEQ else 0)


def algorithmic_bytes_per_update(case, precision):
    """Two-buffer pull update with an int32 list and a type byte:
    2*npop*s + (Q-1)*4 + 4 per cell update."""
    return 2 * npop_of(case) * (precision // 8) + (case.lattice - 1) * 4 + 4


def moved_bytes_per_update(g, case, precision):
    """Bytes this implementation has to move per cell update, weighted over the levels by their share of the updates:
    a cell of a regular brick needs its 2*npop reals and 36 B of tile bases per 64 cells; any
    other cell the list row and the type byte on top, plus its entry of the irregular-cell list on levels that have bricks."""
    Q = case.lattice
    npop = npop_of(case)
    s = precision // 8
    if "matrix" in g.kernel_name():        # Cartesian index, AA pattern: the populations once in, once out (Eq. 14 without its 8 B)
        return float(2 * npop * s)
    bricks = "bricks" in g.kernel_name()
    tot = upd = 0.0
    for l in range(g.depth + 1):
        nb = 64 * int(g.info.n_bricks[l]) if bricks and g.n[l] >= int(g.info.brick_min_level_cells) else 0
        k = 1 << (g.depth - l)
        tot += k * (nb * (2 * npop * s + 36.0 / 64) + (g.n[l] - nb) * (2 * npop * s + (Q - 1) * 4 + 1 + (4 if nb else 0)))
        upd += k * g.n[l]
    return tot / upd


def fine_equivalent_cells(case):
    m = case.mesh
    n = m.nx_coarse * m.ny_coarse * 4 ** m.depth
    for l, s in enumerate(m.solid):
        n -= len(s) * 4 ** l
    return n


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return {"hbm_gbs": FALLBACK_HBM_GBS}, "fallback (B200_PROFILING.md)"


def kernel_source_hash():
    """Hash of the kernel sources the committed ncu counters (profiles/traffic.csv) were taken with: a counter row whose
    hash differs from the current sources is reported as stale instead of silently describing another kernel."""
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2504_04465_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def committed_counters(key):
    """Row `key` of profiles/traffic.csv (ncu counters of the dominant kernel, see profiles/traffic.md) or {}."""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tp):
        return {}
    try:
        for r in csv.DictReader(open(tp)):
            if r["key"] == key:
                return {k: (v if k in ("key", "source", "kernel_hash") else float(v)) for k, v in r.items() if v not in ("", None)}
    except Exception:
        pass
    return {}


def roofline_blocks(case, precision, g, key, scale, upd_per_s, peak, peak_src, fma_peak):
    """HBM roofline in the bytes this implementation must move (the list-addressed figure of SURVEY 8(d) beside it) and,
    for the compute-heavy models, the ALU roofline against the FMA peak measured in this run."""
    bpu = algorithmic_bytes_per_update(case, precision)
    mbpu = moved_bytes_per_update(g, case, precision)
    c = committed_counters(key)
    stale = bool(c) and c.get("kernel_hash") != kernel_source_hash()
    same_launch = bool(c) and scale == 1.0 and int(c.get("cells_per_launch", -1)) == int(g.n[0])
    traffic = int(c["bytes_per_launch"]) if same_launch and "bytes_per_launch" in c and not stale else None
    hbm = {"bound": "hbm", "achieved": upd_per_s * mbpu / 1e9, "peak": peak, "unit": "GB/s", "frac": upd_per_s * mbpu / 1e9 / peak,
           "traffic": traffic, "traffic_source": c.get("source") if traffic else None,
           "bytes_per_update": mbpu, "bytes_per_launch": int(g.n[0] * mbpu), "peak_source": peak_src,
           "achieved_is": "bytes this implementation must move (brick cells: populations + 36 B per 64 cells; list cells: populations + list "
                          "row + type byte) of all level sweeps of the timed region / its CUDA-event time (every launch is this kernel)",
           "kernel": "%s, finest level (%d cells per launch)" % (g.kernel_name(), g.n[0]),
           "list_addressed": {"bytes_per_update": bpu, "achieved": upd_per_s * bpu / 1e9, "frac": upd_per_s * bpu / 1e9 / peak,
                              "what": "the same time charged with SURVEY 8(d)'s list-addressed algorithmic bytes (2 npop s + 4 (Q-1) + 4); "
                                      "exceeds 1 where bricks remove the list traffic"},
           "frac_of_nominal_8TBs": upd_per_s * mbpu / 1e9 / 8000.0}
    hbm["frac_plausible"] = hbm["frac"] <= 1.05
    alu = None
    if fma_peak and "flop_per_update" in c:
        tf = upd_per_s * c["flop_per_update"] / 1e12
        alu = {"bound": "alu", "achieved": tf, "peak": fma_peak, "unit": "TFLOP/s", "frac": tf / fma_peak, "traffic": traffic,
               "peak_source": "lbm_measure_fma_peak(%d) measured in this run" % precision,
               "flop_per_update": c["flop_per_update"], "flop_source": c.get("source"),
               "flop_is": "2 x FMA + ADD + MUL thread instructions of the finest level's launch / its cells (ncu smsp__sass_thread_inst_executed_op_*)",
               "flop_counters_stale": stale or not same_launch, "pipe_pct_ncu": c.get("pipe_pct"),
               "newton_steps_per_solve_at_capture": c.get("newton_steps_per_solve")}
    return hbm, alu


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out = self.p.communicate(timeout=5)[0]
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for k, nme in enumerate(names):
                if c[3 + k].lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def workload_config(info, precision, n_levels, cells, cells_per_level, updates_per_step, world):
    """The keys that name the workload: the same in the CUDA arm and in the reference arm."""
    return dict(workload=info["workload"], precision=precision, cells=int(cells), levels=int(n_levels),
                cells_per_level=[int(x) for x in cells_per_level], updates_per_step=int(updates_per_step),
                step="one coarse step = %d fine steps" % (1 << (n_levels - 1)), parallelism="replicas x%d" % world)


# ----------------------------------------------------------------------------- oracle legs (CPU)
def oracle_grid(case):
    from oracle import oracle as O      # test infrastructure: only these two legs of bench.py may load it
    o = O.OracleGrid(O.make_config(**case.model_kwargs()), case.mesh.split, case.mesh.solid)
    cells = [o.cells(l)[:2] for l in range(o.depth + 1)]
    assert o.init_fields(*W.eval_fields(case, cells)) == 0
    return o


def oracle_rate(o, budget_s, min_fine_steps=1):
    """Times the oracle, single-threaded, fine step by fine step until `budget_s` is spent; MLUPS (actual)."""
    u0 = o.cell_updates()
    t0 = time.perf_counter()
    n = 0
    while True:
        o.step_fine(1)
        n += 1
        dt = time.perf_counter() - t0
        if n >= min_fine_steps and dt >= budget_s:
            break
    return (o.cell_updates() - u0) / dt / 1e6, n, o.cell_updates() - u0, dt


def run_reference(args, case, info):
    """--impl reference: the oracle as it stands on the host cores; each step = one fine step of the schedule on
    the full grid (a bounded sample of the coarse step the CUDA arm times)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    o = oracle_grid(case)
    for _ in range(args.warmup):
        o.step_fine(1)
    u0 = o.cell_updates()
    t0 = time.perf_counter()
    done = 0
    for _ in range(args.steps):
        o.step_fine(1)
        done += 1
        if time.perf_counter() - t0 > REFERENCE_BUDGET_S:      # keep the whole run within a few minutes whatever K is
            break
    dt = time.perf_counter() - t0
    upd = o.cell_updates() - u0
    v = upd / dt / 1e6
    sample = "%d fine steps of the schedule on the full grid (%d cell updates)" % (done, upd)
    if done < args.steps:
        sample += "; stopped at the %d s budget of the reference arm (%d steps asked)" % (REFERENCE_BUDGET_S, args.steps)
        args.steps = done
    upd_coarse = sum(o.n[l] << (o.depth - l) for l in range(o.depth + 1))
    line = {"impl": "reference", "metric": "MLUPS (actual cell updates per second)", "value": v, "unit": "MLUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(info, 64, o.depth + 1, o.ntot, o.n, upd_coarse, max(args.gpus, 1)),
            "cpu_baseline": {"value": v, "unit": "MLUPS", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- N > 1: replicas, max-over-ranks timing
def reduce_max_over_ranks(values, world, device="cpu"):
    """The slowest rank defines the job time (contract: time = max over ranks).  Works on any backend (nccl on the
    GPU box, gloo in tests/test_bench_host.py)."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_mlups(updates_per_rank_step, steps, world, ms):
    """Whole-job throughput of `world` independent replicas (weak scaling): all ranks' updates / the slowest rank's time."""
    return updates_per_rank_step * steps * world / (ms * 1e-3) / 1e6


_FMA_PEAK = {}


def fma_peak_of(lbm, precision):
    """FMA peak of the plain fp64 / fp32 pipe, measured once per run (1 s) -- denominator of the ALU rooflines."""
    if precision not in _FMA_PEAK:
        _FMA_PEAK[precision] = lbm.measure_fma_peak(precision, 1.0)[0]
    return _FMA_PEAK[precision]


def wants_alu(case):
    return case.collision == W.NUMEQ or (case.lattice == 37 and case.ddf)


def newton_block(g, it0, ns0, updates):
    it1, ns1 = g.newton_iterations()
    if ns1 == ns0:
        return None
    return {"steps_per_solve": (it1 - it0) / (ns1 - ns0), "solves_per_update": (ns1 - ns0) / max(updates, 1),
            "what": "Newton steps (unconditional polish step included) per equilibrium solve in the timed region, counted by the kernels "
                    "(lbm_newton_iterations); the paper: about one iteration on smooth fields with a warm start (P:124)"}


def parse_also(entry, precision):
    parts = entry.split("@")
    opts = dict(precision=precision, addressing="auto", pipeline="auto", no_prefetch=0)
    for o in parts[1:]:
        if o in ("f32", "f64"):
            opts["precision"] = int(o[1:])
        elif o in ADDRESSING:
            opts["addressing"] = o
        elif o == "nopipe":
            opts["pipeline"] = "off"
        elif o == "noprefetch":
            opts["no_prefetch"] = 1
        else:
            raise SystemExit("unknown option %r in --also entry %r" % (o, entry))
    return parts[0], opts


def also_measure(lbm, entry, precision, dev, peak, peak_src):
    """Device-resident throughput of another workload with its own step count, for the `also` entries of the default
    line (same timing rules: 3 warm-up steps, CUDA events on the bound stream around the replayed graphs)."""
    name, opts = parse_also(entry, precision)
    prec = opts["precision"]
    case, info = make_case(name, 1.0)
    steps = info.get("also_steps", info["steps"])
    t0 = time.perf_counter()
    g = lbm.Grid.from_case(case, precision=prec, addressing=ADDRESSING[opts["addressing"]], pipeline=PIPELINE[opts["pipeline"]],
                           no_prefetch=opts["no_prefetch"])
    g.bind(dev)
    cells = [g.cells(l)[:2] for l in range(g.depth + 1)]
    rc = g.init_fields(*W.eval_fields(case, cells))
    assert rc == 0, rc
    t_build = time.perf_counter() - t0
    g.step(3)
    assert g.sync() == 0
    it0, ns0 = g.newton_iterations()
    g.step(steps)
    ms = g.last_step_ms()
    status = g.sync()
    assert status == 0, "device status %d after the timed region of %s" % (status, entry)
    upd = int(g.info.updates_per_coarse_step)
    v = upd * steps / (ms * 1e-3) / 1e6
    key = "%s_f%d" % (name, prec) + ("" if opts["addressing"] == "auto" else "@" + opts["addressing"]) + ("" if opts["pipeline"] == "auto" else "@nopipe")
    hbm, alu = roofline_blocks(case, prec, g, key, 1.0, v * 1e6, peak, peak_src, fma_peak_of(lbm, prec) if wants_alu(case) else None)
    out = {"workload": label_for(info, opts["addressing"]), "entry": entry, "dtype": "f%d" % prec, "value": v, "unit": "MLUPS", "steps": steps,
           "ms_per_step": ms / steps, "cells": g.ntot, "levels": g.depth + 1, "gpu_launches": int(g.info.launches_per_coarse_step) * steps,
           "kernel": g.kernel_name(), "build_s": t_build, "arena_bytes": int(g.info.arena_bytes),
           "mlups_paper_eq13": g.ntot * (1 << g.depth) * steps / (ms * 1e-3) / 1e6}
    if case.collision == W.NUMEQ and alu is not None:
        out["roofline"], out["roofline_hbm"] = alu, hbm
    else:
        out["roofline"] = hbm
        if alu is not None:
            out["roofline_alu"] = alu
    nb = newton_block(g, it0, ns0, upd * steps)
    if nb:
        out["newton"] = nb
    if info.get("paper_mlups") and prec == 32:
        out["vs_paper_table3a_a100"] = out["mlups_paper_eq13"] / info["paper_mlups"]
    g.close()
    return out


# ----------------------------------------------------------------------------- CUDA arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cylinder")
    ap.add_argument("--precision", type=int, default=64, choices=[32, 64])
    ap.add_argument("--addressing", default="auto", choices=sorted(ADDRESSING), help="lbm_config.addressing: auto = regular bricks on "
                    "large levels, list = the list-addressed kernel on every level, bricks = bricks on every level")
    ap.add_argument("--pipeline", default="auto", choices=sorted(PIPELINE), help="lbm_config.pipeline: auto = software-pipelined sweep of "
                    "the wide models on large levels, off = one cell per thread everywhere")
    ap.add_argument("--concurrent-levels", type=int, default=0, choices=[0, 1], help="lbm_config.concurrent_levels (graph branches for levels >= 2, P:221)")
    ap.add_argument("--no-prefetch", type=int, default=0, choices=[0, 1], help="lbm_config.no_prefetch (next-wave L2 prefetch of the wide models)")
    ap.add_argument("--scale", type=float, default=1.0, help="linear scale of the workload (1 = BASELINE size)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--cpu-baseline-seconds", type=float, default=15.0, help="0 disables the cpu_baseline leg")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--remesh", action="store_true", help="cylinder only: after the timed region, time lbm_transfer onto a tree with "
                    "other refinement radii (mesh adaptation, Sec. 8.1 of the paper) into the line's `remesh` block")
    ap.add_argument("--also", default=None, help="comma list of other workloads measured briefly into the line's `also` "
                    "(default for the default workload: %s; 'none' disables)" % DEFAULT_ALSO)
    args = ap.parse_args()
    case, info = make_case(args.workload, args.scale)
    if args.steps is None:
        args.steps = info["steps"] if args.impl == "cuda" else 20
    if args.impl == "reference":
        return run_reference(args, case, info)

    import torch
    import torch.distributed as dist
    from paper_2504_04465_b200 import lbm     # raises if the CUDA library is not built: no fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    t_build = time.perf_counter()
    g = lbm.Grid.from_case(case, precision=args.precision, addressing=ADDRESSING[args.addressing], pipeline=PIPELINE[args.pipeline],
                           no_prefetch=args.no_prefetch, concurrent_levels=args.concurrent_levels)
    g.bind(dev)
    ntot = g.ntot
    pin = lambda: torch.empty(ntot, dtype=torch.float64).pin_memory().numpy()
    h_in = [pin() for _ in range(4)]
    h_out = [pin() for _ in range(4)]
    cells = [g.cells(l)[:2] for l in range(g.depth + 1)]
    for dst, src in zip(h_in, W.eval_fields(case, cells)):
        dst[:] = src
    rc = g.init_fields(*h_in)
    assert rc == 0, "lbm_init_fields status %d" % rc
    t_build = time.perf_counter() - t_build

    upd = int(g.info.updates_per_coarse_step)
    launches = int(g.info.launches_per_coarse_step)
    # ---- device-resident throughput: W warm-up steps, then exactly K steps between CUDA events on the bound stream
    g.step(args.warmup)
    assert g.sync() == 0
    # burst figure (GPU still cool, ~30 ms region: comparable with MEASURED_PEAKS' best-of-10 copy); the headline
    # `value` below is the figure over the full K steps, which for long regions on these 1 kW parts runs under sw_power_cap
    g.step(3)
    est = max(g.last_step_ms() / 3, 1e-4)
    kb = int(min(max(3, 30.0 / est), max(3, args.steps)))
    g.step(kb)
    burst_ms = g.last_step_ms() / kb
    assert g.sync() == 0
    it0, ns0 = g.newton_iterations()
    barrier()
    clk = ClockSampler(local)
    t0 = time.perf_counter()
    g.step(args.steps)
    ms = g.last_step_ms()            # events recorded on the grid's stream around the K graph replays; synchronises
    status = g.sync()
    barrier()
    wall = time.perf_counter() - t0
    clocks = clk.stop()
    assert status == 0, "device status %d after the timed region" % status
    newton = newton_block(g, it0, ns0, upd * args.steps)

    # ---- end to end through the C ABI with pinned host buffers, every step: H2D fields -> step -> D2H macroscopic
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_ms = 0.0
    with torch.cuda.stream(g.stream):
        for it in range(args.e2e_steps + 1 if args.e2e_steps > 0 else 0):      # --e2e-steps 0: leg skipped (profiling runs)
            barrier()
            ev0.record(g.stream)
            rc = g.init_fields(*h_in)
            g.step(1)
            g.macroscopic(out=h_out)
            ev1.record(g.stream)
            ev1.synchronize()
            assert rc == 0
            if it > 0:               # first pass is the warm-up
                e2e_ms += ev0.elapsed_time(ev1)
    e2e_ms /= max(args.e2e_steps, 1)

    ms, e2e_ms = reduce_max_over_ranks([ms, e2e_ms], world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    K = args.steps
    mlups = aggregate_mlups(upd, K, world, ms)
    peaks, peak_src = measured_peaks()
    peak = float(peaks.get("hbm_gbs", FALLBACK_HBM_GBS))
    key = "%s_f%d" % (args.workload, args.precision) + ("" if args.addressing == "auto" else "@" + args.addressing) + ("" if args.pipeline == "auto" else "@nopipe")
    rank_upd_per_s = upd * K / (ms * 1e-3)               # this rank's kernel: every launch of the region is the sweep kernel
    hbm, alu = roofline_blocks(case, args.precision, g, key, args.scale, rank_upd_per_s, peak, peak_src,
                               fma_peak_of(lbm, args.precision) if wants_alu(case) else None)
    n_all = ntot
    depth = g.depth
    # vs_baseline only where BASELINE.md holds the paper's number for this exact metric and workload: Table 3a, Eq. 13
    # MLUPS, single precision, full size (another machine's figure: context, not the target)
    vs_baseline = None
    if info.get("paper_mlups") and args.precision == 32 and args.scale == 1.0 and world == 1:
        vs_baseline = n_all * (1 << depth) * K / (ms * 1e-3) / 1e6 / info["paper_mlups"]
    config = workload_config(dict(info, workload=label_for(info, args.addressing)), args.precision, depth + 1, n_all, g.n, upd, world)
    config["l2"] = ("inputs larger than L2 (state %.0f MB)" % (g.info.arena_bytes / 1e6) if g.info.arena_bytes > 4 * 126e6
                    else "working set %.0f MB fits L2: launch-latency-bound case, no flush" % (g.info.arena_bytes / 1e6))
    line = {
        "metric": "MLUPS (actual cell updates per second)", "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": K,
        "warmup": args.warmup, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": vs_baseline,
        "dtype": "f%d" % args.precision, "data": "synthetic", "config": config,
        "kernel": {"name": g.kernel_name(), "addressing": args.addressing, "pipeline": args.pipeline, "arena_bytes": int(g.info.arena_bytes),
                   "brick_cell_share": [round(64 * int(g.info.n_bricks[l]) / max(g.n[l], 1), 4) if g.n[l] >= int(g.info.brick_min_level_cells) else 0.0
                                        for l in range(depth + 1)]},
        "mlups": {"actual": mlups, "paper_eq13": n_all * (1 << depth) * K * world / (ms * 1e-3) / 1e6,
                  "fine_equivalent": fine_equivalent_cells(case) * (1 << depth) * K * world / (ms * 1e-3) / 1e6},
        "roofline": hbm,
        "burst": {"steps": kb, "ms_per_step": burst_ms, "value": upd / (burst_ms * 1e-3) / 1e6, "unit": "MLUPS (this rank)",
                  "roofline_frac": upd * hbm["bytes_per_update"] / (burst_ms * 1e-3) / 1e9 / peak,
                  "what": "short region right after warm-up, before the power cap settles"},
        "e2e": None if e2e_ms <= 0 else {
            "value": upd * world / (e2e_ms * 1e-3) / 1e6, "unit": "MLUPS", "h2d_bytes_per_step": 4 * 8 * ntot,
            "d2h_bytes_per_step": 4 * 8 * ntot, "ms_per_step": e2e_ms,
            "what": "lbm_init_fields (pinned host rho,u,T) + lbm_step(1) + lbm_get_macroscopic (pinned host), every step"},
        "gpu_launches": launches * K,
        "clocks": clocks,
        "wall_s_timed_region": wall, "build_s": t_build,
    }
    if case.collision == W.NUMEQ and alu is not None:       # ALU-bound path: the HBM view stays beside it
        line["roofline"], line["roofline_hbm"] = alu, hbm
    elif alu is not None:
        line["roofline_alu"] = alu
    if newton:
        line["newton"] = newton
    if args.remesh and args.workload == "cylinder" and world == 1:
        # mesh adaptation: the same box with every refinement radius but the outermost moved by one diameter
        D = int(round(200 * args.scale))
        tc = time.perf_counter()
        eps = g.sensor()                 # the refinement criterion (Eq. 52 of the stored state), computed on the device
        tc = time.perf_counter() - tc
        t0 = time.perf_counter()
        case2 = W.cylinder(D=D, radii=tuple(r + (1.0 if k % 2 == 0 else -1.0) for k, r in enumerate(W.CYL_RADII_D[:-1])) + W.CYL_RADII_D[-1:])
        g2 = lbm.Grid.from_case(case2, precision=args.precision, addressing=ADDRESSING[args.addressing])
        g2.bind(dev)
        t1 = time.perf_counter()
        g2.transfer_from(g)
        assert g2.sync() == 0
        t2 = time.perf_counter()
        g2.step(2)
        assert g2.sync() == 0
        line["remesh"] = {"criterion_s": tc, "criterion_max": float(eps.max()), "new_tree_build_and_bind_s": t1 - t0, "transfer_s": t2 - t1, "cells_new": g2.ntot, "cells_old": ntot,
                          "what": "lbm_transfer (position keys uploaded, look-up + copy / explosion / coalescence per cell of the new tree on the device), then two "
                                  "coarse steps on the new tree ran to status 0; the paper: mesh adaptation on the CPU is the bottleneck (P:698)"}
        g2.close()
    also = args.also if args.also is not None else (DEFAULT_ALSO if args.workload == "cylinder" and args.scale == 1.0 and args.addressing == "auto" else "none")
    if also != "none" and world == 1:
        g.close()                # release the arena before building the next grid
        del h_in, h_out
        line["also"] = []
        for entry in [w for w in also.split(",") if w]:
            line["also"].append(also_measure(lbm, entry, args.precision, dev, peak, peak_src))
            torch.cuda.empty_cache()
    if args.cpu_baseline_seconds > 0 and world >= 1:
        o = oracle_grid(case)
        v, nf, nu, dt = oracle_rate(o, args.cpu_baseline_seconds)
        line["cpu_baseline"] = {"value": v, "unit": "MLUPS", "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
                                "sample": "%d fine steps of the schedule on the full grid (%d cell updates, %.1f s)" % (nf, nu, dt)}
    print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
