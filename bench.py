#!/usr/bin/env python
"""bench.py -- throughput of the DIMOS hot path (cell-list Verlet list + rebuild trigger + LJ/RF pair forces)
on synthetic constant-density water boxes (BASELINE.json metric: pair interactions/s and tau per force step).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--precision f32]

One "step" is one pass of the whole hot path on a synthetic ballistic trajectory:
the rebuild trigger is evaluated every step, the list is rebuilt when it fires
 and the nonbonded forces, energy and virial are evaluated every step.
`value` = in-cutoff pair interactions per second, whole job (all ranks), inputs resident in HBM.
`e2e` = the same protocol through dimos_step_host with pinned HOST buffers (H2D + D2H inside the timed region).
`--impl reference` times the CPU fp64 oracle (oracle/, as it stands) on the host cores on a bounded sample.
N > 1 (torchrun): independent replicas, one box per rank, no data-path collective ("scaling": "weak").
"""
from __future__ import annotations

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

from paper_2503_20541_b200 import workloads as wl  # noqa: E402

METRIC = "pair_interactions_per_s"
UNIT = "pair interactions/s"
# algorithmic FLOP model of the pair kernel: per listed pair
# (r < r_nl) the distance test, per in-cutoff pair additionally force + energy
FLOPS_PER_LISTED_PAIR = 9
FLOPS_PER_CUTOFF_PAIR = {"rf": 31, "ewald": 56}
# FP32 ALU peak derived from the guide's unit counts and clocks: 148 SMs x 128 FP32 lanes x 2 (FMA) x 1.965 GHz
FP32_LANES_PER_SM = 128
DT_PS = 0.001  # 1 fs ballistic drift per step (configs[1] recipe: Maxwell-Boltzmann 300 K, dt = 1 fs)
TEMPERATURE = 300.0
TRIANGLE_HALF_PERIOD = 25  # velocities reverse every 25 steps so the box stays near its seeded structure


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (3 = 900,000 atoms, headline)")
    ap.add_argument("--precision", default=None, help="f32 | mixed | f64 (default: first precision of the config)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-scan", action="store_true", help="skip the tau-versus-N scan over smaller boxes of the same recipe")
    return ap.parse_args()


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate_over_ranks(local_seconds: float, local_units: float, world: int, dist=None, device=None):
    """max-over-ranks time, sum-over-ranks units (weak scaling, independent replicas).  Works on gloo or nccl."""
    if world == 1 or dist is None:
        return local_seconds, local_units
    import torch

    t = torch.tensor([local_seconds], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def trajectory_offsets(step: int) -> float:
    """Signed number of dt the positions are displaced from the seeded box at `step` (triangle wave)."""
    p = TRIANGLE_HALF_PERIOD
    k = step % (2 * p)
    return float(k if k <= p else 2 * p - k)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md clocks line)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=self.fh, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, smax, reasons, power = [], [], set(), []
        for line in open(self.path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.path)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "power_w_max": float(max(power)), "samples": len(sm)}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def load_traffic(kernel: str, config_index: int):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture of the same workload
    (profiles/traffic.json, keyed "<kernel>@configs[<i>]"), or None."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        try:
            return json.load(open(path)).get(f"{kernel}@configs[{config_index}]")
        except Exception:
            return None
    return None


# ------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores, on a bounded sample
# ------------------------------------------------------------------------------------------------------
def oracle_box(spec, size: str):
    """The workload's own box ("config"), or a constant-density box of the same recipe 10x / 100x smaller."""
    if size == "config":
        return wl.make_water_box(spec.n_molecules, wl.box_edge_for(spec), wl.SEED_BASE + spec.index, spec)
    n_mol = {"tenth": max(spec.n_molecules // 10, 216), "hundredth": max(spec.n_molecules // 100, 216)}[size]
    return wl.make_scaled(n_mol, seed=wl.SEED_BASE + 50, r_cut=spec.r_cut, skin=spec.skin, method=spec.method)


def time_oracle_step(box, method: str):
    import oracle

    lj = oracle.lorentz_berthelot(box.sigma, box.epsilon)
    t0 = time.perf_counter()
    res = oracle.nonbonded(box.pos, box.charge, box.type, lj, box.box, box.spec.r_cut,
                           method=oracle.METHOD_RF if method == "rf" else oracle.METHOD_EWALD_REAL,
                           alpha=box.spec.alpha, excl_pairs=box.excl_pairs, algorithm="celllist")
    return time.perf_counter() - t0, res.n_pairs


def pick_oracle_box(spec, n_evals: int, budget_s: float):
    """Largest box of the workload's recipe whose n_evals oracle evaluations fit the time budget: the config itself when
    it does (the oracle's cost is linear in N: a probe on the 100x smaller box is scaled up)."""
    probe = oracle_box(spec, "hundredth")
    t_probe, _ = time_oracle_step(probe, spec.method)
    per_atom = t_probe / probe.n_atoms
    for size in ("config", "tenth"):
        n_atoms = 3 * spec.n_molecules if size == "config" else 3 * max(spec.n_molecules // 10, 216)
        if 1.5 * per_atom * n_atoms * n_evals <= budget_s:
            return oracle_box(spec, size), size
    return probe, "hundredth"


def sample_text(box, spec, size):
    what = "the workload's own box" if size == "config" else f"a box of the same recipe, {size} of the atoms (the full box would exceed the time budget)"
    return (f"one oracle cell-list force evaluation (fp64, C, OpenMP over all host cores) of {what}: {box.n_atoms} atoms, "
            f"r_cut={spec.r_cut}, method={spec.method}")


def cpu_baseline(spec, budget_s: float = 30.0) -> dict:
    import oracle

    box, size = pick_oracle_box(spec, 1, budget_s)
    t, n = time_oracle_step(box, spec.method)
    return {"value": n / t, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample_text(box, spec, size),
            "seconds": t, "same_config": size == "config", "n_atoms": int(box.n_atoms), "pairs_in_cutoff": int(n)}


def run_reference(args, spec, precision):
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle

    box, size = pick_oracle_box(spec, args.steps + args.warmup, 240.0)
    for _ in range(args.warmup):
        time_oracle_step(box, spec.method)
    t0 = time.perf_counter()
    pairs = 0
    for _ in range(args.steps):
        _, n = time_oracle_step(box, spec.method)
        pairs += n
    dt = time.perf_counter() - t0
    value = pairs / dt
    sample = "each step = " + sample_text(box, spec, size)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(spec, precision), "sample": sample, "same_config": size == "config"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def tau_vs_n(ctx, dimos, dev, spec, precision, timed, tau_force_main, tau_build_main, n_main, n_cut_main):
    """tau (s per force call) and pair interactions/s versus N on constant-density boxes of the same recipe
    (the shape of the paper's scaling study); the last row is the headline workload itself."""
    import torch

    rows = []
    for n_mol in (216, 3000, 30000, 100000):
        if 3 * n_mol >= n_main:
            continue
        b = wl.make_scaled(n_mol, seed=wl.SEED_BASE + 200 + n_mol % 97, r_cut=spec.r_cut, skin=spec.skin, method=spec.method)
        if spec.r_cut > 0.5 * float(min(b.box)):
            continue  # the minimum-image requirement r_c <= L/2 (reading C-3) rules this size out
        pos = torch.from_numpy(b.pos.astype(np.float32)).to(dev)
        charge = torch.from_numpy(b.charge.astype(np.float32)).to(dev)
        typ = torch.from_numpy(b.type).to(dev)
        excl = torch.from_numpy(b.excl_pairs).to(dev)
        lj = dimos.lj_table_from_types(b.sigma, b.epsilon).to(dev)
        kw = dict(method=spec.method, eps_rf=spec.eps_rf, alpha=spec.alpha)
        nl = dimos.dimos_nl_build(ctx, pos, b.box, spec.r_cut, spec.skin, excl)
        n_cut = ctx.nl_count_within(nl, spec.r_cut)
        F = torch.empty_like(pos)
        E = torch.empty(4, dtype=torch.float64, device=dev)
        W = torch.empty(3, 3, dtype=torch.float64, device=dev)
        for _ in range(3):
            dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw)
        t_f = timed(lambda: dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw), reps=20)
        # a step that keeps the list (trigger with the flag left on the device -> conditional force call), launched call by
        # call and replayed as one CUDA graph: small boxes are launch-bound (tests/test_gpu_graph.py checks the replayed results)
        flag = torch.zeros(1, dtype=torch.int32, device=dev)

        def step_body():
            dimos.dimos_nl_needs_rebuild_static(ctx, pos, nl.pos_at_build, spec.skin, flag)
            dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, skip_flag=flag, **kw)

        t_eager = t_graph = None
        try:
            step_body()
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                step_body()
            t_eager = timed(step_body, reps=50)
            t_graph = timed(graph.replay, reps=50)
            del graph
        except Exception as exc:  # the measurement is context: never let it take the bench line down
            print(f"tau_vs_n: graph capture failed at {b.n_atoms} atoms: {exc}", file=sys.stderr)
        # the same for one whole rigid-water MD step that keeps the list (the three calls of md_step_tau, the last two conditional
        # on the fused trigger's flag); started at rest with dt = 1e-4 fs so that the ~150 timed steps of the unrelaxed box (forces up
        # to 1e5 kJ mol^-1 nm^-1) stay far below the trigger: the kernels' work does not depend on dt
        t_md_eager = t_md_graph = None
        try:
            water = torch.arange(b.n_atoms, dtype=torch.int32, device=dev).reshape(-1, 3)
            m_O, m_H = float(b.mass[0]), float(b.mass[1])
            d_oh = wl.R_OH
            d_hh = 2.0 * wl.R_OH * float(np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0))
            x, v = pos.clone(), torch.zeros_like(pos)
            nl_md = dimos.dimos_nl_build(ctx, x, b.box, spec.r_cut, spec.skin, excl)
            dimos.dimos_nonbonded(ctx, nl_md, x, charge, typ, lj, F=F, E=E, virial=W, **kw)

            def md_body():
                fl = dimos.dimos_water_kick_drift_settle(ctx, x, v, F, water, m_O, m_H, d_oh, d_hh, 1e-7, pos_at_build=nl_md.pos_at_build,
                                                         skin=spec.skin, sync=False)
                dimos.dimos_nonbonded(ctx, nl_md, x, charge, typ, lj, F=F, E=E, virial=W, skip_flag=fl, **kw)
                dimos.dimos_water_kick_settle_velocities(ctx, x, v, F, water, m_O, m_H, 1e-7, skip_flag=fl)
                return fl

            fl = md_body()
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                md_body()
            t_e, t_g = timed(md_body, reps=50), timed(graph.replay, reps=50)
            assert int(fl.item()) == 0 and bool(torch.isfinite(x).all()), "the timed MD steps crossed the rebuild trigger"
            t_md_eager, t_md_graph = t_e, t_g
            del graph
            ctx.lib.dimos_nl_destroy(ctx.handle, nl_md.handle)
        except Exception as exc:
            print(f"tau_vs_n: MD-step graph measurement failed at {b.n_atoms} atoms: {exc}", file=sys.stderr)
        t_b = timed(lambda: dimos.dimos_nl_build(ctx, pos, b.box, spec.r_cut, spec.skin, excl, nl=nl), reps=5)
        rows.append({"n_atoms": int(b.n_atoms), "tau_force_s": t_f, "tau_build_s": t_b, "pairs_in_cutoff": int(n_cut),
                     "pairs_per_s_force_only": n_cut / t_f, "tau_step_eager_s": t_eager, "tau_step_cuda_graph_s": t_graph,
                     "tau_md_step_eager_s": t_md_eager, "tau_md_step_cuda_graph_s": t_md_graph})
    rows.append({"n_atoms": int(n_main), "tau_force_s": tau_force_main, "tau_build_s": tau_build_main,
                 "pairs_in_cutoff": int(n_cut_main), "pairs_per_s_force_only": n_cut_main / tau_force_main})
    return rows


class DeviceFlag:
    """Reads the rebuild flag the trigger left on the device WITHOUT stalling the GPU: an asynchronous copy to a pinned word
    and an event recorded right behind the trigger kernel.  The force call (dimos_nb_params.skip_flag = the same device word)
    is enqueued before the host waits for that event, so the GPU computes forces while the host reads the flag; when the flag
    is set the force kernels return at once and the host rebuilds the list and repeats the force call."""

    def __init__(self, torch):
        self.host = torch.zeros(1, dtype=torch.int32).pin_memory()
        self.event = torch.cuda.Event()

    def fetch(self, flag):
        self.host.copy_(flag, non_blocking=True)
        self.event.record()

    def fired(self) -> bool:
        self.event.synchronize()
        return bool(self.host[0])


def md_step_tau(ctx, dimos, torch, box, spec, pos0, vel_np, charge, typ, excl, lj, kw, steps=60, warmup=10, dt=0.0005):
    """tau of one rigid-water MD step made of library calls only (the quantity the paper's Fig. 1 plots):
    dimos_water_kick_drift_settle (velocity-Verlet steps 1-3 of PAPER.md:281-292 + the rebuild trigger) -> dimos_nl_build when
    it fired -> dimos_nonbonded (step 4) -> dimos_water_kick_settle_velocities (steps 5-6).  NVE from Maxwell-Boltzmann 300 K
    velocities on the seeded (unrelaxed) box, dt = 0.5 fs (the time step of the paper's water-box benchmark)."""
    dev = pos0.device
    n = pos0.shape[0]
    water = torch.arange(n, dtype=torch.int32, device=dev).reshape(-1, 3)
    m_O, m_H = float(box.mass[0]), float(box.mass[1])
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * float(np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0))
    pos = pos0.clone()
    vel = torch.from_numpy(vel_np.astype(np.float64 if pos0.dtype == torch.float64 else np.float32)).to(dev)
    dimos.dimos_settle_velocities(ctx, pos, vel, water, m_O, m_H)
    nl = dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl)
    F = torch.empty_like(pos)
    E = torch.empty(4, dtype=torch.float64, device=dev)
    W = torch.empty(3, 3, dtype=torch.float64, device=dev)
    dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw)
    rebuilds = 0

    reader = DeviceFlag(torch)

    def one():
        nonlocal rebuilds
        flag = dimos.dimos_water_kick_drift_settle(ctx, pos, vel, F, water, m_O, m_H, d_oh, d_hh, dt, pos_at_build=nl.pos_at_build,
                                                   skin=spec.skin, sync=False)
        reader.fetch(flag)
        dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, skip_flag=flag, **kw)
        if reader.fired():
            dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl, nl=nl)
            dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw)
            rebuilds += 1
        dimos.dimos_water_kick_settle_velocities(ctx, pos, vel, F, water, m_O, m_H, dt)

    for _ in range(warmup):
        one()
    rebuilds = 0
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(steps):
        one()
    b.record()
    torch.cuda.synchronize()
    assert bool(torch.isfinite(E).all()) and bool(torch.isfinite(pos).all()), "non-finite state in the MD-step timing"
    return {"tau_s": a.elapsed_time(b) * 1e-3 / steps, "steps": steps, "rebuilds": rebuilds, "dt_fs": 1e3 * dt,
            "what": "rigid-water velocity-Verlet step: water_kick_drift_settle -> (nl_build) -> nonbonded -> water_kick_settle_velocities"}


def workload_name(spec, precision):
    return (f"configs[{spec.index}] {spec.name}: {3 * spec.n_molecules} atoms, density {wl.DENSITY} molecules/nm^3, "
            f"r_cut={spec.r_cut} nm, skin={spec.skin} nm, LJ + {'reaction field' if spec.method == 'rf' else 'Ewald real space'}, {precision}")


# ------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------
def run_ours(args, spec, precision):
    import torch

    from paper_2503_20541_b200 import binding as dimos

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    real = torch.float64 if precision == "f64" else torch.float32
    np_real = np.float64 if precision == "f64" else np.float32

    # one independent box per rank (weak scaling: replicas of the same recipe, different seeds)
    box = wl.make_water_box(spec.n_molecules, wl.box_edge_for(spec), wl.SEED_BASE + spec.index + 1000 * rank, spec)
    n = box.n_atoms
    vel = wl.maxwell_boltzmann_velocities(box.mass, TEMPERATURE, wl.SEED_BASE + 7 + rank)
    lj_host = dimos.lj_table_from_types(box.sigma, box.epsilon)
    pos0 = torch.from_numpy(box.pos.astype(np_real)).to(dev)
    dstep = torch.from_numpy((vel * DT_PS).astype(np_real)).to(dev)
    charge = torch.from_numpy(box.charge.astype(np_real)).to(dev)
    typ = torch.from_numpy(box.type).to(dev)
    excl = torch.from_numpy(box.excl_pairs).to(dev)
    lj = lj_host.to(dev)
    pos = pos0.clone()
    F = torch.empty_like(pos)
    E = torch.empty(4, dtype=torch.float64, device=dev)
    W = torch.empty(3, 3, dtype=torch.float64, device=dev)

    ctx = dimos.Context(local_rank, precision)
    kw = dict(method=spec.method, eps_rf=spec.eps_rf, alpha=spec.alpha)
    nl = dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl)
    n_cut = ctx.nl_count_within(nl, spec.r_cut)
    n_listed = ctx.nl_count_within(nl, spec.r_cut + spec.skin)
    # one force call and one rebuild before anything is timed: the builder files its rows by the LJ-activity flags of the
    # last force call, which the very first list of a context cannot have
    dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw)
    dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl, nl=nl)
    stats = nl.stats()
    state = {"step": 0, "rebuilds": 0}

    reader = DeviceFlag(torch)

    def step():
        # harness: ballistic drift (one fused axpy); library: trigger (flag stays on the device), forces conditional on the
        # flag, enqueued before the host has read it; when it fired: rebuild, forces again
        torch.add(pos0, dstep, alpha=trajectory_offsets(state["step"]), out=pos)
        flag = dimos.dimos_nl_needs_rebuild(ctx, pos, nl.pos_at_build, spec.skin, sync=False)
        reader.fetch(flag)
        dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, skip_flag=flag, **kw)
        if reader.fired():
            dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl, nl=nl)
            dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw)
            state["rebuilds"] += 1
        state["step"] += 1

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ctx.profile_enable(True)
    launches0 = ctx.launch_count()
    state["rebuilds"] = 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    seconds = e0.elapsed_time(e1) * 1e-3
    launches = ctx.launch_count() - launches0
    pair_ms, pair_n = ctx.profile_read()
    ctx.profile_enable(False)
    clocks = sampler.stop() if rank == 0 else None
    rebuilds = state["rebuilds"]
    assert bool(torch.isfinite(E).all()), "non-finite energy in the timed region"
    # the forces the timed loop left behind are those of its last step's positions: a fresh, unconditional evaluation on a
    # list rebuilt at these positions must reproduce them (to the summation order of the reductions)
    F_loop, E_loop = F.clone(), E.clone()
    nl_chk = dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl)
    F_chk, E_chk, _ = dimos.dimos_nonbonded(ctx, nl_chk, pos, charge, typ, lj, **kw)
    torch.cuda.synchronize()
    f_rms = float(F_chk.double().pow(2).sum(1).mean().sqrt())
    last_step_check = {"max_dF_over_rms": float((F_loop.double() - F_chk.double()).pow(2).sum(1).sqrt().max()) / f_rms,
                       "dE_over_E": abs(float(E_loop[0] - E_chk[0])) / max(abs(float(E_chk[0])), 1e-300)}
    tol_f, tol_e = (1e-9, 1e-10) if precision == "f64" else (2e-4, 1e-5)
    assert last_step_check["max_dF_over_rms"] < tol_f and last_step_check["dE_over_E"] < tol_e, last_step_check
    ctx.lib.dimos_nl_destroy(ctx.handle, nl_chk.handle)
    del F_chk, E_chk, nl_chk

    # separate timings of the three calls (tau_force, tau_build, tau_check), list valid, median of 20
    def timed(fn, reps=20):
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b) * 1e-3)
        return float(np.median(ts))

    pos.copy_(pos0)
    dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl, nl=nl)
    tau_force = timed(lambda: dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F, E=E, virial=W, **kw))
    tau_check = timed(lambda: dimos.dimos_nl_needs_rebuild(ctx, pos, nl.pos_at_build, spec.skin, sync=False))
    tau_build = timed(lambda: dimos.dimos_nl_build(ctx, pos, box.box, spec.r_cut, spec.skin, excl, nl=nl), reps=5)
    fp32_probe = ctx.probe_fp32_peak(3.0) if rank == 0 else None
    # Ewald configs: the reciprocal-space half (smooth PME) beside the real-space tau (the paper's Fig. 1(b))
    pme = None
    if spec.method == "ewald" and rank == 0:
        delta = float(np.exp(-(spec.alpha * spec.r_cut) ** 2) / 2.0)  # Eq. 13 solved for delta (2.96e-5 at alpha = 3.12, r_c = 1)
        mesh = dimos.dimos_pme_mesh_size(spec.alpha, box.box, delta)
        Er = torch.empty(2, dtype=torch.float64, device=dev)
        Fr = torch.empty_like(pos)
        dimos.dimos_pme_recip(ctx, pos, charge, box.box, spec.alpha, mesh, order=5, F=Fr, E=Er, virial=W)
        t_pme = timed(lambda: dimos.dimos_pme_recip(ctx, pos, charge, box.box, spec.alpha, mesh, order=5, F=Fr, E=Er, virial=W))
        pme = {"tau_recip_s": t_pme, "mesh": list(mesh), "order": 5, "delta": delta,
               "what": "dimos_pme_recip: spread, cuFFT R2C, influence function + energy/virial, cuFFT C2R, force interpolation, self term"}

    # e2e: the same protocol through dimos_step_host, pinned host buffers, H2D/D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        ring = 2 * TRIANGLE_HALF_PERIOD
        host_pos = [(box.pos.astype(np.float64) + vel * DT_PS * trajectory_offsets(k)).astype(np_real) for k in range(ring)]
        host_pos = [torch.from_numpy(p).pin_memory() for p in host_pos]
        h_charge = torch.from_numpy(box.charge.astype(np_real)).pin_memory()
        h_type = torch.from_numpy(box.type).pin_memory()
        h_excl = torch.from_numpy(box.excl_pairs).pin_memory()
        h_lj = lj_host.pin_memory()
        h_F = torch.empty((n, 3), dtype=real).pin_memory()
        h_E = torch.empty(4, dtype=torch.float64).pin_memory()
        h_W = torch.empty((3, 3), dtype=torch.float64).pin_memory()
        hnl = None
        k = 0
        # first DMA of a freshly page-locked buffer is up to 10x slower on this box (lazy mapping): touch every staging
        # buffer once before anything is timed, as a caller's buffers would have been after its first step
        scratch = torch.empty_like(pos)
        for hp in host_pos:
            scratch.copy_(hp, non_blocking=True)
        h_F.copy_(scratch, non_blocking=True)
        torch.cuda.synchronize()
        del scratch
        # charge / type / lj_table travel once (first call); afterwards only the positions do
        hnl, _ = ctx.step_host(None, host_pos[0], h_charge, h_type, h_lj, box.box, spec.r_cut, spec.skin, h_excl, h_F, h_E, h_W, **kw)
        k = 1
        for _ in range(max(args.warmup, 3)):
            hnl, _ = ctx.step_host(hnl, host_pos[k % ring], None, None, None, box.box, spec.r_cut, spec.skin, h_excl, h_F, h_E,
                                   h_W, ntypes=h_lj.shape[0], **kw)
            k += 1
        # settle: up to 60 more untimed steps until 10 steps in a row without a rebuild take within 8 % of the fastest seen
        # (the first CUDA process on a fresh box has shown host-side transfer times that take a while to come down)
        best, streak = float("inf"), 0
        for _ in range(60):
            ts = time.perf_counter()
            hnl, rb = ctx.step_host(hnl, host_pos[k % ring], None, None, None, box.box, spec.r_cut, spec.skin, h_excl, h_F, h_E,
                                    h_W, ntypes=h_lj.shape[0], **kw)
            k += 1
            if rb:
                continue
            dt_ = time.perf_counter() - ts
            best = min(best, dt_)
            streak = streak + 1 if dt_ <= 1.08 * best else 0
            if streak >= 10:
                break
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        t0 = time.perf_counter()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        e2e_rebuilds = 0
        for _ in range(args.steps):
            hnl, rb = ctx.step_host(hnl, host_pos[k % ring], None, None, None, box.box, spec.r_cut, spec.skin, h_excl, h_F,
                                    h_E, h_W, ntypes=h_lj.shape[0], **kw)
            e2e_rebuilds += int(rb)
            k += 1
        assert bool(torch.isfinite(h_E).all()) and bool(torch.isfinite(h_F).all()), "non-finite result in the e2e region"
        b.record()
        torch.cuda.synchronize()
        e2e_seconds = max(a.elapsed_time(b) * 1e-3, 0.0)
        wall = time.perf_counter() - t0
        if dist:
            dist.barrier()
        rs = 8 if precision == "f64" else 4
        e2e_t, e2e_units = aggregate_over_ranks(e2e_seconds, float(n_cut) * args.steps, world, dist, dev)
        e2e = {"value": e2e_units / e2e_t, "unit": UNIT, "h2d_bytes_per_step": n * 3 * rs,
               "d2h_bytes_per_step": n * 3 * rs + 13 * 8 + 4, "ms_per_step": 1e3 * e2e_t / args.steps, "rebuilds": e2e_rebuilds,
               "wall_ms_per_step": 1e3 * wall / args.steps, "api": "dimos_step_host (pinned host buffers; positions up and F/E/W down every step, charge/type/lj_table once)"}

    total_t, total_units = aggregate_over_ranks(seconds, float(n_cut) * args.steps, world, dist, dev)
    if rank != 0:
        ctx.close()
        if dist:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    flops_per_launch = FLOPS_PER_LISTED_PAIR * n_listed + FLOPS_PER_CUTOFF_PAIR[spec.method] * n_cut
    # every rebuild step holds one pair-kernel launch that found the flag set and returned at once: its few microseconds stay
    # in the numerator, but it is not counted as a launch (the average is over the launches that did the work)
    pair_skipped = rebuilds
    pair_n = max(pair_n - pair_skipped, 0)
    pair_s = pair_ms * 1e-3 / max(pair_n, 1)
    achieved_tflops = flops_per_launch / pair_s * 1e-12 if pair_n else None
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    fp32_peak = n_sm * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 * 1e-12  # TFLOP/s
    if precision == "f64":
        fp32_peak = 40.0  # NVIDIA's nominal B200 FP64 vector rate (no measured figure on this pool); context only
    # the packed kernel runs fp32 boxes with at least three cells per axis, either method (csrc/nonbonded.cu use_f32x2)
    # ... the fp64 kernel every DIMOS_F64 call (csrc/pair_f64.cu), the generic kernel the rest (mixed; small fp32 boxes)
    kernel_name = ("pair_force_f32x2_kernel" if (precision == "f32" and stats["pbc_mode"] == 0)
                   else "pair_force_f64_kernel" if precision == "f64" else "pair_force_kernel")
    list_bytes = stats["list_bytes"] + stats["n_slots"] * (16 + 4 + 16 + 16)
    roofline = {
        "bound": "alu", "kernel": kernel_name, "achieved": achieved_tflops, "peak": fp32_peak, "unit": "TFLOP/s",
        "frac": (achieved_tflops / fp32_peak) if achieved_tflops else None, "traffic": load_traffic(kernel_name, spec.index),
        "traffic_source": "committed ncu --set full capture of this kernel on this workload (profiles/traffic.json), not this run",
        "peak_source": f"derived: {n_sm} SMs x 128 FP32 lanes x 2 x {peaks['sm_max_mhz']:.0f} MHz (DESIGN.md); FFMA probe measured "
                       f"{fp32_probe:.1f} TFLOP/s in this run",
        "fp32_probe_tflops": fp32_probe,
        "flops_per_launch": flops_per_launch, "flop_model": f"{FLOPS_PER_LISTED_PAIR}*N_nl + {FLOPS_PER_CUTOFF_PAIR[spec.method]}*N_c",
        "kernel_ms": 1e3 * pair_s, "kernel_launches_timed": pair_n, "kernel_launches_skipped_on_device": pair_skipped, "kernel_share_of_step": pair_ms * 1e-3 / seconds,
        "hbm_bytes_per_launch": list_bytes, "hbm_gbs_achieved": list_bytes / pair_s * 1e-9 if pair_n else None,
        "hbm_peak_gbs": peaks["hbm_gbs"], "hbm_peak_source": peaks["source"],
        "pair_slots_executed": stats["n_pair_slots"], "fill_in_cutoff": n_cut / stats["n_pair_slots"],
    }
    line = {
        "metric": METRIC, "value": total_units / total_t, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": precision, "data": "synthetic",
        "config": {"workload": workload_name(spec, precision), "n_atoms": n, "pairs_in_cutoff": n_cut, "pairs_listed": n_listed,
                   "protocol": f"ballistic Maxwell-Boltzmann {TEMPERATURE:.0f} K drift, dt=1 fs, trigger checked every step, "
                               f"list rebuilt when it fires ({rebuilds} rebuilds in {args.steps} steps); the force call is "
                               f"enqueued behind the trigger with skip_flag = the device flag and repeated after a rebuild",
                   "l2": f"inputs larger than L2: the pair list streamed per force call is {stats['list_bytes'] / 1e6:.0f} MB",
                   "parallelism": "replicas" if world > 1 else "single"},
        "tau": {"force_s": tau_force, "check_s": tau_check, "build_s": tau_build, "rebuilds": rebuilds,
                "pairs_per_s_force_only": n_cut / tau_force},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "pme": pme,
        "last_step_check": last_step_check,
        "list": {k: stats[k] for k in ("n_units", "n_entries", "n_entries_padded", "n_pair_slots", "list_bytes", "row_capacity")},
    }
    if not args.no_scan and world == 1 and precision != "f64":
        line["tau_vs_n"] = tau_vs_n(ctx, dimos, dev, spec, precision, timed, tau_force, tau_build, n, n_cut)
    if not args.no_scan and world == 1 and box.n_atoms % 3 == 0:
        line["md_step"] = md_step_tau(ctx, dimos, torch, box, spec, pos0, vel, charge, typ, excl, lj, kw)
    if not args.no_cpu_baseline and world >= 1:
        line["cpu_baseline"] = cpu_baseline(spec)
    ctx.close()
    if dist:
        dist.destroy_process_group()
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    spec = wl.CONFIGS[args.config]
    precision = args.precision or ("f32" if "f32" in spec.precisions else spec.precisions[0])
    if args.impl == "reference":
        run_reference(args, spec, precision)
    else:
        run_ours(args, spec, precision)


if __name__ == "__main__":
    main()
