"""`-m gpu`: the steps between two list rebuilds as a CUDA graph.  The per-step sequence trigger -> forces
(dimos_nl_needs_rebuild_static with the flag left on the device, dimos_nonbonded with dimos_nb_params.skip_flag = that
flag) enqueues only kernels and one memset, allocates nothing once the list's per-step workspace
exists and never synchronises, so a stream capture records it and a replay runs it with one launch.  A rebuild changes
the list's buffers and sizes, so the graph is captured again after every dimos_nl_build.  Every step's forces, energies and
virial are compared with the oracle at that step's positions, and the flag with the oracle's rebuild decision."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

from gpu_harness import BAND, METHOD, DeviceBox, check_nonbonded

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f64", "ewald")])
def test_steps_between_rebuilds_replayed_as_a_cuda_graph(precision, method):
    wb = wl.make_config(1)
    db = DeviceBox(wb, precision)
    dev = db.pos.device
    real = db.pos.dtype
    vel = wl.maxwell_boltzmann_velocities(wb.mass, 300.0, wl.SEED_BASE + 21)
    dstep = torch.from_numpy(vel * 0.003).to(dev, real)  # 3 fs of ballistic drift per step: a rebuild every few steps
    pos = db.pos.clone()
    F = torch.zeros_like(pos)
    E = torch.zeros(4, dtype=torch.float64, device=dev)
    W = torch.zeros(3, 3, dtype=torch.float64, device=dev)
    flag = torch.zeros(1, dtype=torch.int32, device=dev)
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, pos, db.box, 1.0, 0.1, db.excl)
        dimos.dimos_nonbonded(ctx, nl, pos, db.charge, db.type, db.lj, method=method, F=F, E=E, virial=W)  # workspace exists now
        e_scale = abs(float(E[0]))

        def step_body():
            pos.add_(dstep)  # the harness's "integrator" is part of the graph as well
            dimos.dimos_nl_needs_rebuild_static(ctx, pos, nl.pos_at_build, 0.1, flag)
            dimos.dimos_nonbonded(ctx, nl, pos, db.charge, db.type, db.lj, method=method, F=F, E=E, virial=W, skip_flag=flag)

        def capture():
            # torch's capture recipe: the captured calls ran once before (here: the force call above), capture on a side stream
            g = torch.cuda.CUDAGraph()
            keep = pos.clone()
            with torch.cuda.graph(g):
                step_body()
            pos.copy_(keep)  # capturing does not execute, but be explicit: the positions are those before the step
            return g

        launches0 = ctx.launch_count()
        graph = capture()
        per_capture = ctx.launch_count() - launches0
        assert per_capture >= 4  # trigger, gather, pair kernel, finalize (+ exclusion correction under Ewald)
        replays, rebuilds = 0, 0
        for step in range(14):
            graph.replay()
            replays += 1
            torch.cuda.synchronize()
            want, m = oracle.needs_rebuild(pos.cpu().numpy(), nl.pos_at_build.cpu().numpy(), 0.1)
            fired = bool(flag.item())
            assert fired == want or abs(m - 0.05) < 1e-6
            if fired:  # the force kernels of the replay did nothing: rebuild, compute, and record the graph for the new list
                nl = dimos.dimos_nl_build(ctx, pos, db.box, 1.0, 0.1, db.excl, nl=nl)
                dimos.dimos_nonbonded(ctx, nl, pos, db.charge, db.type, db.lj, method=method, F=F, E=E, virial=W)
                graph = capture()
                rebuilds += 1
            orc = oracle.nonbonded(pos.double().cpu().numpy(), db.charge.double().cpu().numpy(), wb.type, db.lj_np, db.box, 1.0,
                                   method=METHOD[method], excl_pairs=wb.excl_pairs, band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision, e_floor=e_scale)
        assert 2 <= rebuilds <= 8, rebuilds
        # replays launch the recorded kernels without passing through the library: its launch counter only saw the captures
        assert ctx.launch_count() - launches0 <= (rebuilds + 1) * per_capture + rebuilds * 60
    finally:
        ctx.close()


def test_rigid_water_md_steps_replayed_as_a_cuda_graph_f32():
    """The whole velocity-Verlet step of PAPER.md:281-292 for rigid water as ONE graph: dimos_water_kick_drift_settle (steps
    1-3 and the trigger, which leaves its flag on the device), dimos_nonbonded (step 4) and dimos_water_kick_settle_velocities
    (steps 5-6), the last two conditional on that flag.  On the step where the trigger fires the replay has advanced the
    positions and done nothing else; the host rebuilds the list, computes the forces, applies the second kick and records
    the graph again.  Every step's forces against the oracle at the trajectory's own positions; the molecules stay rigid;
    and the trajectory equals, to the rounding of the force sums, the one the same calls produce without a graph."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    dev = db.pos.device
    n = wb.n_atoms
    m_O, m_H = float(wb.mass[0]), float(wb.mass[1])
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * float(np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0))
    water = torch.arange(n, dtype=torch.int32, device=dev).reshape(-1, 3)
    v0 = torch.from_numpy(wl.maxwell_boltzmann_velocities(wb.mass, 300.0, wl.SEED_BASE + 31).astype(np.float32)).to(dev)
    dt, skin, n_steps = 0.001, 0.1, 36

    def run(use_graph):
        ctx = dimos.Context(0, "f32")
        try:
            x, v = db.pos.clone(), v0.clone()
            dimos.dimos_settle_velocities(ctx, x, v, water, m_O, m_H)
            nl = dimos.dimos_nl_build(ctx, x, db.box, 1.0, skin, db.excl)
            F, E, W = dimos.dimos_nonbonded(ctx, nl, x, db.charge, db.type, db.lj)
            e_scale = abs(float(E[0]))

            def body():
                dimos.dimos_water_kick_drift_settle(ctx, x, v, F, water, m_O, m_H, d_oh, d_hh, dt, pos_at_build=nl.pos_at_build,
                                                    skin=skin, sync=False, flag=flag)
                dimos.dimos_nonbonded(ctx, nl, x, db.charge, db.type, db.lj, F=F, E=E, virial=W, skip_flag=flag)
                dimos.dimos_water_kick_settle_velocities(ctx, x, v, F, water, m_O, m_H, dt, skip_flag=flag)
                return flag

            def capture():
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    body()
                return g

            flag = torch.zeros(1, dtype=torch.int32, device=dev)  # the device word the trigger writes and the other two calls read
            graph = capture() if use_graph else None
            rebuilds = 0
            for step in range(n_steps):
                if use_graph:
                    graph.replay()
                else:
                    body()
                torch.cuda.synchronize()
                if int(flag.item()):
                    nl = dimos.dimos_nl_build(ctx, x, db.box, 1.0, skin, db.excl, nl=nl)
                    dimos.dimos_nonbonded(ctx, nl, x, db.charge, db.type, db.lj, F=F, E=E, virial=W)
                    dimos.dimos_water_kick_settle_velocities(ctx, x, v, F, water, m_O, m_H, dt)
                    rebuilds += 1
                    if use_graph:
                        graph = capture()
                if use_graph:  # forces of this step against the oracle at this step's positions
                    orc = oracle.nonbonded(x.double().cpu().numpy(), wb.charge, wb.type, db.lj_np, db.box, 1.0,
                                           excl_pairs=wb.excl_pairs, band=BAND)
                    check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32", e_floor=e_scale)
            torch.cuda.synchronize()
            return x.double().cpu().numpy(), v.double().cpu().numpy(), rebuilds
        finally:
            ctx.close()

    xg, vg, rebuilds_g = run(True)
    xe, ve, rebuilds_e = run(False)
    assert rebuilds_g == rebuilds_e and 2 <= rebuilds_g <= 20, (rebuilds_g, rebuilds_e)
    mol = xg.reshape(-1, 3, 3)
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):
        assert np.abs(np.linalg.norm(mol[:, i] - mol[:, j], axis=1) - d).max() < 3e-6
    # same calls, same order: the two trajectories differ only by the summation order of the force reductions
    assert np.abs(xg - xe).max() < 2e-5 and np.abs(vg - ve).max() < 2e-3 * np.abs(ve).max()


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_pme_recip_replayed_as_a_cuda_graph(precision):
    """dimos_pme_recip after a first call with the same mesh, order, alpha and box (which makes the cuFFT plans and the
    per-axis tables) only enqueues kernels, memsets and the two cuFFT executions: recorded once, replayed for moved atoms,
    against the numpy PME oracle."""
    from oracle import pme_oracle as pme

    wb = wl.make_config(1)
    real = torch.float64 if precision == "f64" else torch.float32
    dev = torch.device("cuda", 0)
    pos = torch.from_numpy(wb.pos).to(dev, real)
    q = torch.from_numpy(wb.charge).to(dev, real)
    mesh, order, alpha = (36, 40, 42), 5, 3.12
    F = torch.zeros_like(pos)
    E = torch.zeros(2, dtype=torch.float64, device=dev)
    W = torch.zeros(3, 3, dtype=torch.float64, device=dev)
    ctx = dimos.Context(0, precision)
    try:
        dimos.dimos_pme_recip(ctx, pos, q, wb.box, alpha, mesh, order=order, F=F, E=E, virial=W)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            dimos.dimos_pme_recip(ctx, pos, q, wb.box, alpha, mesh, order=order, F=F, E=E, virial=W)
        rng = np.random.default_rng(2)
        for rep in range(3):
            pos.add_(torch.from_numpy(rng.normal(0.0, 0.02, size=tuple(pos.shape))).to(dev, real))
            F.fill_(7.0)
            E.fill_(-1.0)
            graph.replay()
            torch.cuda.synchronize()
            U0, F0, W0 = pme.pme_recip(pos.double().cpu().numpy(), q.double().cpu().numpy(), wb.box, alpha, mesh, order)
            e_tol, f_tol, w_tol = (1e-10, 1e-10, 1e-9) if precision == "f64" else (1e-5, 1e-4, 1e-4)
            assert abs(float(E[0]) - U0) <= e_tol * abs(U0)
            rms = np.sqrt((F0 ** 2).sum(axis=1).mean())
            assert np.sqrt(((F.double().cpu().numpy() - F0) ** 2).sum(axis=1)).max() <= f_tol * rms
            assert np.abs(W.cpu().numpy() - W0).max() <= w_tol * np.abs(W0).max()
    finally:
        ctx.close()
