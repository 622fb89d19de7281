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
