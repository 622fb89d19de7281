"""`-m gpu`: dimos_step_host, the host-buffer entry point behind bench.py's `e2e` number, on bench.py's own trajectory
(ballistic Maxwell-Boltzmann drift, triangle wave) of configs[1]: every step's F_host / E_host / W_host against the oracle
at that step's positions, and rebuilt_host against oracle.needs_rebuild relative to the positions of the last rebuild."""
import numpy as np
import pytest
import torch

import bench
import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

from gpu_harness import BAND, check_nonbonded, lj_table_np

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f64", "ewald")])
def test_step_host_trajectory_matches_oracle_every_step(precision, method):
    wb = wl.make_config(1)
    n = wb.n_atoms
    rc, skin = 1.0, 0.1
    real = np.float64 if precision == "f64" else np.float32
    treal = torch.float64 if precision == "f64" else torch.float32
    vel = wl.maxwell_boltzmann_velocities(wb.mass, bench.TEMPERATURE, wl.SEED_BASE + 7)
    lj_np = lj_table_np(wb)
    h_charge = torch.from_numpy(wb.charge.astype(real)).pin_memory()
    h_type = torch.from_numpy(wb.type).pin_memory()
    h_excl = torch.from_numpy(wb.excl_pairs).pin_memory()
    h_lj = torch.from_numpy(lj_np).pin_memory()
    h_F = torch.empty((n, 3), dtype=treal).pin_memory()
    h_E = torch.empty(4, dtype=torch.float64).pin_memory()
    h_W = torch.empty((3, 3), dtype=torch.float64).pin_memory()
    h_pos = torch.empty((n, 3), dtype=treal).pin_memory()
    ometh = oracle.METHOD_RF if method == "rf" else oracle.METHOD_EWALD_REAL
    ctx = dimos.Context(0, precision)
    try:
        nl, ref, rebuilds, ambiguous = None, None, 0, 0
        for step in range(30):
            p = (wb.pos.astype(np.float64) + vel * bench.DT_PS * bench.trajectory_offsets(step)).astype(real)
            h_pos.copy_(torch.from_numpy(p))
            h_F.fill_(float("nan"))
            h_E.fill_(float("nan"))
            h_W.fill_(float("nan"))
            if step % 3 == 1:  # static inputs omitted: the list's device copies are used again
                nl, rebuilt = ctx.step_host(nl, h_pos, None, None, None, wb.box, rc, skin, h_excl, h_F, h_E, h_W, method=method, ntypes=2)
            else:
                nl, rebuilt = ctx.step_host(nl, h_pos, h_charge, h_type, h_lj, wb.box, rc, skin, h_excl, h_F, h_E, h_W, method=method)
            if step == 0:
                assert rebuilt, "the first call builds the list"
            else:
                want, m = oracle.needs_rebuild(p, ref, skin)
                if abs(m - 0.5 * skin) > 1e-6:  # reading C-5
                    assert rebuilt == want, (step, m)
                else:
                    ambiguous += 1
            if rebuilt:
                ref = p.copy()
                rebuilds += 1
            orc = oracle.nonbonded(p, wb.charge, wb.type, lj_np, wb.box, rc, method=ometh, excl_pairs=wb.excl_pairs, band=BAND)
            check_nonbonded(h_F.numpy(), h_E.numpy(), h_W.numpy(), orc, precision)
        assert 3 <= rebuilds <= 15, rebuilds  # the trigger fired several times and not every step
        # charge / type / lj_table changes are picked up by the next call (they are inputs of every call)
        h_charge.mul_(0.5)
        nl, rebuilt = ctx.step_host(nl, h_pos, h_charge, h_type, h_lj, wb.box, rc, skin, h_excl, h_F, h_E, h_W, method=method)
        orc = oracle.nonbonded(p, 0.5 * wb.charge.astype(np.float64), wb.type, lj_np, wb.box, rc, method=ometh,
                               excl_pairs=wb.excl_pairs, band=BAND)
        check_nonbonded(h_F.numpy(), h_E.numpy(), h_W.numpy(), orc, precision)
        # without a list there is nothing to reuse
        with pytest.raises(dimos.DimosError):
            ctx.step_host(None, h_pos, None, None, None, wb.box, rc, skin, h_excl, h_F, h_E, h_W, method=method, ntypes=2)
    finally:
        ctx.close()
