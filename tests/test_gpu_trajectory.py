"""configs[1] as BASELINE.json states it: 3,000 rigid TIP3P-geometry waters, LJ + reaction field, fp32, 100 steps of
velocity Verlet at dt = 1 fs from seeded Maxwell-Boltzmann velocities at 300 K, exercising the skin rebuild trigger
(PAPER.md:175, 58, 281-301).  The whole step is library calls: dimos_water_kick_drift_settle (steps 1-3 with SETTLE and the
fused trigger), dimos_nl_build when it fired, dimos_nonbonded (step 4), dimos_water_kick_settle_velocities (steps 5-6).
Every step the CUDA path's rebuild decision, forces, energy and virial are compared with the oracle AT THE TRAJECTORY'S OWN
POSITIONS, the list-validity invariant (every in-cutoff pair is in the list built earlier) is checked against the
oracle's pair set, and the water geometry must stay rigid."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

from gpu_harness import BAND, check_nonbonded, lj_table_np, pair_keys

pytestmark = pytest.mark.gpu


def test_config1_100_steps_rigid_water_velocity_verlet_f32():
    wb = wl.make_config(1)
    n = wb.n_atoms
    rc, skin, dt = 1.0, 0.1, 0.001
    dev = torch.device("cuda", 0)
    m_O, m_H = float(wb.mass[0]), float(wb.mass[1])
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * float(np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0))
    x = torch.from_numpy(wb.pos.astype(np.float32)).to(dev)
    v = torch.from_numpy(wl.maxwell_boltzmann_velocities(wb.mass, 300.0, wl.SEED_BASE + 11).astype(np.float32)).to(dev)
    water = torch.arange(n, dtype=torch.int32, device=dev).reshape(-1, 3)
    charge = torch.from_numpy(wb.charge).to(dev)
    typ = torch.from_numpy(wb.type).to(dev)
    excl = torch.from_numpy(wb.excl_pairs).to(dev)
    lj_np = lj_table_np(wb)
    lj = torch.from_numpy(lj_np).to(dev)

    ctx = dimos.Context(0, "f32")
    try:
        dimos.dimos_settle_velocities(ctx, x, v, water, m_O, m_H)  # start on the constraint manifold
        nl = dimos.dimos_nl_build(ctx, x, wb.box, rc, skin, excl)
        listed = set(pair_keys(dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy(), n).tolist())
        F, E, W = dimos.dimos_nonbonded(ctx, nl, x, charge, typ, lj)
        e_scale = abs(float(E[0]))  # +7.6e3 kJ/mol; the box relaxes through E = 0 within the 100 steps
        rebuilds, worst_f, worst_e, ambiguous = 0, 0.0, 0.0, 0
        for step in range(100):
            # steps 1-3 + the trigger on the constrained positions
            got = dimos.dimos_water_kick_drift_settle(ctx, x, v, F, water, m_O, m_H, d_oh, d_hh, dt, pos_at_build=nl.pos_at_build,
                                                      skin=skin)
            x_np = x.double().cpu().numpy()
            # A3: rebuild decision vs the oracle's, on the same fp32 positions
            want, m = oracle.needs_rebuild(x.cpu().numpy(), nl.pos_at_build.cpu().numpy(), skin)
            if abs(m - 0.5 * skin) > 1e-6:
                assert got == want, (step, m)
            else:
                ambiguous += 1
            if got:
                nl = dimos.dimos_nl_build(ctx, x, wb.box, rc, skin, excl, nl=nl)
                listed = set(pair_keys(dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy(), n).tolist())
                rebuilds += 1
            # list validity: every pair inside r_c now is in the list built earlier
            now = pair_keys(oracle.neighbor_pairs(x_np, wb.box, rc - BAND, wb.excl_pairs, "celllist"), n)
            missing = [k for k in now.tolist() if k not in listed]
            assert not missing, f"step {step}: {len(missing)} in-cutoff pairs missing from the list"
            # A4-A6: forces, energy, virial at these positions     (4. compute a(t+dt))
            F, E, W = dimos.dimos_nonbonded(ctx, nl, x, charge, typ, lj, F=F)
            orc = oracle.nonbonded(x_np, wb.charge, wb.type, lj_np, wb.box, rc, excl_pairs=wb.excl_pairs, band=BAND)
            rep = check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32", e_floor=e_scale)
            worst_f, worst_e = max(worst_f, rep["max_dF_over_rms"]), max(worst_e, rep["e_rel"])
            # steps 5-6
            dimos.dimos_water_kick_settle_velocities(ctx, x, v, F, water, m_O, m_H, dt)
        assert 3 <= rebuilds <= 60, rebuilds  # the trigger fired several times, and not every step
        mol = x.double().cpu().numpy().reshape(-1, 3, 3)
        for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):
            assert np.abs(np.linalg.norm(mol[:, i] - mol[:, j], axis=1) - d).max() < 3e-6  # rigid to fp32 rounding
        print(f"rebuilds={rebuilds} worst max|dF|/rms={worst_f:.2e} worst |dE|/|E|={worst_e:.2e} ambiguous flags={ambiguous}")
    finally:
        ctx.close()
