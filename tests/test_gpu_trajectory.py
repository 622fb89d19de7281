"""configs[1] as BASELINE.json states it: 3,000 waters, LJ + reaction field, fp32, 100 steps of velocity-Verlet at
dt = 1 fs from seeded Maxwell-Boltzmann velocities at 300 K, exercising the skin rebuild trigger (PAPER.md:175, 58,
281-301).  The integrator is harness code (reading C-12): per-atom velocity-Verlet, the rigid geometry held
by harness-side harmonic O-H and H-H springs of the Eq. 1 form.  Every step the CUDA path's rebuild
decision, forces and energy are compared with the oracle AT THE TRAJECTORY'S OWN POSITIONS, and the list-validity
invariant (every in-cutoff pair is in the list built earlier) is checked against the oracle's pair set."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

from gpu_harness import BAND, check_nonbonded, lj_table_np, pair_keys

pytestmark = pytest.mark.gpu

K_OH, K_HH = 2.5e5, 1.0e5  # kJ mol^-1 nm^-2, U = k (r - r0)^2 (Eq. 1, no 1/2)


def spring_forces(pos, bonds, r0, k):
    d = pos[bonds[:, 0]] - pos[bonds[:, 1]]
    r = d.norm(dim=1, keepdim=True)
    f = (-2.0 * k * (r - r0) / r) * d  # force on the first atom
    out = torch.zeros_like(pos)
    out.index_add_(0, bonds[:, 0], f)
    out.index_add_(0, bonds[:, 1], -f)
    return out


def test_config1_100_steps_velocity_verlet_f32():
    wb = wl.make_config(1)
    n = wb.n_atoms
    rc, skin, dt = 1.0, 0.1, 0.001
    dev = torch.device("cuda", 0)
    x = torch.from_numpy(wb.pos.astype(np.float64)).to(dev)
    v = torch.from_numpy(wl.maxwell_boltzmann_velocities(wb.mass, 300.0, wl.SEED_BASE + 11)).to(dev)
    inv_m = torch.from_numpy(1.0 / wb.mass).to(dev)[:, None]
    charge = torch.from_numpy(wb.charge).to(dev)
    typ = torch.from_numpy(wb.type).to(dev)
    excl = torch.from_numpy(wb.excl_pairs).to(dev)
    lj_np = lj_table_np(wb)
    lj = torch.from_numpy(lj_np).to(dev)
    bonds = excl.long()
    is_hh = (typ[bonds[:, 0]] == 1) & (typ[bonds[:, 1]] == 1)
    hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    r0 = torch.where(is_hh, torch.tensor(hh, device=dev, dtype=torch.float64), torch.tensor(wl.R_OH, device=dev, dtype=torch.float64))[:, None]
    kk = torch.where(is_hh, torch.tensor(K_HH, device=dev, dtype=torch.float64), torch.tensor(K_OH, device=dev, dtype=torch.float64))[:, None]

    ctx = dimos.Context(0, "f32")
    try:
        x32 = x.float().contiguous()
        nl = dimos.dimos_nl_build(ctx, x32, wb.box, rc, skin, excl)
        listed = set(pair_keys(dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy(), n).tolist())
        F, E, W = dimos.dimos_nonbonded(ctx, nl, x32, charge, typ, lj)
        f = F.double() + spring_forces(x, bonds, r0, kk)
        rebuilds, worst_f, worst_e, ambiguous = 0, 0.0, 0.0, 0
        for step in range(100):
            v += 0.5 * dt * f * inv_m          # 1. half kick
            x += dt * v                        # 2. drift
            x32 = x.float().contiguous()
            x_np = x32.double().cpu().numpy()
            # A3: rebuild decision vs the oracle's, on the same fp32 positions
            want, m = oracle.needs_rebuild(x32.cpu().numpy(), nl.pos_at_build.cpu().numpy(), skin)
            got = dimos.dimos_nl_needs_rebuild(ctx, x32, nl.pos_at_build, skin)
            if abs(m - 0.5 * skin) > 1e-6:
                assert got == want, (step, m)
            else:
                ambiguous += 1
            if got:
                nl = dimos.dimos_nl_build(ctx, x32, wb.box, rc, skin, excl, nl=nl)
                listed = set(pair_keys(dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy(), n).tolist())
                rebuilds += 1
            # list validity: every pair inside r_c now is in the list built earlier
            now = pair_keys(oracle.neighbor_pairs(x_np, wb.box, rc - BAND, wb.excl_pairs, "celllist"), n)
            missing = [k for k in now.tolist() if k not in listed]
            assert not missing, f"step {step}: {len(missing)} in-cutoff pairs missing from the list"
            # A4-A6: forces, energy, virial at these positions     (4. compute a(t+dt))
            F, E, W = dimos.dimos_nonbonded(ctx, nl, x32, charge, typ, lj)
            orc = oracle.nonbonded(x_np, wb.charge, wb.type, lj_np, wb.box, rc, excl_pairs=wb.excl_pairs, band=BAND)
            rep = check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32")
            worst_f, worst_e = max(worst_f, rep["max_dF_over_rms"]), max(worst_e, rep["e_rel"])
            f = F.double() + spring_forces(x, bonds, r0, kk)
            v += 0.5 * dt * f * inv_m          # 5. half kick
        assert 3 <= rebuilds <= 60, rebuilds  # the trigger fired several times, and not every step
        # the molecules stayed intact (the harness springs did their job, so the workload stayed water-like)
        d = (x[bonds[:, 0]] - x[bonds[:, 1]]).norm(dim=1)
        assert float((d - r0[:, 0]).abs().max()) < 0.02
        print(f"rebuilds={rebuilds} worst max|dF|/rms={worst_f:.2e} worst |dE|/|E|={worst_e:.2e} ambiguous flags={ambiguous}")
    finally:
        ctx.close()
