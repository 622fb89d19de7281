"""Velocity-Verlet kernels (steps 1, 2, 5) against the numpy fp64 oracle, element by element, and the
rebuild trigger fused into the drift against the oracle's trigger on the same new positions."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n", [1, 7, 1000, 70001])
def test_kick_drift_and_kick_match_oracle(precision, n):
    rng = np.random.default_rng(40 + n)
    np_real = np.float64 if precision == "f64" else np.float32
    pos = rng.uniform(0.0, 5.0, size=(n, 3)).astype(np_real)
    vel = rng.normal(0.0, 1.5, size=(n, 3)).astype(np_real)
    F = rng.normal(0.0, 700.0, size=(n, 3)).astype(np_real)
    F2 = rng.normal(0.0, 700.0, size=(n, 3)).astype(np_real)
    inv_m = (1.0 / rng.choice(np.array([15.9994, 1.008]), size=n)).astype(np_real)
    dt = 0.001
    dev = torch.device("cuda", 0)
    ctx = dimos.Context(0, precision)
    try:
        ref = torch.from_numpy(pos.copy()).to(dev)
        x, v = torch.from_numpy(pos.copy()).to(dev), torch.from_numpy(vel.copy()).to(dev)
        skin = 0.016  # of the order of dt * max speed, so the flag is not trivially decided
        flag = dimos.dimos_vv_kick_drift(ctx, x, v, torch.from_numpy(F).to(dev), torch.from_numpy(inv_m).to(dev), dt,
                                         pos_at_build=ref, skin=skin)
        x_o, v_o = oracle.vv_kick_drift(pos, vel, F, inv_m, dt)
        tol = 1e-14 if precision == "f64" else 2e-7
        assert np.abs(x.cpu().numpy() - x_o).max() <= tol * 5.0
        assert np.abs(v.cpu().numpy() - v_o).max() <= tol * max(1.0, np.abs(v_o).max())
        want, m = oracle.needs_rebuild(x.cpu().numpy(), pos, skin)  # the trigger on the kernel's own new positions
        if abs(m - 0.5 * skin) > 1e-6:
            assert flag == want, (m, skin)
        dimos.dimos_vv_kick(ctx, v, torch.from_numpy(F2).to(dev), torch.from_numpy(inv_m).to(dev), dt)
        v2_o = oracle.vv_kick(v_o, F2, inv_m, dt)
        assert np.abs(v.cpu().numpy() - v2_o).max() <= 2 * tol * max(1.0, np.abs(v2_o).max())
        # without reference positions the same update runs with no flag
        x3, v3 = torch.from_numpy(pos.copy()).to(dev), torch.from_numpy(vel.copy()).to(dev)
        assert dimos.dimos_vv_kick_drift(ctx, x3, v3, torch.from_numpy(F).to(dev), torch.from_numpy(inv_m).to(dev), dt) is None
        assert torch.equal(x3, x) and torch.allclose(v3 + 0.0, torch.from_numpy(v_o.astype(np_real)).to(dev), rtol=1e-5, atol=1e-5)
    finally:
        ctx.close()


def test_md_loop_through_the_library_f32():
    """A short MD loop made only of library calls (kick + drift with the fused trigger, rebuild when it fires,
    nonbonded, kick) on a box of LJ + RF point particles: momentum is conserved by the pair forces and the trigger /
    rebuild sequence equals the one a separate dimos_nl_needs_rebuild call gives."""
    wb = wl.make_config(1)
    dev = torch.device("cuda", 0)
    sel = np.arange(0, wb.n_atoms, 3)  # oxygens only: a stable LJ + RF fluid without bonded terms
    pos = torch.from_numpy(wb.pos[sel].copy()).to(dev)
    charge = torch.from_numpy(wb.charge[sel].copy()).to(dev)
    typ = torch.from_numpy(wb.type[sel].copy()).to(dev)
    lj = dimos.lj_table_from_types(wb.sigma, wb.epsilon).to(dev)
    mass = wb.mass[sel]
    vel = torch.from_numpy(wl.maxwell_boltzmann_velocities(mass, 300.0, 5).astype(np.float32)).to(dev)
    inv_m = torch.from_numpy((1.0 / mass).astype(np.float32)).to(dev)
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, pos, wb.box, 1.0, 0.1, None)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj)
        p0 = (vel.double() / inv_m.double()[:, None]).sum(0)
        rebuilds = 0
        for _ in range(60):
            fired = dimos.dimos_vv_kick_drift(ctx, pos, vel, F, inv_m, 0.004, pos_at_build=nl.pos_at_build, skin=0.1)
            assert fired == dimos.dimos_nl_needs_rebuild(ctx, pos, nl.pos_at_build, 0.1)
            if fired:
                nl = dimos.dimos_nl_build(ctx, pos, wb.box, 1.0, 0.1, None, nl=nl)
                rebuilds += 1
            F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F)
            dimos.dimos_vv_kick(ctx, vel, F, inv_m, 0.004)
        p1 = (vel.double() / inv_m.double()[:, None]).sum(0)
        assert rebuilds >= 1
        scale = float((vel.double() / inv_m.double()[:, None]).abs().sum(0).max())  # sum of |p_i| per axis
        assert float((p1 - p0).abs().max()) < 1e-4 * scale  # pair forces are antisymmetric: total momentum is conserved
        assert bool(torch.isfinite(E).all())
    finally:
        ctx.close()
