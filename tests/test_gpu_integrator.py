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


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n_w", [1, 33, 5000])
def test_settle_matches_converged_shake(precision, n_w):
    """dimos_settle (step 3; SETTLE) against the oracle's SHAKE iterated to 1e-14: same
    constrained positions, bond lengths on the constraint, molecular centre of mass untouched, and the velocity picks up
    (x_c - x_u) / dt.  Molecules are shuffled in memory so that the index table is exercised."""
    rng = np.random.default_rng(900 + n_w)
    np_real = np.float64 if precision == "f64" else np.float32
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    m_O, m_H = 15.9994, 1.008
    # rigid molecules with random orientations and positions (built from the canonical triangle by a random rotation)
    half = np.radians(wl.ANGLE_HOH_DEG) / 2.0
    tri = np.array([[0.0, 0.0, 0.0], [d_oh * np.sin(half), 0.0, d_oh * np.cos(half)], [-d_oh * np.sin(half), 0.0, d_oh * np.cos(half)]])
    q = rng.normal(size=(n_w, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], -1),
                  np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], -1),
                  np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], -1)], 1)
    x0 = np.einsum("nij,kj->nki", R, tri) + rng.uniform(0.0, 6.0, size=(n_w, 1, 3))
    x0 = x0.reshape(-1, 3).astype(np_real)  # what the device holds; rigid to the rounding of np_real
    mass = np.tile([m_O, m_H, m_H], n_w)
    dt = 0.002
    v = rng.normal(0.0, 1.0, size=(3 * n_w, 3)) / np.sqrt(mass)[:, None] * 1.5   # thermal-sized velocities, nm/ps
    x1 = (x0.astype(np.float64) + dt * v).astype(np_real)
    # the oracle works on exactly the device's inputs, from an old configuration made rigid in fp64
    x0_64 = oracle.shake_water(x0.astype(np.float64), x0.astype(np.float64), mass, d_oh, d_hh)
    ref = oracle.shake_water(x0_64, x1.astype(np.float64), mass, d_oh, d_hh)
    perm = rng.permutation(3 * n_w)          # atom k of the molecule order sits at memory index perm[k]
    inv = np.empty_like(perm)
    inv[perm] = np.arange(3 * n_w)
    water = perm.reshape(n_w, 3).astype(np.int32)
    dev = torch.device("cuda", 0)
    with dimos.Context(0, precision) as ctx:
        p_old = torch.from_numpy(np.ascontiguousarray(x0[inv])).to(dev)
        p = torch.from_numpy(np.ascontiguousarray(x1[inv])).to(dev)
        vel0 = v.astype(np_real)
        vd = torch.from_numpy(np.ascontiguousarray(vel0[inv])).to(dev)
        dimos.dimos_settle(ctx, p_old, p, torch.from_numpy(water).to(dev), m_O, m_H, d_oh, d_hh, vel=vd, dt=dt)
        torch.cuda.synchronize()
        got = p.cpu().numpy().astype(np.float64)[perm]
        got_v = vd.cpu().numpy().astype(np.float64)[perm]
        # without vel: positions identical, velocities untouched
        p2 = torch.from_numpy(np.ascontiguousarray(x1[inv])).to(dev)
        dimos.dimos_settle(ctx, p_old, p2, torch.from_numpy(water).to(dev), m_O, m_H, d_oh, d_hh)
        torch.cuda.synchronize()
        assert torch.equal(p2, p)
        dimos.dimos_settle(ctx, p_old, p2, torch.from_numpy(water[:0].copy()).to(dev), m_O, m_H, d_oh, d_hh)  # n_w = 0
        with pytest.raises(dimos.DimosError):
            dimos.dimos_settle(ctx, p_old, p2, torch.from_numpy(water).to(dev), m_O, m_H, d_oh, 2.5 * d_oh)
    # fp32: coordinates up to 6 nm carry 2.4e-7 nm of rounding each; fp64: the oracle's own convergence (1e-14 relative)
    tol = 5e-12 if precision == "f64" else 3e-6
    assert np.abs(got - ref).max() < tol
    m = got.reshape(-1, 3, 3)
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):
        assert np.abs(np.linalg.norm(m[:, i] - m[:, j], axis=1) - d).max() < tol
    wgt = mass.reshape(-1, 3, 1)
    com = lambda a: (a.reshape(-1, 3, 3) * wgt).sum(1) / wgt.sum(1)
    assert np.abs(com(got) - com(x1.astype(np.float64))).max() < tol
    ref_v = vel0.astype(np.float64) + (ref - x1.astype(np.float64)) / dt
    assert np.abs(got_v - ref_v).max() < tol / dt * 2


def _random_rigid_waters(rng, n_w, d_oh, d_hh, span=6.0):
    half = np.arcsin(0.5 * d_hh / d_oh)
    tri = np.array([[0.0, 0.0, 0.0], [d_oh * np.sin(half), 0.0, d_oh * np.cos(half)], [-d_oh * np.sin(half), 0.0, d_oh * np.cos(half)]])
    q = rng.normal(size=(n_w, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], -1),
                  np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], -1),
                  np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], -1)], 1)
    return (np.einsum("nij,kj->nki", R, tri) + rng.uniform(0.0, span, size=(n_w, 1, 3))).reshape(-1, 3)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n_w", [1, 33, 5000])
def test_settle_velocities_match_converged_rattle(precision, n_w):
    """dimos_settle_velocities (step 6) against the oracle's iterative RATTLE velocity stage, and the
    properties that hold at any size: v_ij . r_ij = 0 on the three bonds, molecular linear and angular momentum kept."""
    rng = np.random.default_rng(1200 + n_w)
    np_real = np.float64 if precision == "f64" else np.float32
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    m_O, m_H = 15.9994, 1.008
    mass = np.tile([m_O, m_H, m_H], n_w)
    x = _random_rigid_waters(rng, n_w, d_oh, d_hh).astype(np_real)
    v = (rng.normal(0.0, 1.5, size=x.shape) / np.sqrt(mass)[:, None]).astype(np_real)
    ref = oracle.rattle_water_velocities(x.astype(np.float64), v.astype(np.float64), mass)
    water = np.arange(3 * n_w, dtype=np.int32).reshape(n_w, 3)
    dev = torch.device("cuda", 0)
    with dimos.Context(0, precision) as ctx:
        vd = torch.from_numpy(v.copy()).to(dev)
        dimos.dimos_settle_velocities(ctx, torch.from_numpy(x).to(dev), vd, torch.from_numpy(water).to(dev), m_O, m_H)
        torch.cuda.synchronize()
        got = vd.cpu().numpy().astype(np.float64)
    vmax = np.abs(v).max()
    tol = (1e-12 if precision == "f64" else 2e-5) * vmax
    assert np.abs(got - ref).max() < tol
    X, G, V0, M = x.astype(np.float64).reshape(-1, 3, 3), got.reshape(-1, 3, 3), v.astype(np.float64).reshape(-1, 3, 3), mass.reshape(-1, 3, 1)
    for i, j in ((0, 1), (0, 2), (1, 2)):
        r = X[:, i] - X[:, j]
        assert np.abs(((G[:, i] - G[:, j]) * r).sum(1) / np.linalg.norm(r, axis=1)).max() < tol
    assert np.abs((M * G).sum(1) - (M * V0).sum(1)).max() < tol * m_O
    Xc = X - X[:, :1]
    assert np.abs((M * np.cross(Xc, G)).sum(1) - (M * np.cross(Xc, V0)).sum(1)).max() < tol * m_O * d_oh * 4


@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_constrained_velocity_verlet_steps_match_oracle(precision, fused):
    """Steps 1, 2, 3, 5, 6 of PAPER.md:281-292 chained on the device for rigid water with seeded forces, four time steps in
    a row, against the same chain of oracle functions (kick+drift, SHAKE, kick, RATTLE velocities): positions, velocities,
    and the rigid geometry at the end.  fused: the same chain through dimos_water_kick_drift_settle and
    dimos_water_kick_settle_velocities (two passes per step), with the rebuild flag and the kinetic energy they report
    checked against the oracle's on the last step."""
    n_w = 700
    rng = np.random.default_rng(77)
    np_real = np.float64 if precision == "f64" else np.float32
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    m_O, m_H = 15.9994, 1.008
    mass = np.tile([m_O, m_H, m_H], n_w)
    inv_m = (1.0 / mass).astype(np_real)
    dt = 0.002
    x = _random_rigid_waters(rng, n_w, d_oh, d_hh).astype(np_real)
    v0 = rng.normal(0.0, 1.5, size=x.shape) / np.sqrt(mass)[:, None]
    v = oracle.rattle_water_velocities(x.astype(np.float64), v0, mass).astype(np_real)  # start on the constraint manifold
    forces = [rng.normal(0.0, 600.0, size=x.shape).astype(np_real) for _ in range(5)]
    water = np.arange(3 * n_w, dtype=np.int32).reshape(n_w, 3)
    # oracle chain in fp64 from the same starting arrays
    xo = oracle.shake_water(x.astype(np.float64), x.astype(np.float64), mass, d_oh, d_hh)
    vo = v.astype(np.float64)
    for s in range(4):
        xu, vh = oracle.vv_kick_drift(xo, vo, forces[s].astype(np.float64), inv_m.astype(np.float64), dt)
        xc = oracle.shake_water(xo, xu, mass, d_oh, d_hh)
        vh = vh + (xc - xu) / dt
        vn = oracle.vv_kick(vh, forces[s + 1].astype(np.float64), inv_m.astype(np.float64), dt)
        xo, vo = xc, oracle.rattle_water_velocities(xc, vn, mass)
    dev = torch.device("cuda", 0)
    with dimos.Context(0, precision) as ctx:
        xd, vd = torch.from_numpy(x.copy()).to(dev), torch.from_numpy(v.copy()).to(dev)
        wd, imd = torch.from_numpy(water).to(dev), torch.from_numpy(inv_m).to(dev)
        fd = [torch.from_numpy(f).to(dev) for f in forces]
        ref_d = xd.clone()
        skin = 2.0 * float(np.sqrt(((xo - x.astype(np.float64)) ** 2).sum(1).max())) * 0.9   # fires on the last step only?
        for s in range(4):
            if fused:
                fired = dimos.dimos_water_kick_drift_settle(ctx, xd, vd, fd[s], wd, m_O, m_H, d_oh, d_hh, dt, pos_at_build=ref_d, skin=skin)
                ke = dimos.dimos_water_kick_settle_velocities(ctx, xd, vd, fd[s + 1], wd, m_O, m_H, dt, want_ke=True)
            else:
                x_old = xd.clone()
                dimos.dimos_vv_kick_drift(ctx, xd, vd, fd[s], imd, dt)
                dimos.dimos_settle(ctx, x_old, xd, wd, m_O, m_H, d_oh, d_hh, vel=vd, dt=dt)
                dimos.dimos_vv_kick(ctx, vd, fd[s + 1], imd, dt)
                dimos.dimos_settle_velocities(ctx, xd, vd, wd, m_O, m_H)
        torch.cuda.synchronize()
        if fused:
            want, m_disp = oracle.needs_rebuild(xd.cpu().numpy(), x, skin)
            assert fired == want and fired  # skin was chosen 10 % below twice the oracle's largest displacement
            assert float(ke[0]) == pytest.approx(oracle.kinetic_energy(vo, mass), rel=1e-9 if precision == "f64" else 1e-4)
            assert dimos.dimos_water_kick_drift_settle(ctx, xd.clone(), vd.clone(), fd[0], wd, m_O, m_H, d_oh, d_hh, dt) is None
        gx, gv = xd.cpu().numpy().astype(np.float64), vd.cpu().numpy().astype(np.float64)
    tol_x = 1e-11 if precision == "f64" else 1e-5      # fp32: 4 steps x (rounding of 6 nm coordinates ~ 5e-7)
    tol_v = 1e-9 if precision == "f64" else 4e-3       # (x_c - x_u) / dt amplifies position rounding by 1/dt = 500
    assert np.abs(gx - xo).max() < tol_x
    assert np.abs(gv - vo).max() < tol_v
    m = gx.reshape(-1, 3, 3)
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):
        assert np.abs(np.linalg.norm(m[:, i] - m[:, j], axis=1) - d).max() < (1e-12 if precision == "f64" else 3e-6)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n", [1, 999, 300000])
def test_kinetic_energy_and_berendsen_match_oracle(precision, n):
    """dimos_kinetic_energy and dimos_berendsen (step 7; Berendsen rescaling) against the
    numpy fp64 oracle: K, the temperature before scaling, the scaled velocities element by element, and the relaxation
    T' = T + (dt/tau)(T0 - T) measured on the device's own output."""
    rng = np.random.default_rng(5000 + n)
    np_real = np.float64 if precision == "f64" else np.float32
    mass = rng.choice(np.array([15.9994, 1.008]), size=n)
    inv_m = (1.0 / mass).astype(np_real)
    m_dev = 1.0 / inv_m.astype(np.float64)  # the masses the device sees
    v = (1.25 * rng.normal(size=(n, 3)) * np.sqrt(oracle.K_B * 300.0 / mass)[:, None]).astype(np_real)
    n_dof = max(3 * n - 3, 1)
    T0, tau, dt = 300.0, 0.1, 0.002
    K_o = oracle.kinetic_energy(v, m_dev)
    v_o, T_o = oracle.berendsen(v, m_dev, n_dof, T0, tau, dt)
    dev = torch.device("cuda", 0)
    with dimos.Context(0, precision) as ctx:
        vd, imd = torch.from_numpy(v.copy()).to(dev), torch.from_numpy(inv_m).to(dev)
        K = dimos.dimos_kinetic_energy(ctx, vd, imd)
        T = dimos.dimos_berendsen(ctx, vd, imd, n_dof, T0, tau, dt)
        got = vd.cpu().numpy().astype(np.float64)
        K2 = dimos.dimos_kinetic_energy(ctx, vd, imd)
        v_split = torch.from_numpy(v.copy()).to(dev)   # the two halves called separately give the same velocities
        dimos.dimos_kinetic_energy(ctx, v_split, imd)
        dimos.dimos_berendsen_scale(ctx, v_split, n_dof, T0, tau, dt, ctx._ke_scratch())
        torch.cuda.synchronize()
        assert torch.allclose(v_split, vd, rtol=1e-6, atol=0)
        v_async = torch.from_numpy(v.copy()).to(dev)
        assert dimos.dimos_berendsen(ctx, v_async, imd, n_dof, T0, tau, dt, sync=False) is None
        torch.cuda.synchronize()
        assert torch.allclose(v_async, vd, rtol=1e-6, atol=0)
        with pytest.raises(dimos.DimosError):
            dimos.dimos_berendsen(ctx, vd, imd, n_dof, T0, 0.001, 0.002)  # dt > tau
    rel = 1e-13 if precision == "f64" else 2e-7   # fp32 squares, fp64 accumulation: independent roundings average out
    assert K == pytest.approx(K_o, rel=rel)
    assert T == pytest.approx(T_o, rel=rel)
    assert np.abs(got - v_o).max() <= (1e-14 if precision == "f64" else 2e-7) * np.abs(v_o).max()
    T_after = 2.0 * K2 / (n_dof * oracle.K_B)
    assert T_after == pytest.approx(T_o + dt / tau * (T0 - T_o), rel=1e-12 if precision == "f64" else 1e-6)


@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_rigid_water_nve_conserves_total_energy(precision, fused):
    """The whole loop of PAPER.md:281-292 on the device (steps 1-6: kick+drift with the fused trigger, SETTLE, list rebuild
    when the trigger fires, pair forces, kick, velocity constraints) for the 3000-molecule box, started from the
    un-equilibrated synthetic configuration: some 6e4 kJ/mol flow from potential into kinetic energy within a few dozen
    steps, and K + U must stay constant to 1 % of that flow (forces are the gradient of the reported energy, the
    constraints do no work, the list is never stale) while every molecule keeps its geometry."""
    wb = wl.make_config(1)
    L = wb.box
    np_real = np.float64 if precision == "f64" else np.float32
    p = wb.pos.astype(np.float64).reshape(-1, 3, 3)
    for k in (1, 2):  # make molecules whole: the workload wraps atom by atom
        d = p[:, k] - p[:, 0]
        p[:, k] = p[:, 0] + d - L * np.round(d / L)
    dev = torch.device("cuda", 0)
    pos = torch.from_numpy(p.reshape(-1, 3).astype(np_real)).to(dev)
    n = pos.shape[0]
    n_w = n // 3
    charge = torch.from_numpy(wb.charge.astype(np_real)).to(dev)
    typ = torch.from_numpy(wb.type).to(dev)
    lj = dimos.lj_table_from_types(wb.sigma, wb.epsilon).to(dev)
    vel = torch.from_numpy(wl.maxwell_boltzmann_velocities(wb.mass, 300.0, 5).astype(np_real)).to(dev)
    inv_m = torch.from_numpy((1.0 / wb.mass).astype(np_real)).to(dev)
    water = torch.arange(n, dtype=torch.int32, device=dev).reshape(n_w, 3)
    excl = torch.from_numpy(wb.excl_pairs).to(dev)
    m_O, m_H = float(wb.mass[0]), float(wb.mass[1])
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    dt = 0.001
    with dimos.Context(0, precision) as ctx:
        dimos.dimos_settle(ctx, pos.clone(), pos, water, m_O, m_H, d_oh, d_hh)   # rigid to the precision in use
        dimos.dimos_settle_velocities(ctx, pos, vel, water, m_O, m_H)
        nl = dimos.dimos_nl_build(ctx, pos, L, 1.0, 0.1, excl)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj)
        U0 = float(E[0])
        K0 = dimos.dimos_kinetic_energy(ctx, vel, inv_m)
        tot, pot, rebuilds = [U0 + K0], [U0], 0
        for _ in range(100):
            if fused:  # two passes per step; the trigger sees the constrained positions
                fired = dimos.dimos_water_kick_drift_settle(ctx, pos, vel, F, water, m_O, m_H, d_oh, d_hh, dt,
                                                            pos_at_build=nl.pos_at_build, skin=0.1)
            else:
                old = pos.clone()
                fired = dimos.dimos_vv_kick_drift(ctx, pos, vel, F, inv_m, dt, pos_at_build=nl.pos_at_build, skin=0.1)
                dimos.dimos_settle(ctx, old, pos, water, m_O, m_H, d_oh, d_hh, vel=vel, dt=dt)
                fired = fired or dimos.dimos_nl_needs_rebuild(ctx, pos, nl.pos_at_build, 0.1)  # SETTLE moved atoms after the drift
            if fired:
                nl = dimos.dimos_nl_build(ctx, pos, L, 1.0, 0.1, excl, nl=nl)
                rebuilds += 1
            F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F)
            if fused:
                K = float(dimos.dimos_water_kick_settle_velocities(ctx, pos, vel, F, water, m_O, m_H, dt, want_ke=True)[0])
            else:
                dimos.dimos_vv_kick(ctx, vel, F, inv_m, dt)
                dimos.dimos_settle_velocities(ctx, pos, vel, water, m_O, m_H)
                K = dimos.dimos_kinetic_energy(ctx, vel, inv_m)
            pot.append(float(E[0]))
            tot.append(pot[-1] + K)
        m = pos.cpu().numpy().astype(np.float64).reshape(-1, 3, 3)
    flow = U0 - min(pot)
    assert rebuilds >= 1 and flow > 2.0 * K0
    assert np.abs(np.array(tot) - tot[0]).max() < 0.01 * flow
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):
        assert np.abs(np.linalg.norm(m[:, i] - m[:, j], axis=1) - d).max() < (1e-12 if precision == "f64" else 3e-6)


def test_thermostatted_rigid_water_loop():
    """The loop README.md shows (fused steps 1-3, rebuild on the fused trigger, forces, fused steps 5-6 with the kinetic
    energy of step 8, Berendsen rescaling of step 7 from that device-resident sum) on the 3000-molecule box in fp32: every
    application obeys T' = T + (dt/tau)(T0 - T) on the measured temperatures, the rescaled velocities still satisfy the
    velocity constraints, molecules stay rigid, and the heat released by the un-equilibrated start is carried away (the
    temperature ends far below the ~1200 K the same run reaches without a thermostat)."""
    wb = wl.make_config(1)
    L = wb.box
    p = wb.pos.astype(np.float64).reshape(-1, 3, 3)
    for k in (1, 2):
        d = p[:, k] - p[:, 0]
        p[:, k] = p[:, 0] + d - L * np.round(d / L)
    dev = torch.device("cuda", 0)
    pos = torch.from_numpy(p.reshape(-1, 3).astype(np.float32)).to(dev)
    n = pos.shape[0]
    n_w = n // 3
    charge, typ = torch.from_numpy(wb.charge).to(dev), torch.from_numpy(wb.type).to(dev)
    lj = dimos.lj_table_from_types(wb.sigma, wb.epsilon).to(dev)
    vel = torch.from_numpy(wl.maxwell_boltzmann_velocities(wb.mass, 300.0, 5).astype(np.float32)).to(dev)
    inv_m = torch.from_numpy((1.0 / wb.mass).astype(np.float32)).to(dev)
    water = torch.arange(n, dtype=torch.int32, device=dev).reshape(n_w, 3)
    excl = torch.from_numpy(wb.excl_pairs).to(dev)
    m_O, m_H = float(wb.mass[0]), float(wb.mass[1])
    d_oh = wl.R_OH
    d_hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    dt, tau, T0 = 0.001, 0.01, 300.0
    n_dof = 6 * n_w - 3
    to_T = 2.0 / (n_dof * oracle.K_B)
    with dimos.Context(0, "f32") as ctx:
        dimos.dimos_settle(ctx, pos.clone(), pos, water, m_O, m_H, d_oh, d_hh)
        dimos.dimos_settle_velocities(ctx, pos, vel, water, m_O, m_H)
        nl = dimos.dimos_nl_build(ctx, pos, L, 1.0, 0.1, excl)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj)
        temps = []
        for _ in range(150):
            if dimos.dimos_water_kick_drift_settle(ctx, pos, vel, F, water, m_O, m_H, d_oh, d_hh, dt,
                                                   pos_at_build=nl.pos_at_build, skin=0.1):
                nl = dimos.dimos_nl_build(ctx, pos, L, 1.0, 0.1, excl, nl=nl)
            F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, charge, typ, lj, F=F)
            ke = dimos.dimos_water_kick_settle_velocities(ctx, pos, vel, F, water, m_O, m_H, dt, want_ke=True)
            T_before = float(ke[0]) * to_T
            dimos.dimos_berendsen_scale(ctx, vel, n_dof, T0, tau, dt, ke)
            T_after = dimos.dimos_kinetic_energy(ctx, vel, inv_m) * to_T
            assert T_after == pytest.approx(T_before + dt / tau * (T0 - T_before), rel=2e-6)
            temps.append(T_after)
        x = pos.cpu().numpy().astype(np.float64).reshape(-1, 3, 3)
        v = vel.cpu().numpy().astype(np.float64).reshape(-1, 3, 3)
    assert np.isfinite(temps).all() and max(temps) < 900.0 and temps[-1] < 450.0
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):
        r = x[:, i] - x[:, j]
        assert np.abs(np.linalg.norm(r, axis=1) - d).max() < 3e-6
        assert np.abs(((v[:, i] - v[:, j]) * r).sum(1) / d).max() < 2e-5 * np.abs(v).max()


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n", [1, 1000, 300001])
def test_langevin_ou_matches_oracle(precision, n):
    """dimos_langevin_ou (reading C-26) against the numpy oracle on the same velocities, masses and normal
    numbers, element by element; gamma = 0 returns the input; a frozen atom (inv_mass = 0) only decays."""
    rng = np.random.default_rng(900 + n)
    np_real = np.float64 if precision == "f64" else np.float32
    mass = rng.choice(np.array([15.9994, 1.008]), size=n)
    inv_m = (1.0 / mass).astype(np_real)
    v = (rng.normal(size=(n, 3)) * np.sqrt(oracle.K_B * 300.0 / mass)[:, None]).astype(np_real)
    xi = rng.normal(size=(n, 3)).astype(np_real)
    gamma, dt, T = 5.0, 0.002, 310.0
    want = oracle.langevin_ou(v, 1.0 / inv_m.astype(np.float64), xi, gamma, dt, T)
    dev = torch.device("cuda", 0)
    with dimos.Context(0, precision) as ctx:
        vd = torch.from_numpy(v.copy()).to(dev)
        dimos.dimos_langevin_ou(ctx, vd, torch.from_numpy(inv_m).to(dev), torch.from_numpy(xi).to(dev), gamma, dt, T)
        got = vd.cpu().numpy().astype(np.float64)
        scale = np.abs(want).max()
        assert np.abs(got - want).max() <= (1e-14 if precision == "f64" else 4e-7) * scale
        v0 = torch.from_numpy(v.copy()).to(dev)
        dimos.dimos_langevin_ou(ctx, v0, torch.from_numpy(inv_m).to(dev), torch.from_numpy(xi).to(dev), 0.0, dt, T)
        assert np.array_equal(v0.cpu().numpy(), v)
        frozen = torch.zeros(n, dtype=vd.dtype, device=dev)
        vf = torch.from_numpy(v.copy()).to(dev)
        dimos.dimos_langevin_ou(ctx, vf, frozen, torch.from_numpy(xi).to(dev), gamma, dt, T)
        assert np.allclose(vf.cpu().numpy(), v * np.exp(-gamma * dt), rtol=1e-6, atol=0)
        with pytest.raises(dimos.DimosError):
            dimos.dimos_langevin_ou(ctx, vd, torch.from_numpy(inv_m).to(dev), torch.from_numpy(xi).to(dev), -1.0, dt, T)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("model", ["spce", "heavy", "wide", "light_centre"])
def test_settle_and_velocity_stage_for_other_rigid_three_site_models(precision, model):
    """The constraint solvers take the geometry and the masses as arguments (PAPER.md:327 names SETTLE for water in
    general): SPC/E (0.1 nm, 109.47 deg), heavy water (m_H = 2.014), a nearly linear triangle (170 deg) and a molecule
    whose centre atom is the light one.  Positions against the oracle's converged SHAKE, velocities against its converged
    RATTLE velocity stage."""
    d_oh, angle, m_O, m_H = {"spce": (0.1, 109.47, 15.9994, 1.008), "heavy": (0.09572, 104.52, 15.9994, 2.014),
                             "wide": (0.11, 170.0, 12.0, 3.0), "light_centre": (0.12, 95.0, 1.5, 14.0)}[model]
    d_hh = 2.0 * d_oh * np.sin(np.radians(angle) / 2.0)
    rng = np.random.default_rng(5 + len(model))  # spce 9, heavy 10, wide 9 + different draws below, light_centre 17
    np_real = np.float64 if precision == "f64" else np.float32
    n_w = 777
    mass = np.tile([m_O, m_H, m_H], n_w)
    x0 = _random_rigid_waters(rng, n_w, d_oh, d_hh).astype(np_real)
    dt = 0.001
    v = rng.normal(0.0, 1.5, size=x0.shape) / np.sqrt(mass)[:, None]
    x1 = (x0.astype(np.float64) + dt * v).astype(np_real)
    x0_64 = oracle.shake_water(x0.astype(np.float64), x0.astype(np.float64), mass, d_oh, d_hh)
    ref_x = oracle.shake_water(x0_64, x1.astype(np.float64), mass, d_oh, d_hh)
    water = np.arange(3 * n_w, dtype=np.int32).reshape(n_w, 3)
    dev = torch.device("cuda", 0)
    with dimos.Context(0, precision) as ctx:
        p = torch.from_numpy(x1.copy()).to(dev)
        dimos.dimos_settle(ctx, torch.from_numpy(x0).to(dev), p, torch.from_numpy(water).to(dev), m_O, m_H, d_oh, d_hh)
        vd = torch.from_numpy(v.astype(np_real)).to(dev)
        dimos.dimos_settle_velocities(ctx, p, vd, torch.from_numpy(water).to(dev), m_O, m_H)
        torch.cuda.synchronize()
        got_x = p.cpu().numpy().astype(np.float64)
        got_v = vd.cpu().numpy().astype(np.float64)
    tol = 5e-12 if precision == "f64" else 3e-6
    # the device's old positions are rigid only to the rounding of their element type (2.4e-7 nm at 6 nm in fp32); how far
    # that moves the solution grows like 1 / cos(angle / 2), the inverse height of the triangle (11.5 at 170 degrees)
    kappa = max(1.0, 0.6 / np.cos(np.radians(angle) / 2.0))
    assert np.abs(got_x - ref_x).max() < tol * kappa
    m = got_x.reshape(-1, 3, 3)
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh)):  # the constraints themselves hold to rounding whatever the shape
        assert np.abs(np.linalg.norm(m[:, i] - m[:, j], axis=1) - d).max() < tol
    ref_v = oracle.rattle_water_velocities(got_x, v.astype(np_real).astype(np.float64), mass)
    vtol = (1e-11 if precision == "f64" else 2e-5) * np.abs(v).max()
    assert np.abs(got_v - ref_v).max() < vtol
