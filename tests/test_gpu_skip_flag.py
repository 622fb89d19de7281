"""dimos_nb_params.skip_flag: the force call enqueued behind the rebuild trigger without a host
round trip.  If the device flag is set when the kernels run, the call must leave F, E and the virial untouched; if it is
clear, the call is the ordinary force call (compared with the oracle).  Covers the three pair kernels (packed fp32,
generic fp32 with fp64 accumulation, rolled fp64), the Ewald exclusion correction and the 1-4 exception kernel."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

from gpu_harness import BAND, METHOD, DeviceBox, check_nonbonded

pytestmark = pytest.mark.gpu


def _sentinels(db):
    F = torch.full_like(db.pos, 7.25)
    E = torch.full((4,), -3.5, dtype=torch.float64, device=db.pos.device)
    W = torch.full((3, 3), 11.0, dtype=torch.float64, device=db.pos.device)
    return F, E, W


@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f32", "ewald"), ("mixed", "rf"), ("f64", "ewald")])
def test_skip_flag_set_leaves_outputs_untouched_and_clear_is_the_plain_call(precision, method):
    wb = wl.make_config(1)  # 9,000 atoms: >= 3 cells per axis, the kernels bench.py times
    db = DeviceBox(wb, precision)
    n = wb.n_atoms
    exc_pairs = np.array([[3 * k, 3 * k + 1] for k in range(0, 40, 2)], dtype=np.int32)  # O-H pairs: excluded, so legal exceptions
    exc_scale = np.tile(np.array([[0.5, 0.8333]]), (len(exc_pairs), 1))
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        dimos.dimos_nl_set_exceptions(ctx, nl, torch.from_numpy(exc_pairs).to(db.pos.device), torch.from_numpy(exc_scale).to(db.pos.device))
        flag = torch.ones(1, dtype=torch.int32, device=db.pos.device)
        F, E, W = _sentinels(db)
        F0, E0, W0 = F.clone(), E.clone(), W.clone()
        dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method=method, F=F, E=E, virial=W, skip_flag=flag)
        torch.cuda.synchronize()
        assert torch.equal(F, F0) and torch.equal(E, E0) and torch.equal(W, W0)
        # a skipped call leaves the list's state usable: the next (unconditional or clear-flag) call is correct
        flag.zero_()
        dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method=method, F=F, E=E, virial=W, skip_flag=flag)
        torch.cuda.synchronize()
        pos64 = db.pos.double().cpu().numpy()
        orc = oracle.nonbonded(pos64, db.charge.double().cpu().numpy(), wb.type, db.lj_np, db.box, 1.0, method=METHOD[method],
                               excl_pairs=wb.excl_pairs, band=BAND, exceptions=(exc_pairs, exc_scale))
        check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
        # set again after a valid call: the valid results stay
        F1, E1, W1 = F.clone(), E.clone(), W.clone()
        flag.fill_(5)
        dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method=method, F=F, E=E, virial=W, skip_flag=flag)
        torch.cuda.synchronize()
        assert torch.equal(F, F1) and torch.equal(E, E1) and torch.equal(W, W1)
    finally:
        ctx.close()


def test_force_call_enqueued_behind_the_trigger_f32():
    """The protocol bench.py runs: trigger with the flag left on the device, the force call conditional on it, the flag read
    afterwards; when it fired, rebuild and call again.  Every step's forces against the oracle at that step's positions."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    dev = db.pos.device
    vel = wl.maxwell_boltzmann_velocities(wb.mass, 300.0, wl.SEED_BASE + 3).astype(np.float32)
    dstep = torch.from_numpy(vel * 0.004).to(dev)  # 4 fs of ballistic drift per step: the trigger fires every few steps
    pos = db.pos.clone()
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, pos, db.box, 1.0, 0.1, db.excl)
        flag = torch.zeros(1, dtype=torch.int32, device=dev)
        F, E, W = _sentinels(db)
        dimos.dimos_nonbonded(ctx, nl, pos, db.charge, db.type, db.lj, F=F, E=E, virial=W)
        e_scale = abs(float(E[0]))  # the unrelaxed box drifts through E = 0: errors are taken relative to the first frame
        fired = 0
        for step in range(12):
            pos.add_(dstep)
            got = dimos.dimos_nl_needs_rebuild(ctx, pos, nl.pos_at_build, 0.1, sync=False, flag=flag)
            assert got is flag
            dimos.dimos_nonbonded(ctx, nl, pos, db.charge, db.type, db.lj, F=F, E=E, virial=W, skip_flag=flag)
            want, m = oracle.needs_rebuild(pos.cpu().numpy(), nl.pos_at_build.cpu().numpy(), 0.1)
            got = bool(flag.item())
            assert got == want or abs(m - 0.05) < 1e-6
            if got:
                fired += 1
                nl = dimos.dimos_nl_build(ctx, pos, db.box, 1.0, 0.1, db.excl, nl=nl)
                dimos.dimos_nonbonded(ctx, nl, pos, db.charge, db.type, db.lj, F=F, E=E, virial=W)
            orc = oracle.nonbonded(pos.double().cpu().numpy(), wb.charge, wb.type, db.lj_np, db.box, 1.0, excl_pairs=wb.excl_pairs,
                                   band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32", e_floor=e_scale)
        assert 2 <= fired <= 10, fired
    finally:
        ctx.close()


def test_host_entry_points_reject_a_skip_flag():
    wb = wl.make_config(0)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 0.9, 0.1, db.excl)
        flag = torch.zeros(1, dtype=torch.int32, device=db.pos.device)
        prm = ctx._params(nl, "rf", 78.5, 3.12, 138.935456, 0.0, flag)
        h = lambda a: torch.from_numpy(np.ascontiguousarray(a))
        pos, q, t, lj = h(wb.pos.astype(np.float32)), h(wb.charge.astype(np.float32)), h(wb.type), h(db.lj_np)
        F, E, W = torch.empty_like(pos), torch.empty(4, dtype=torch.float64), torch.empty(3, 3, dtype=torch.float64)
        box = (ctypes.c_double * 3)(*[float(x) for x in db.box])
        rc = ctx.lib.dimos_nonbonded_host(ctx.handle, nl.handle, pos.data_ptr(), q.data_ptr(), t.data_ptr(), lj.data_ptr(), lj.shape[0],
                                          box, ctypes.byref(prm), F.data_ptr(), E.data_ptr(), W.data_ptr(), None)
        assert rc == -1  # DIMOS_EINVAL
    finally:
        ctx.close()


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_second_kick_honours_the_skip_flag(precision):
    """dimos_vv_kick and dimos_water_kick_settle_velocities with the device word set leave the velocities untouched (the
    kinetic-energy output is 0); with it clear they are the plain calls, bit for bit."""
    real = torch.float64 if precision == "f64" else torch.float32
    dev = torch.device("cuda", 0)
    n_w = 1000
    g = torch.Generator(device="cpu").manual_seed(5)
    wb = wl.make_scaled(n_w, seed=wl.SEED_BASE + 8)
    pos = torch.from_numpy(wb.pos).to(dev, real)
    vel = torch.randn(3 * n_w, 3, generator=g, dtype=torch.float64).to(dev, real)
    F = (100.0 * torch.randn(3 * n_w, 3, generator=g, dtype=torch.float64)).to(dev, real)
    inv_m = torch.from_numpy(1.0 / wb.mass).to(dev, real)
    water = torch.arange(3 * n_w, dtype=torch.int32, device=dev).reshape(-1, 3)
    m_O, m_H = float(wb.mass[0]), float(wb.mass[1])
    flag = torch.ones(1, dtype=torch.int32, device=dev)
    ctx = dimos.Context(0, precision)
    try:
        v = vel.clone()
        dimos.dimos_vv_kick(ctx, v, F, inv_m, 0.002, skip_flag=flag)
        assert torch.equal(v, vel)
        ke = dimos.dimos_water_kick_settle_velocities(ctx, pos, v, F, water, m_O, m_H, 0.002, want_ke=True, skip_flag=flag)
        assert torch.equal(v, vel) and float(ke.item()) == 0.0
        flag.zero_()
        v_plain, v_flag = vel.clone(), vel.clone()
        dimos.dimos_vv_kick(ctx, v_plain, F, inv_m, 0.002)
        dimos.dimos_vv_kick(ctx, v_flag, F, inv_m, 0.002, skip_flag=flag)
        assert torch.equal(v_plain, v_flag) and not torch.equal(v_plain, vel)
        ke_plain = float(dimos.dimos_water_kick_settle_velocities(ctx, pos, v_plain, F, water, m_O, m_H, 0.002, want_ke=True).item())
        ke_flag = float(dimos.dimos_water_kick_settle_velocities(ctx, pos, v_flag, F, water, m_O, m_H, 0.002, want_ke=True,
                                                                 skip_flag=flag).item())
        assert torch.equal(v_plain, v_flag) and ke_plain > 0.0 and abs(ke_flag - ke_plain) <= 1e-12 * ke_plain
    finally:
        ctx.close()
