"""`-m gpu`: out-of-bounds-write check of the library's workspace.  compute-sanitizer is closed on this pool (its runs left
GPUs needing a reset; the refusal is recorded in profiles/r2_sanitizer.md), so the check SURVEY.md §5 asked of it is done
with the allocator callback the C ABI already has: every block the library allocates gets 4 KiB of 0xA5 on both sides, the
whole path runs (both pair kernels, Ewald, fp64, exceptions, export, rebuilds in place with growing rows, integrator, PME),
and no guard byte may have changed.  The pair kernels' reads past a row's end stay inside their allocation by design
(LIST_SLACK in csrc/common.cuh, clamped slot indices): reads cannot be caught this way, writes are."""
import numpy as np
import pytest
import torch

from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", ["f32", "mixed", "f64"])
def test_no_workspace_block_is_written_out_of_bounds(precision):
    real = torch.float64 if precision == "f64" else torch.float32
    ctx = dimos.Context(0, precision, guard_bytes=4096)
    try:
        for index, rc, method in ((0, 0.9, "rf"), (1, 1.0, "rf"), (1, 1.0, "ewald")):
            wb = wl.make_config(index)
            pos = torch.from_numpy(wb.pos).to("cuda", real)
            q = torch.from_numpy(wb.charge).to("cuda", real)
            typ = torch.from_numpy(wb.type).cuda()
            excl = torch.from_numpy(wb.excl_pairs).cuda()
            lj = dimos.lj_table_from_types(wb.sigma, wb.epsilon).cuda()
            nl = dimos.dimos_nl_build(ctx, pos, wb.box, rc, 0.1, excl)
            dimos.dimos_nl_set_exceptions(ctx, nl, excl[:7].contiguous(), torch.full((7, 2), 0.5, dtype=torch.float64, device="cuda"))
            for k in range(3):
                F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, q, typ, lj, method=method, r_switch=0.8 if k == 2 else 0.0)
                # squeeze the box contents together and rebuild in place: denser rows, the row capacity has to grow
                pos = (pos * 0.93).contiguous()
                nl = dimos.dimos_nl_build(ctx, pos, wb.box, rc, 0.1, excl, nl=nl)
            dimos.dimos_nl_export_pairs(ctx, nl)
            dimos.dimos_nl_export_edges(ctx, nl, rc)
            assert torch.isfinite(F).all() and torch.isfinite(E).all()
            if index == 1:
                vel = torch.zeros_like(pos)
                water = torch.arange(wb.n_atoms, dtype=torch.int32, device="cuda").reshape(-1, 3)
                fresh = torch.from_numpy(wb.pos).to("cuda", real)
                dimos.dimos_water_kick_drift_settle(ctx, fresh, vel, F, water, 15.9994, 1.008, wl.R_OH, 0.15139, 0.001,
                                                    pos_at_build=nl.pos_at_build, skin=0.1)
                dimos.dimos_pme_recip(ctx, fresh, q, wb.box, 3.12, (45, 48, 50), order=5)
                dimos.dimos_pme_recip(ctx, fresh, q, wb.box, 3.12, (32, 32, 36), order=6)
        torch.cuda.synchronize()
        assert ctx.check_guards() == []
    finally:
        ctx.close()
    assert ctx._guard_violations == []


def test_the_guard_check_itself_detects_a_stray_write():
    ctx = dimos.Context(0, "f32", guard_bytes=256)
    try:
        wb = wl.make_config(0)
        pos = torch.from_numpy(wb.pos).cuda()
        dimos.dimos_nl_build(ctx, pos, wb.box, 0.9, 0.1, torch.from_numpy(wb.excl_pairs).cuda())
        t = next(iter(ctx._blocks.values()))
        t[t.numel() - 3] = 0  # one byte of a trailing guard
        assert len(ctx.check_guards()) == 1
    finally:
        ctx.close()


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_every_allocation_failure_is_reported_and_leaves_the_context_usable(precision):
    """The dimos_allocator callback returns NULL at the k-th request, for every k until the whole sequence (list build,
    force call, exceptions, PME, in-place rebuild) succeeds: each failure must come back as DIMOS_ENOMEM (-3) -- no crash, no
    other status -- and afterwards the same calls on the same context must succeed and agree with the oracle."""
    import oracle
    from gpu_harness import BAND, DeviceBox, METHOD, check_nonbonded
    from oracle import pme_oracle as pme

    wb = wl.make_config(1)
    db = DeviceBox(wb, precision)
    dev = db.pos.device
    exc = torch.from_numpy(wb.excl_pairs[:50].copy()).to(dev)
    scale = torch.full((50, 2), 0.5, dtype=torch.float64, device=dev)
    mesh = (30, 32, 36)
    ctx = dimos.Context(0, precision)

    def sequence():
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        try:
            dimos.dimos_nl_set_exceptions(ctx, nl, exc, scale)
            out = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method="ewald")
            rec = dimos.dimos_pme_recip(ctx, db.pos, db.charge, db.box, 3.12, mesh, order=5)
            nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl, nl=nl)
            torch.cuda.synchronize()
            return out, rec
        finally:
            ctx.lib.dimos_nl_destroy(ctx.handle, nl.handle)

    try:
        failures = 0
        for k in range(400):
            ctx.fail_alloc_after = k
            try:
                out, rec = sequence()
                break
            except dimos.DimosError as err:
                assert err.args[0].endswith("(status -3)"), err.args[0]
                failures += 1
            finally:
                ctx.fail_alloc_after = None
        else:
            raise AssertionError("the sequence never completed")
        assert failures >= 10, failures  # the sequence makes dozens of requests
        out, rec = sequence()  # and once more with a healthy allocator
        F, E, W = out
        pos64 = db.pos.double().cpu().numpy()
        orc = oracle.nonbonded(pos64, db.charge.double().cpu().numpy(), wb.type, db.lj_np, db.box, 1.0, method=METHOD["ewald"],
                               excl_pairs=wb.excl_pairs, band=BAND, exceptions=(wb.excl_pairs[:50], np.full((50, 2), 0.5)))
        check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
        U0, _, _ = pme.pme_recip(pos64, db.charge.double().cpu().numpy(), db.box, 3.12, mesh, 5)
        assert abs(float(rec[1][0]) - U0) <= (1e-10 if precision == "f64" else 1e-5) * abs(U0)
    finally:
        ctx.close()
