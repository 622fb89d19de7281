"""`-m gpu`: dimos_pme_recip (smooth PME reciprocal space + self energy) against the numpy oracle
oracle/pme_oracle.py on the same seeded inputs: the same mesh, order and alpha on both sides, so what is compared is the
arithmetic of the mesh method (fp32: energy 1e-5 relative, forces 1e-4 RMS(F_recip), virial 1e-4 max|W|; fp64: 1e-10)."""
import numpy as np
import pytest
import torch

from oracle import pme_oracle as pme
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f32": (1e-5, 1e-4, 1e-4), "f64": (1e-10, 1e-10, 1e-9)}


def run(pos, q, box, alpha, mesh, order, precision, accumulate=False):
    real = torch.float64 if precision == "f64" else torch.float32
    ctx = dimos.Context(0, precision)
    try:
        dp = torch.from_numpy(np.ascontiguousarray(pos)).to("cuda", real)
        dq = torch.from_numpy(np.ascontiguousarray(q)).to("cuda", real)
        F0 = None
        if accumulate:
            F0 = torch.full((len(q), 3), 2.5, dtype=real, device="cuda")
        F, E, W = dimos.dimos_pme_recip(ctx, dp, dq, box, alpha, mesh, order=order, F=F0, accumulate=accumulate)
        torch.cuda.synchronize()
        return F.double().cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), dp.double().cpu().numpy(), dq.double().cpu().numpy()
    finally:
        ctx.close()


def compare(F, E, W, ref, precision, q, alpha):
    U0, F0, W0 = ref
    e_tol, f_tol, w_tol = TOL[precision]
    assert abs(E[0] - U0) <= e_tol * abs(U0), (E[0], U0)
    assert abs(E[1] - pme.ewald_self(q, alpha)) <= 1e-12 * abs(E[1]) + 1e-12
    rms = np.sqrt((F0**2).sum(axis=1).mean())
    dF = np.sqrt(((F - F0) ** 2).sum(axis=1)).max()
    assert dF <= f_tol * rms, (dF, rms)
    assert np.abs(W - W0).max() <= w_tol * np.abs(W0).max()
    return dF / rms


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("order", [4, 5, 6])
def test_pme_recip_water216_matches_oracle(precision, order):
    wb = wl.make_config(0)  # 648 atoms, L = 1.8621
    mesh = (20, 24, 21)     # mixed radices, several mesh cells per atom support, wraps on every axis
    F, E, W, p64, q64 = run(wb.pos, wb.charge, wb.box, 3.12, mesh, order, precision)
    compare(F, E, W, pme.pme_recip(p64, q64, wb.box, 3.12, mesh, order), precision, q64, 3.12)


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_pme_recip_2000_waters_heuristic_mesh_unwrapped_positions(precision):
    """6,000 atoms, the paper's mesh heuristic for alpha = 3.12 <-> delta = 2.96e-5, positions shifted out
    of the box; forces accumulated onto an existing array."""
    wb = wl.make_scaled(2000, seed=wl.SEED_BASE + 4, method="ewald")
    mesh = dimos.dimos_pme_mesh_size(3.12, wb.box, 2.96e-5)
    assert mesh == tuple(int(k) for k in mesh) and all(k >= 66 for k in mesh)
    pos = wb.pos.astype(np.float64) + np.array([3.0, -7.5, 11.25])
    pos = pos.astype(np.float32 if precision == "f32" else np.float64)
    F, E, W, p64, q64 = run(pos, wb.charge, wb.box, 3.12, mesh, 5, precision, accumulate=True)
    compare(F - 2.5, E, W, pme.pme_recip(p64, q64, wb.box, 3.12, mesh, 5), precision, q64, 3.12)


def test_pme_mesh_size_heuristic_and_bad_arguments():
    box = np.array([14.41289, 14.41289, 14.41289])
    want = int(np.ceil(2 * 3.12 * box[0] / (3 * 2.96e-5**0.2)))
    m = dimos.dimos_pme_mesh_size(3.12, box, 2.96e-5)
    assert all(k >= want and k < want + 16 for k in m)
    for k in m:
        r = k
        for f in (2, 3, 5, 7):
            while r % f == 0:
                r //= f
        assert r == 1
    ctx = dimos.Context(0, "f32")
    try:
        p = torch.zeros((10, 3), device="cuda")
        q = torch.zeros(10, device="cuda")
        for bad in (dict(mesh=(4, 32, 32)), dict(mesh=(32, 32, 32), order=7), dict(mesh=(32, 32, 32), alpha=0.0)):
            kw = dict(mesh=(32, 32, 32), order=5, alpha=3.0)
            kw.update(bad)
            with pytest.raises(dimos.DimosError) as ei:
                dimos.dimos_pme_recip(ctx, p, q, [3.0, 3.0, 3.0], kw["alpha"], kw["mesh"], order=kw["order"])
            assert ei.value.status == -1
    finally:
        ctx.close()


def test_pme_total_ewald_energy_is_independent_of_alpha_f64():
    """Real space (dimos_nonbonded, DIMOS_EWALD_REAL) + reciprocal + self from the library alone: the total does not depend
    on alpha up to the mesh error -- the three terms fit together."""
    wb = wl.make_scaled(300, seed=wl.SEED_BASE + 9, method="ewald")
    ctx = dimos.Context(0, "f64")
    try:
        pos = torch.from_numpy(wb.pos.astype(np.float64)).cuda()
        q = torch.from_numpy(wb.charge.astype(np.float64)).cuda()
        typ = torch.from_numpy(wb.type).cuda()
        excl = torch.from_numpy(wb.excl_pairs).cuda()
        lj = dimos.lj_table_from_types(wb.sigma, wb.epsilon).cuda()
        rc = 0.5 * float(min(wb.box)) - 1e-6
        nl = dimos.dimos_nl_build(ctx, pos, wb.box, rc, 0.0, excl)
        totals, scale = [], 0.0
        for alpha in (4.5, 5.5):
            F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, q, typ, lj, method="ewald", alpha=alpha)
            Fr, Er, Wr = dimos.dimos_pme_recip(ctx, pos, q, wb.box, alpha, (72, 72, 72), order=6)
            totals.append(float(E[2] + E[3] + Er[0] + Er[1]))
            scale = max(scale, abs(float(Er[1])))
        # the total is a small difference of large terms (|U_self| ~ 1e5 kJ/mol here): compare on that scale
        assert abs(totals[1] - totals[0]) <= 2e-7 * scale, (totals, scale)
    finally:
        ctx.close()


def test_pme_recip_config4_full_size_f32():
    """configs[4] (300,000 atoms) with the mesh bench.py times (the paper's heuristic): the whole force array,
    energy and virial against the numpy oracle."""
    wb = wl.make_config(4)
    delta = float(np.exp(-(3.12 * 1.0) ** 2) / 2.0)
    mesh = dimos.dimos_pme_mesh_size(3.12, wb.box, delta)
    F, E, W, p64, q64 = run(wb.pos, wb.charge, wb.box, 3.12, mesh, 5, "f32")
    compare(F, E, W, pme.pme_recip(p64, q64, wb.box, 3.12, mesh, 5), "f32", q64, 3.12)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("order", [3, 5])
def test_pme_recip_orthorhombic_box_and_mesh(precision, order):
    """Box edges 2.1 x 3.3 x 2.7 nm and a mesh of 21 x 36 x 25 points (odd sizes included: the half spectrum of the
    real-to-complex transform then has no Nyquist plane): 700 point charges, neutral, at random positions, a tail of 21
    atoms beyond the last full warp of 32."""
    rng = np.random.default_rng(17)
    n = 32 * 21 + 21 + 7
    box = np.array([2.1, 3.3, 2.7])
    pos = rng.uniform(0.0, 1.0, size=(n, 3)) * box
    q = rng.uniform(-1.0, 1.0, size=n)
    q -= q.mean()
    if precision == "f32":
        pos, q = pos.astype(np.float32), q.astype(np.float32)
    mesh = (21, 36, 25)
    F, E, W, p64, q64 = run(pos, q, box, 3.0, mesh, order, precision)
    compare(F, E, W, pme.pme_recip(p64, q64, box, 3.0, mesh, order), precision, q64, 3.0)


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_pme_plan_is_rebuilt_when_mesh_order_or_system_change_within_one_context(precision):
    """One context, a sequence of calls with different meshes, spline orders, boxes, Ewald parameters and atom counts (the
    cuFFT plans, the mesh and the per-axis tables are cached in the context and must follow), each against the oracle."""
    real = torch.float64 if precision == "f64" else torch.float32
    rng = np.random.default_rng(23)
    ctx = dimos.Context(0, precision)
    try:
        for n, box, alpha, mesh, order in [(300, (2.0, 2.0, 2.0), 3.0, (20, 20, 20), 5), (300, (2.0, 2.0, 2.0), 3.0, (32, 30, 28), 5),
                                           (1000, (2.0, 2.6, 3.1), 2.6, (32, 30, 28), 4), (300, (2.0, 2.0, 2.0), 3.4, (20, 20, 20), 6),
                                           (300, (2.2, 2.0, 2.0), 3.4, (20, 20, 20), 6)]:
            box = np.array(box)
            pos = rng.uniform(0.0, 1.0, size=(n, 3)) * box
            q = rng.uniform(-1.0, 1.0, size=n)
            q -= q.mean()
            dp = torch.from_numpy(pos).to("cuda", real)
            dq = torch.from_numpy(q).to("cuda", real)
            F, E, W = dimos.dimos_pme_recip(ctx, dp, dq, box, alpha, mesh, order=order)
            torch.cuda.synchronize()
            p64, q64 = dp.double().cpu().numpy(), dq.double().cpu().numpy()
            compare(F.double().cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), pme.pme_recip(p64, q64, box, alpha, mesh, order),
                    precision, q64, alpha)
    finally:
        ctx.close()
