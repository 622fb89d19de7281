"""`-m gpu` parity tests: the CUDA path, called through the C ABI, against the CPU fp64 oracle on the same
seeded inputs, element by element (tolerances in tests/gpu_harness.py and DESIGN.md)."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos
from paper_2503_20541_b200 import workloads as wl

from gpu_harness import BAND, METHOD, DeviceBox, check_neighbor_set, check_nonbonded, lj_table_np, run_case

pytestmark = pytest.mark.gpu


# --- A3: rebuild trigger (reading C-5) -----------------------------------------------------
@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n", [1, 5, 1000, 70001])
def test_needs_rebuild_matches_oracle(precision, n):
    rng = np.random.default_rng(n)
    real = np.float64 if precision == "f64" else np.float32
    ref = rng.uniform(0, 5, size=(n, 3)).astype(real)
    ctx = dimos.Context(0, precision)
    skin = 0.1
    try:
        for scale in (0.0, 0.02, 0.0288, 0.0290, 0.05, 1.0):
            step = rng.standard_normal((n, 3))
            step *= scale / np.maximum(np.linalg.norm(step, axis=1, keepdims=True), 1e-30)
            step[rng.integers(0, n)] *= 1.7  # one atom moves furthest
            pos = (ref.astype(np.float64) + step).astype(real)
            want, m = oracle.needs_rebuild(pos, ref, skin)
            got = dimos.dimos_nl_needs_rebuild(ctx, torch.from_numpy(pos).cuda(), torch.from_numpy(ref).cuda(), skin)
            if abs(m - 0.5 * skin) > 1e-6:  # reading C-5: within 1e-6 nm of skin/2 either answer is legal
                assert got == want, (scale, m)
            flag = dimos.dimos_nl_needs_rebuild(ctx, torch.from_numpy(pos).cuda(), torch.from_numpy(ref).cuda(), skin, sync=False)
            assert bool(flag.item()) == got  # the no-sync variant writes the same device flag
    finally:
        ctx.close()


def test_needs_rebuild_strict_and_raw_coordinates():
    ctx = dimos.Context(0, "f64")
    try:
        ref = torch.zeros(4, 3, dtype=torch.float64, device="cuda")
        pos = ref.clone()
        pos[2] = torch.tensor([0.03, 0.04, 0.0], dtype=torch.float64)  # |dr| == skin/2 exactly: strict > => False
        assert dimos.dimos_nl_needs_rebuild(ctx, pos, ref, 0.1) == oracle.needs_rebuild(pos.cpu().numpy(), ref.cpu().numpy(), 0.1)[0]
        pos[2, 2] = 0.001
        assert dimos.dimos_nl_needs_rebuild(ctx, pos, ref, 0.1) is True
        pos[2] = torch.tensor([2.0, 0.0, 0.0], dtype=torch.float64)  # a whole-box jump counts (no re-wrap)
        assert dimos.dimos_nl_needs_rebuild(ctx, pos, ref, 0.1) is True
    finally:
        ctx.close()


# --- A1 + A2 + A4 + A6 on the BASELINE configs the oracle finishes in seconds ----------------------------
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_config0_water216(precision):
    """configs[0]: 648 atoms, L = 1.8621 < 2 r_nl: degenerate 1x1x1 grid, r_nl > L/2 (readings C-3, C-18)."""
    wb = wl.make_config(0)
    rep = run_case(wb, precision, 0.9, 0.1, "rf", oracle_alg="bruteforce")
    assert rep["stats"]["n_cells"] == (1, 1, 1) and rep["stats"]["pbc_mode"] == 1
    assert rep["n_pairs_cut"] == 95574


@pytest.mark.parametrize("precision", ["f32", "mixed", "f64"])
def test_config1_water3k(precision):
    """configs[1] geometry: 9,000 atoms, 4^3 grid; several units per cell, ragged last unit in every cell."""
    wb = wl.make_config(1)
    rep = run_case(wb, precision, 1.0, 0.1, "rf")
    assert rep["stats"]["n_cells"] == (4, 4, 4) and rep["stats"]["pbc_mode"] == 0


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_ewald_real_space_and_exclusion_correction(precision):
    """configs[4] method on a box the oracle finishes quickly (2,000 waters): Eq. 10 + reading C-15."""
    wb = wl.make_scaled(2000, seed=wl.SEED_BASE + 4, method="ewald")
    rep = run_case(wb, precision, 1.0, 0.1, "ewald", alpha=3.12)
    assert rep["stats"]["pbc_mode"] == 0


def test_ewald_degenerate_grid_f32():
    wb = wl.make_water_box(100, 2.2, 4)
    run_case(wb, "f32", 1.0, 0.1, "ewald", oracle_alg="bruteforce")


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_slab_box_two_cells_per_axis(precision):
    """2 cells along x and y, 3 along z: stencil de-duplication, non-cubic box (reading C-18)."""
    wb = wl.make_water_box(150, 2.5, 21)
    run_case(wb, precision, 1.0, 0.1, "rf", box=np.array([2.5, 2.3, 3.4]), oracle_alg="bruteforce")


def test_unwrapped_and_shifted_positions_f32():
    """Positions need not lie in [0,L): shift by an arbitrary vector (> L) and move single atoms by +-L."""
    wb = wl.make_config(1)
    rng = np.random.default_rng(5)
    pos = wb.pos.astype(np.float64) + np.array([7.3, -11.9, 0.25])
    pos[rng.integers(0, wb.n_atoms, 200)] += np.array([wb.box[0], 0, 0])
    pos[rng.integers(0, wb.n_atoms, 200)] -= np.array([0, 2 * wb.box[1], 0])
    run_case(wb, "f32", 1.0, 0.1, "rf", pos=pos.astype(np.float32))


def test_no_exclusions_and_zero_skin_f64():
    """Empty exclusion list (NULL pointer), skin = 0; an LJ + RF fluid of well separated O atoms."""
    wb = wl.make_water_box(400, 3.3, 77)
    sel = np.arange(0, wb.n_atoms, 3)  # oxygens only: no close contacts
    import dataclasses
    sub = dataclasses.replace(wb, pos=wb.pos[sel].copy(), charge=wb.charge[sel].copy(), type=wb.type[sel].copy(),
                              excl_pairs=np.zeros((0, 2), np.int32), mass=wb.mass[sel].copy())
    run_case(sub, "f64", 1.0, 0.0, "rf")


def _mixture_box(n_side, edge, seed):
    """A non-water workload for the same path: point particles of three LJ types (one without LJ) with random
    charges (neutral in total) on a jittered lattice with vacancies, and a random exclusion list between lattice
    neighbours.  Units then mix types freely, some atoms have no exclusions and rows differ widely in length."""
    import dataclasses

    rng = np.random.default_rng(seed)
    a = edge / n_side
    sites = np.stack(np.meshgrid(*[np.arange(n_side)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)
    keep = rng.random(sites.shape[0]) > 0.15
    sites = sites[keep]
    n = sites.shape[0]
    pos = ((sites + 0.5) * a + rng.uniform(-0.06, 0.06, size=(n, 3))) % edge
    pos = pos.astype(np.float32)
    charge = rng.choice(np.array([-0.6, -0.2, 0.0, 0.3, 0.5]), size=n)
    charge -= charge.mean()
    typ = rng.integers(0, 3, size=n).astype(np.int32)
    cand = np.arange(0, n - 1, dtype=np.int32)
    pick = cand[rng.random(cand.size) < 0.3]
    excl = np.stack([pick, pick + 1], axis=1).astype(np.int32)
    base = wl.make_water_box(2, 5.0, 3)
    box = np.array([np.float32(edge)] * 3, dtype=np.float64)
    return dataclasses.replace(base, box=box, pos=pos, charge=charge.astype(np.float32), type=typ,
                               sigma=np.array([0.28, 0.22, 0.0]), epsilon=np.array([0.6, 0.3, 0.0]), excl_pairs=excl,
                               mass=np.ones(n))


@pytest.mark.gpu
@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f32", "ewald"), ("mixed", "rf"), ("f64", "ewald")])
def test_three_type_mixture_with_vacancies(precision, method):
    """Generality of the list and of both pair kernels beyond water: see _mixture_box."""
    wb = _mixture_box(16, 4.6, 2024)
    rep = run_case(wb, precision, 1.0, 0.1, method)
    assert rep["stats"]["pbc_mode"] == 0  # 4 cells per axis: the packed-FP32 kernel for f32, the generic one otherwise


@pytest.mark.gpu
@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f32", "ewald"), ("mixed", "rf"), ("f64", "rf")])
def test_lj_switching_function(precision, method):
    """LJ switching function S(x) of Eq. 6 between r_s = 0.8 nm and r_c = 1.0 nm: water (LJ on O
    only) and the three-type mixture, on the packed-FP32 kernel (f32) and on the generic one (mixed, f64)."""
    rep_w = run_case(wl.make_config(1), precision, 1.0, 0.1, method, r_switch=0.8, check_set=False)
    rep_m = run_case(_mixture_box(16, 4.6, 99), precision, 1.0, 0.1, method, r_switch=0.75, check_set=False)
    assert rep_w["n_pairs_cut"] > 0 and rep_m["n_pairs_cut"] > 0


def test_lj_switch_outside_range_is_plain_truncation_f32():
    """r_switch <= 0 or >= r_cut means no switching (include/dimos.h); NaN is rejected."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        ref = [t.clone() for t in dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)]
        for rs in (-1.0, 1.0, 2.5):
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, r_switch=rs)
            assert abs(float(E[1] - ref[1][1])) <= 1e-9 * abs(float(ref[1][1]))
        Fs, Es, _ = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, r_switch=0.8)
        assert float(Es[1]) != float(ref[1][1]) and abs(float(Es[2] - ref[1][2])) <= 1e-9 * abs(float(ref[1][2]))
        with pytest.raises(Exception):
            dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, r_switch=float("nan"))
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f32", "ewald"), ("mixed", "rf"), ("f64", "ewald")])
def test_one_four_exceptions(precision, method):
    """1-4 exceptions (reading C-21): a third of the excluded pairs of a water box (LJ on H too, so
    that the LJ scale acts) and of the three-type mixture add back scaled bare LJ + Coulomb."""
    import dataclasses

    wb = dataclasses.replace(wl.make_config(1), sigma=np.array([wl.SIGMA_O, 0.1]), epsilon=np.array([wl.EPS_O, 0.2]))
    exc = wb.excl_pairs[::3].copy()
    scale = np.tile(np.array([[0.8333, 0.5]]), (exc.shape[0], 1))
    scale[::2, 1] = 0.25  # individual factors
    plain = run_case(wb, precision, 1.0, 0.1, method, check_set=False)
    rep = run_case(wb, precision, 1.0, 0.1, method, check_set=False, exceptions=(exc, scale))
    assert rep["n_pairs_cut"] == plain["n_pairs_cut"]
    mix = _mixture_box(16, 4.6, 7)
    exc_m = mix.excl_pairs[1::2].copy()
    run_case(mix, precision, 1.0, 0.1, method, check_set=False, exceptions=(exc_m, np.full((exc_m.shape[0], 2), 0.5)))


def test_exceptions_survive_rebuild_and_can_be_cleared_f32():
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        E0 = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)[1].clone()
        exc = db.excl[::3].contiguous()
        sc = torch.full((exc.shape[0], 2), 0.5, dtype=torch.float64, device=exc.device)
        dimos.dimos_nl_set_exceptions(ctx, nl, exc, sc)
        E1 = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)[1].clone()
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl, nl=nl)  # rebuild in place keeps them
        E2 = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)[1].clone()
        dimos.dimos_nl_set_exceptions(ctx, nl, None, None)
        E3 = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)[1].clone()
        assert abs(float(E1[2] - E0[2])) > 1.0  # intramolecular Coulomb added back at half strength: large
        assert abs(float(E2[0] - E1[0])) <= 1e-6 * abs(float(E1[0])) and abs(float(E3[0] - E0[0])) <= 1e-6 * abs(float(E0[0]))
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("precision,index", [("f32", 1), ("f64", 1), ("f32", 0), ("f64", 0), ("f32", "ortho"), ("f64", "ortho"),
                                             ("f64", "ortho_unwrapped")])
def test_edge_list_with_vectors_and_shifts(precision, index):
    """dimos_nl_export_edges: the edge set within r_cut equals the oracle's (outside the +-1e-5 nm
    band), and every edge carries d = r_a - r_b - shift L and the shift the oracle computes.  configs[1] has 4 cells per
    axis (image from the cell offsets), configs[0] a single cell (per-pair minimum image)."""
    pos = None
    if isinstance(index, str):  # 3 x 4 x 6 cells with different edges; "unwrapped": atoms moved by whole boxes, so that the
        wb = _ortho_mixture_box((12, 16, 23), 0.2875, 32)  # shifts of an edge are large and differ from atom to atom
        if index == "ortho_unwrapped":
            k = np.random.default_rng(3).integers(-3, 4, size=wb.pos.shape)
            pos = wb.pos.astype(np.float64) + k * wb.box
    else:
        wb = wl.make_config(index)
    r_cut = 0.9 if index == 0 else 1.0
    db = DeviceBox(wb, precision, pos=pos)
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, r_cut, 0.1, db.excl)
        pairs, dvec, shift = dimos.dimos_nl_export_edges(ctx, nl, r_cut)
        pairs = pairs.cpu().numpy().astype(np.int64)
        dvec = dvec.double().cpu().numpy()
        shift = shift.cpu().numpy().astype(np.int64)
        pos64 = db.pos.double().cpu().numpy()
        n = wb.n_atoms
        key = pairs[:, 0] * n + pairs[:, 1]
        assert np.all(pairs[:, 0] < pairs[:, 1]) and np.unique(key).size == key.size
        must = oracle.neighbor_pairs(pos64, db.box, r_cut - BAND, wb.excl_pairs, "celllist").astype(np.int64)
        may = oracle.neighbor_pairs(pos64, db.box, r_cut + BAND, wb.excl_pairs, "celllist").astype(np.int64)
        assert np.setdiff1d(must[:, 0] * n + must[:, 1], key).size == 0
        assert np.setdiff1d(key, may[:, 0] * n + may[:, 1]).size == 0
        d_o, s_o = oracle.edge_vectors(pos64, db.box, pairs)
        tol = 1e-12 if precision == "f64" else 2e-6
        # a component within rounding of +-L/2 may legitimately take either image: compare d modulo L there
        alt = np.abs(np.abs(d_o) - 0.5 * db.box) < 1e-5
        assert np.all((shift == s_o) | alt)
        assert np.abs(dvec - d_o)[~alt].max() <= tol
        assert np.all(np.sqrt((dvec * dvec).sum(1)) < r_cut + BAND)
        assert np.abs(pos64[pairs[:, 0]] - pos64[pairs[:, 1]] - shift * db.box - dvec).max() <= tol
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_open_boundaries_through_the_virtual_box(precision):
    """Non-periodic system: a water droplet in vacuum, far from the origin and partly at negative
    coordinates.  The GPU path runs in the virtual periodic box dimos_virtual_box returns; the oracle in a box twenty
    times larger, where no periodic image exists at all: neighbour set, forces, energy and virial must agree."""
    import dataclasses

    full = wl.make_config(1)
    centre = 0.5 * full.box
    mol = np.arange(full.n_atoms) // 3
    keep_mol = np.unique(mol[(np.linalg.norm(full.pos[::3].astype(np.float64) - centre, axis=1) < 1.6).repeat(3)])
    sel = np.isin(mol, keep_mol)
    new_index = -np.ones(full.n_atoms, dtype=np.int64)
    new_index[sel] = np.arange(sel.sum())
    excl = full.excl_pairs[sel[full.excl_pairs[:, 0]] & sel[full.excl_pairs[:, 1]]]
    excl = new_index[excl].astype(np.int32)
    np_real = np.float64 if precision == "f64" else np.float32
    pos = (full.pos[sel].astype(np.float64) - centre + np.array([-0.7, 31.25, 5.5])).astype(np_real)
    drop = dataclasses.replace(full, pos=pos, charge=full.charge[sel].copy(), type=full.type[sel].copy(), excl_pairs=excl,
                               mass=full.mass[sel].copy())
    dev = torch.device("cuda", 0)
    ctx = dimos.Context(0, precision)
    try:
        box, lo = dimos.dimos_virtual_box(ctx, torch.from_numpy(pos).to(dev), 1.0, 0.1)
        ext = pos.astype(np.float64).max(0) - pos.astype(np.float64).min(0)
        assert np.all(box >= ext + 1.0 + 0.2) and np.all(box <= ext + 1.0 + 0.2 + 0.01) and np.allclose(lo, pos.min(0), atol=1e-6)
    finally:
        ctx.close()
    db = DeviceBox(drop, precision, box=box)
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, box, 1.0, 0.1, db.excl)
        pos64 = db.pos.double().cpu().numpy()
        big = 20.0 * box
        gp = dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy()
        check_neighbor_set(gp, pos64, big, 1.1, drop.excl_pairs)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method="rf")
        torch.cuda.synchronize()
        orc = oracle.nonbonded(pos64, db.charge.double().cpu().numpy(), drop.type, db.lj_np, big, 1.0, method=METHOD["rf"],
                               excl_pairs=drop.excl_pairs, band=BAND, algorithm="bruteforce")
        check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
    finally:
        ctx.close()


@pytest.mark.gpu
def test_uneven_density_grows_the_row_capacity_f32():
    """configs[1] squeezed into half of its box along x (a slab at twice the mean density next to vacuum): the first
    row-capacity estimate comes from the mean density, so the build must notice the overflow, grow and repeat
    (n_rebuild_grow > 0), and the result must still match the oracle."""
    import dataclasses

    wb = wl.make_config(1)
    pos = wb.pos.copy()
    pos[:, 0] *= np.float32(0.5)
    rep = run_case(dataclasses.replace(wb, pos=pos), "f32", 1.0, 0.1, "rf")
    assert rep["stats"]["n_rebuild_grow"] >= 1, rep["stats"]


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_exclusion_partner_limit(precision):
    """Every atom of the mixture excluded from its 16 successors and 16 predecessors in index order: 32 partners, the
    documented limit per atom (include/dimos.h), so every unit carries on the order of a hundred partially masked
    entries; neighbour set, Ewald exclusion correction and forces must match.  One partner more is an error."""
    import dataclasses

    mix = _mixture_box(16, 4.6, 5)
    n = mix.n_atoms
    i = np.arange(n, dtype=np.int32)

    def chain(kmax):
        e = np.concatenate([np.stack([i[:-k], i[k:]], axis=1) for k in range(1, kmax + 1)]).astype(np.int32)
        return e[np.lexsort((e[:, 1], e[:, 0]))]

    run_case(dataclasses.replace(mix, excl_pairs=chain(16)), precision, 1.0, 0.1, "ewald")
    with pytest.raises(dimos.DimosError):
        run_case(dataclasses.replace(mix, excl_pairs=chain(17)), precision, 1.0, 0.1, "ewald")


@pytest.mark.gpu
def test_dispersion_correction_matches_oracle():
    """LJ tail correction (reading C-22): device type histogram + host integrals against the oracle's
    adaptive quadrature of the definition, for water (one LJ species) and the three-type mixture, with and without switch."""
    ctx = dimos.Context(0, "f32")
    try:
        for wb in (wl.make_config(1), _mixture_box(16, 4.6, 3)):
            db = DeviceBox(wb, "f32")
            for rs in (0.0, 0.8, 0.95):
                e, w = dimos.dimos_dispersion_correction(ctx, db.type, db.lj, db.box, 1.0, rs)
                e_o, w_o = oracle.dispersion_correction(wb.type, db.lj_np, db.box, 1.0, rs)
                assert e == pytest.approx(e_o, rel=1e-10) and np.allclose(w, w_o, rtol=1e-10, atol=0)
                assert e < 0.0
        with pytest.raises(dimos.DimosError):
            dimos.dimos_dispersion_correction(ctx, db.type + 7, db.lj, db.box, 1.0, 0.0)  # type index out of range
    finally:
        ctx.close()


def test_tiny_systems_f64():
    """One water (everything excluded => E = 0, F = 0 under RF) and two waters (9 pairs)."""
    two = wl.make_water_box(2, 5.0, 3)
    pos = two.pos.astype(np.float64)
    pos[3:] = pos[3:] - pos[3] + pos[0] + np.array([0.31, 0.05, -0.02])
    import dataclasses
    one = dataclasses.replace(two, pos=two.pos[:3].copy(), charge=two.charge[:3].copy(), type=two.type[:3].copy(),
                              excl_pairs=two.excl_pairs[:3].copy(), mass=two.mass[:3].copy())
    db = DeviceBox(one, "f64")
    ctx = dimos.Context(0, "f64")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        assert dimos.dimos_nl_export_pairs(ctx, nl).shape[0] == 0
        F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)
        assert float(F.abs().max()) == 0.0 and float(E.abs().max()) == 0.0 and float(W.abs().max()) == 0.0
    finally:
        ctx.close()
    rep = run_case(two, "f64", 1.0, 0.1, "rf", pos=pos, oracle_alg="bruteforce")
    assert rep["set"][0] == 9 and rep["n_pairs_cut"] == 9


def test_two_particle_closed_form_through_gpu():
    """The golden two-particle values (tests/golden/two_particle_closed_forms.txt) through the CUDA path."""
    u = np.array([0.3, -0.5, 0.81])
    u /= np.linalg.norm(u)
    lj = torch.from_numpy(oracle.lorentz_berthelot([wl.SIGMA_O, 0.0], [wl.EPS_O, 0.0])).cuda()
    ctx = dimos.Context(0, "f64")
    try:
        for (qa, ta, qb, tb, r, rc, e_want, f_want) in [
            (wl.Q_O, 0, wl.Q_O, 0, 0.30, 0.9, 1.16685351179584 + 167.933704824648, 1149.71580381198),
            (wl.Q_O, 0, wl.Q_O, 0, 0.35, 1.0, 137.241056774674, 757.184487000131),
            (wl.Q_O, 0, wl.Q_H, 1, 0.20, 0.9, -162.872453453971, -1194.96291686214),
            (wl.Q_H, 1, wl.Q_H, 1, 0.25, 1.0, 61.3683742187847, 380.624403704081),
        ]:
            pos = torch.tensor(np.array([[10.0, 11.0, 12.0] + r * u, [10.0, 11.0, 12.0]]), device="cuda")
            q = torch.tensor([qa, qb], dtype=torch.float64, device="cuda")
            t = torch.tensor([ta, tb], dtype=torch.int32, device="cuda")
            nl = dimos.dimos_nl_build(ctx, pos, [50.0, 50.0, 50.0], rc, 0.1)
            F, E, W = dimos.dimos_nonbonded(ctx, nl, pos, q, t, lj)
            assert float(E[0]) == pytest.approx(e_want, rel=1e-12)
            assert float(F[0].cpu().numpy() @ u) == pytest.approx(f_want, rel=1e-12)
            assert np.allclose(F[0].cpu().numpy(), -F[1].cpu().numpy(), rtol=0, atol=1e-9)
            assert float(torch.trace(W)) == pytest.approx(r * f_want, rel=1e-12)
    finally:
        ctx.close()


# --- list reuse: forces from a list built at earlier positions ----------------------------
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_list_stays_valid_under_half_skin_displacement(precision):
    wb = wl.make_config(1)
    rc, skin = 1.0, 0.1
    db = DeviceBox(wb, precision)
    rng = np.random.default_rng(11)
    step = rng.standard_normal(wb.pos.shape)
    step *= (0.5 * skin * 0.98) / np.linalg.norm(step, axis=1, keepdims=True)
    moved = (wb.pos.astype(np.float64) + step).astype(np.float64 if precision == "f64" else np.float32)
    db2 = DeviceBox(wb, precision, pos=moved)
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, rc, skin, db.excl)
        assert dimos.dimos_nl_needs_rebuild(ctx, db2.pos, nl.pos_at_build, skin) is False
        F, E, W = dimos.dimos_nonbonded(ctx, nl, db2.pos, db.charge, db.type, db.lj)
        orc = oracle.nonbonded(db2.pos.double().cpu().numpy(), db.charge.double().cpu().numpy(), wb.type, db.lj_np, db.box, rc,
                               excl_pairs=wb.excl_pairs, band=BAND)
        check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
        # rebuilding in place at the new positions gives the same answer and the oracle's new pair set
        nl = dimos.dimos_nl_build(ctx, db2.pos, db.box, rc, skin, db.excl, nl=nl)
        check_neighbor_set(dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy(), db2.pos.double().cpu().numpy(), db.box, rc + skin,
                           wb.excl_pairs)
        F2, E2, W2 = dimos.dimos_nonbonded(ctx, nl, db2.pos, db.charge, db.type, db.lj)
        check_nonbonded(F2.cpu().numpy(), E2.cpu().numpy(), W2.cpu().numpy(), orc, precision)
    finally:
        ctx.close()


def test_repeat_calls_are_consistent_f32():
    """Two force calls on one list agree to summation-order noise; two builds export the identical set."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        a = dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy().astype(np.int64)
        F1, E1, _ = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)
        F1, E1 = F1.clone(), E1.clone()
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl, nl=nl)
        b = dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy().astype(np.int64)
        n = wb.n_atoms
        assert np.array_equal(np.sort(a[:, 0] * n + a[:, 1]), np.sort(b[:, 0] * n + b[:, 1]))
        F2, E2, _ = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)
        rms = float(F1.double().pow(2).sum(1).mean().sqrt())
        assert float((F1 - F2).abs().max()) <= 2e-5 * rms
        assert abs(float(E1[0] - E2[0])) <= 1e-6 * abs(float(E1[0]))
    finally:
        ctx.close()


def test_lj_table_change_after_row_reorder_f32():
    """The first force call after a build partitions every row by the LJ activity of the j-atoms (an optimisation of
    the packed-FP32 kernel).  A later call with a table in which the OTHER type carries LJ (stale order, every
    i-atom pair LJ-active on the hydrogen side) must still match the oracle: the kernel decides per chunk."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        pos64 = db.pos.double().cpu().numpy()
        q64 = db.charge.double().cpu().numpy()
        for sigma, eps in ((wb.sigma, wb.epsilon), ([0.0, 0.12], [0.0, 0.25]), ([0.30, 0.10], [0.5, 0.2])):
            lj_np = oracle.lorentz_berthelot(np.asarray(sigma, dtype=np.float64), np.asarray(eps, dtype=np.float64))
            lj = torch.from_numpy(lj_np).to(db.pos.device).contiguous()
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, lj)
            torch.cuda.synchronize()
            orc = oracle.nonbonded(pos64, q64, wb.type, lj_np, db.box, 1.0, method=METHOD["rf"], eps_rf=78.5,
                                   excl_pairs=wb.excl_pairs, band=BAND, algorithm="celllist")
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32")
    finally:
        ctx.close()


def test_host_buffer_entry_point_f32():
    """dimos_nonbonded_host (the e2e leg of bench.py): same result as the device call."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)
        hp = torch.from_numpy(wb.pos).pin_memory()
        hq = torch.from_numpy(wb.charge).pin_memory()
        ht = torch.from_numpy(wb.type).pin_memory()
        hl = torch.from_numpy(db.lj_np).pin_memory()
        hF = torch.empty_like(hp).pin_memory()
        hE = torch.empty(4, dtype=torch.float64).pin_memory()
        hW = torch.empty(3, 3, dtype=torch.float64).pin_memory()
        ctx.nonbonded_host(nl, hp, hq, ht, hl, hF, hE, hW)
        rms = float(F.double().pow(2).sum(1).mean().sqrt())
        assert float((F.cpu() - hF).abs().max()) <= 2e-5 * rms
        assert abs(float(E[0].cpu() - hE[0])) <= 1e-6 * abs(float(hE[0]))
    finally:
        ctx.close()


# --- error behaviour of the boundary (include/dimos.h) ----------------------------------------------------
def test_error_codes():
    wb = wl.make_config(0)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        with pytest.raises(dimos.DimosError) as ei:
            dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)  # r_cut > L/2
        assert ei.value.status == -2
        with pytest.raises(dimos.DimosError) as ei:
            dimos.dimos_nl_build(ctx, db.pos, [1.0, -1.0, 1.0], 0.4, 0.1, db.excl)
        assert ei.value.status == -1
        bad = db.pos.clone()
        bad[17, 1] = float("nan")
        with pytest.raises(dimos.DimosError) as ei:
            dimos.dimos_nl_build(ctx, bad, db.box, 0.9, 0.1, db.excl)
        assert ei.value.status == -1
        bad_excl = db.excl.clone()
        bad_excl[5, 1] = wb.n_atoms + 3
        with pytest.raises(dimos.DimosError) as ei:
            dimos.dimos_nl_build(ctx, db.pos, db.box, 0.9, 0.1, bad_excl)
        assert ei.value.status == -1
        dup_excl = torch.cat([db.excl, db.excl[7:8]])  # one pair listed twice (reading C-17: rows are unique)
        with pytest.raises(dimos.DimosError, match="more than once") as ei:
            dimos.dimos_nl_build(ctx, db.pos, db.box, 0.9, 0.1, dup_excl)
        assert ei.value.status == -1
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 0.9, 0.1, db.excl)
        nl.r_cut = 0.8  # params.r_cut differs from the build r_cut
        with pytest.raises(dimos.DimosError) as ei:
            dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)
        assert ei.value.status == -6
        nl.r_cut = 0.9
        F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)  # still usable afterwards
        assert torch.isfinite(F).all()
        rc = ctx.lib.dimos_nl_build(None, None, 0, None, 0.0, 0.0, None, 0, None, None, None)
        assert rc == -1
    finally:
        ctx.close()


# --- full-size configs in bench.py's launch configuration: the WHOLE system against the oracle ----------------
# north_star "Target": pair sets matching the oracle exactly and forces / energies within tolerance on all five
# configs.  The oracle's cell list evaluates these boxes in seconds, so nothing is sampled: the exported pair set (as
# sorted keys, outside the +-1e-5 band), every atom's force, E[0..3], the virial and the in-cutoff pair count that
# bench.py's metric uses are compared for the whole box.
@pytest.mark.parametrize("precision", ["f32", "mixed"])
def test_config2_water30k_whole_system(precision):
    wb = wl.make_config(2)
    rep = run_case(wb, precision, 1.0, 0.1, "rf", on_device=True)
    assert rep["stats"]["n_cells"] == (8, 8, 8) and rep["stats"]["pbc_mode"] == 0
    assert abs(rep["set"][0] / (wb.n_atoms * 278.8) - 1.0) < 0.02  # pairs < r_nl per atom at this density


def test_config3_water300k_headline_whole_system_f32():
    """The bench workload (configs[3], 900,000 atoms) in the launch configuration bench.py times."""
    wb = wl.make_config(3)
    rep = run_case(wb, "f32", 1.0, 0.1, "rf", on_device=True)
    assert rep["stats"]["n_cells"] == (18, 18, 18) and rep["stats"]["pbc_mode"] == 0
    assert abs(rep["set"][0] / (wb.n_atoms * 278.8) - 1.0) < 0.02


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_config4_water100k_ewald_whole_system(precision):
    wb = wl.make_config(4)
    rep = run_case(wb, precision, 1.0, 0.1, "ewald", alpha=3.12, on_device=True)
    assert rep["stats"]["n_cells"] == (13, 13, 13) and rep["stats"]["pbc_mode"] == 0


def test_invalid_types_and_exception_lists_are_reported():
    """a type index outside [0, ntypes) and an exception pair that is not an excluded pair return DIMOS_EINVAL
    instead of garbage (types: at the next synchronising call on the list; exceptions: when they are set)."""
    wb = wl.make_config(0)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 0.9, 0.1, db.excl)
        good = db.excl[:5].clone()
        scale = torch.full((5, 2), 0.5, dtype=torch.float64, device="cuda")
        dimos.dimos_nl_set_exceptions(ctx, nl, good, scale)
        bad = good.clone()
        bad[2, 1] = bad[2, 0] + 5  # (O of one molecule, an atom of the next): in range, i < j, not excluded
        with pytest.raises(dimos.DimosError) as ei:
            dimos.dimos_nl_set_exceptions(ctx, nl, bad, scale)
        assert ei.value.status == -1
        bad[2, 1] = wb.n_atoms
        with pytest.raises(dimos.DimosError):
            dimos.dimos_nl_set_exceptions(ctx, nl, bad, scale)
        dimos.dimos_nl_set_exceptions(ctx, nl, good[:0], scale[:0])
        # out-of-range type through the host entry point
        n = wb.n_atoms
        h = dict(pos=torch.from_numpy(wb.pos).pin_memory(), charge=torch.from_numpy(wb.charge).pin_memory(),
                 lj=torch.from_numpy(db.lj_np).pin_memory(), F=torch.empty((n, 3)).pin_memory(),
                 E=torch.empty(4, dtype=torch.float64).pin_memory(), W=torch.empty((3, 3), dtype=torch.float64).pin_memory())
        t_bad = torch.from_numpy(wb.type.copy())
        t_bad[17] = 2
        with pytest.raises(dimos.DimosError) as ei:
            ctx.nonbonded_host(nl, h["pos"], h["charge"], t_bad.pin_memory(), h["lj"], h["F"], h["E"], h["W"])
        assert ei.value.status == -1
    finally:
        ctx.close()


def test_needs_rebuild_on_two_streams_at_once():
    """Two trigger evaluations in flight on different streams: each has its own reduction state, so
    neither sees the other's partial maximum or ticket count."""
    n = 2_000_000
    g = torch.Generator(device="cuda").manual_seed(3)
    ref = torch.rand((n, 3), device="cuda", generator=g) * 20
    moved = ref.clone()
    moved[n - 7, 1] += 0.2       # beyond skin/2 = 0.05
    still = ref + 1e-3
    ctx = dimos.Context(0, "f32")
    try:
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        f1 = torch.zeros(1, dtype=torch.int32, device="cuda")
        f2 = torch.zeros(1, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        for _ in range(20):
            with torch.cuda.stream(s1):
                dimos.dimos_nl_needs_rebuild(ctx, moved, ref, 0.1, sync=False, flag=f1)
            with torch.cuda.stream(s2):
                dimos.dimos_nl_needs_rebuild(ctx, still, ref, 0.1, sync=False, flag=f2)
            torch.cuda.synchronize()
            assert int(f1.item()) == 1 and int(f2.item()) == 0
    finally:
        ctx.close()


@pytest.mark.parametrize("precision", ["f32", "f64", "mixed"])
def test_lj_activity_changes_after_the_build(precision):
    """The builder files the rows by the LJ-activity flags of the LAST force call (a hint).  If the types or the LJ table
    change afterwards so that an atom assumed LJ-free has LJ partners, the pair kernels must notice and evaluate LJ in
    every chunk: forces and energies still match the oracle, before and after the next rebuild; the opposite change
    (atoms lose their LJ partners) needs no fallback and must match as well."""
    wb = wl.make_config(1)
    db = DeviceBox(wb, precision)
    pos64 = db.pos.double().cpu().numpy()
    q64 = db.charge.double().cpu().numpy()
    lj_water = lj_table_np(wb)                                     # LJ on O only
    lj_all = oracle.lorentz_berthelot([wl.SIGMA_O, 0.12], [wl.EPS_O, 0.2])   # H gets a small LJ core too
    lj_none = oracle.lorentz_berthelot([wl.SIGMA_O, 0.0], [0.0, 0.0])        # nobody has LJ
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        for table in (lj_water, lj_water):  # second call: after a rebuild that used the first call's flags
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, torch.from_numpy(table).cuda())
            nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl, nl=nl)
        for table in (lj_all, lj_all, lj_none, lj_water, lj_all):
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, torch.from_numpy(table).cuda())
            orc = oracle.nonbonded(pos64, q64, wb.type, table, db.box, 1.0, excl_pairs=wb.excl_pairs, band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl, nl=nl)  # hint: everybody active
        for table in (lj_all, lj_water):
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, torch.from_numpy(table).cuda())
            orc = oracle.nonbonded(pos64, q64, wb.type, table, db.box, 1.0, excl_pairs=wb.excl_pairs, band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
        gp = dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy()
        check_neighbor_set(gp, pos64, db.box, 1.1, wb.excl_pairs)
    finally:
        ctx.close()


def test_sparse_gas_with_isolated_atoms_f32():
    """A dilute gas in a box with many cells: most units hold one or two atoms and many have no list entry at all (the
    packed kernel then copies no row for them and must keep its buffer bookkeeping straight); a few close pairs carry the
    whole energy."""
    rng = np.random.default_rng(31)
    n = 1500
    box = np.array([14.0, 13.0, 15.0])
    pos = rng.uniform(0, 1, size=(n, 3)) * box
    pos[1::2][:300] = pos[0::2][:300] + rng.normal(0, 0.2, size=(300, 3))  # 300 pairs at ~0.35 nm
    pos = pos.astype(np.float32)
    q = rng.choice([-0.5, 0.5], size=n).astype(np.float32)
    typ = rng.integers(0, 2, size=n).astype(np.int32)
    lj_np = oracle.lorentz_berthelot([0.3, 0.0], [0.5, 0.0])
    ctx = dimos.Context(0, "f32")
    try:
        dp, dq, dt = torch.from_numpy(pos).cuda(), torch.from_numpy(q).cuda(), torch.from_numpy(typ).cuda()
        lj = torch.from_numpy(lj_np).cuda()
        nl = dimos.dimos_nl_build(ctx, dp, box, 1.0, 0.1, None)
        assert nl.stats()["pbc_mode"] == 0
        for _ in range(2):
            F, E, W = dimos.dimos_nonbonded(ctx, nl, dp, dq, dt, lj)
            orc = oracle.nonbonded(pos.astype(np.float64), q, typ, lj_np, box, 1.0, band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32")
            nl = dimos.dimos_nl_build(ctx, dp, box, 1.0, 0.1, None, nl=nl)
        check_neighbor_set(dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy(), pos.astype(np.float64), box, 1.1, None)
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("precision,method,nt", [("f32", "rf", 17), ("f32", "ewald", 40), ("f32", "rf", 64), ("mixed", "rf", 64),
                                                 ("f64", "ewald", 64), ("f64", "rf", 23)])
def test_many_atom_types(precision, method, nt):
    """Up to MAX_TYPES = 64 atom types (Eq. 5 table of nt x nt entries in shared memory; the packed kernel hands over to the
    generic one when the table does not fit beside its row buffers): the mixture of _mixture_box with random types, a third
    of the types without LJ partners, compared with the oracle as a whole system."""
    import dataclasses

    wb = _mixture_box(16, 4.6, 99 + nt)
    rng = np.random.default_rng(nt)
    sigma = rng.uniform(0.18, 0.30, size=nt)
    eps = rng.uniform(0.1, 0.8, size=nt)
    eps[rng.random(nt) < 0.33] = 0.0
    eps[0] = 0.5  # at least one LJ-active type
    wb = dataclasses.replace(wb, type=rng.integers(0, nt, size=wb.n_atoms).astype(np.int32), sigma=sigma, epsilon=eps)
    rep = run_case(wb, precision, 1.0, 0.1, method, check_set=False)
    assert rep["stats"]["pbc_mode"] == 0


@pytest.mark.gpu
def test_more_than_64_types_is_rejected():
    wb = _mixture_box(12, 3.5, 5)
    db = DeviceBox(wb, "f32")
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        lj = torch.ones(65, 65, 2, dtype=torch.float64, device=db.pos.device)
        with pytest.raises(dimos.DimosError) as err:
            dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, lj)
        assert err.value.args[0].endswith("(status -1)")
    finally:
        ctx.close()


@pytest.mark.gpu
def test_short_rows_as_the_first_call_of_a_process_f32():
    """Regression: a list with short rows (a box of a third of water's density: row capacity 576) gives the packed kernel
    25 .. 48 KB of dynamic shared memory, which together with its ~17 KB of static shared memory needs the opt-in attribute;
    the launch failed with `invalid argument` unless an earlier call of the same process (a water box) had raised the
    attribute.  Runs the mixture as the FIRST force call of a fresh process, against the oracle."""
    import os
    import subprocess
    import sys

    here = os.path.dirname(os.path.abspath(__file__))
    script = ("import sys; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
              "from test_gpu_parity import _mixture_box\n"
              "from gpu_harness import run_case\n"
              "rep = run_case(_mixture_box(16, 4.6, 2024), 'f32', 1.0, 0.1, 'rf')\n"
              "assert rep['stats']['row_capacity'] < 1000, rep['stats']\n"
              "print('fresh-process ok', rep['stats']['row_capacity'])\n") % (os.path.dirname(here), here)
    res = subprocess.run([sys.executable, "-c", script], capture_output=True, text=True, timeout=600)
    assert res.returncode == 0 and "fresh-process ok" in res.stdout, res.stdout[-2000:] + res.stderr[-4000:]


def _ortho_mixture_box(n_sites, a, seed):
    """_mixture_box on an nx x ny x nz lattice: an orthorhombic box with different edges (and cell counts) per axis."""
    import dataclasses

    rng = np.random.default_rng(seed)
    n_sites = np.asarray(n_sites)
    box = np.array([np.float32(k * a) for k in n_sites], dtype=np.float64)
    sites = np.stack(np.meshgrid(*[np.arange(k) for k in n_sites], indexing="ij"), axis=-1).reshape(-1, 3)
    sites = sites[rng.random(sites.shape[0]) > 0.1]
    n = sites.shape[0]
    pos = ((sites + 0.5) * (box / n_sites) + rng.uniform(-0.06, 0.06, size=(n, 3))) % box
    pos = np.minimum(pos.astype(np.float32), np.nextafter(box.astype(np.float32), np.float32(0)))
    charge = rng.choice(np.array([-0.6, -0.2, 0.0, 0.3, 0.5]), size=n)
    charge -= charge.mean()
    pick = np.arange(0, n - 1, dtype=np.int32)[rng.random(n - 1) < 0.3]
    base = wl.make_water_box(2, 5.0, 3)
    return dataclasses.replace(base, box=box, pos=pos, charge=charge.astype(np.float32), type=rng.integers(0, 3, size=n).astype(np.int32),
                               sigma=np.array([0.28, 0.22, 0.0]), epsilon=np.array([0.6, 0.3, 0.0]),
                               excl_pairs=np.stack([pick, pick + 1], axis=1).astype(np.int32), mass=np.ones(n))


@pytest.mark.gpu
@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f32", "ewald"), ("mixed", "rf"), ("f64", "ewald"), ("f64", "rf")])
def test_orthorhombic_box_with_different_cell_counts_per_axis(precision, method):
    """3 x 4 x 6 cells (edges 3.45, 4.6, 6.61 nm): the image shift of a list entry comes from the cell offsets, whose edge
    differs per axis; pair set, forces, energies and virial of the whole system against the oracle."""
    wb = _ortho_mixture_box((12, 16, 23), 0.2875, 31)
    rep = run_case(wb, precision, 1.0, 0.1, method)
    assert rep["stats"]["pbc_mode"] == 0 and list(rep["stats"]["n_cells"]) == [3, 4, 6]
    # the same system with the axes permuted: another assignment of lengths to the fastest / slowest cell index
    import dataclasses

    perm = [2, 0, 1]
    wb2 = dataclasses.replace(wb, box=wb.box[perm].copy(), pos=np.ascontiguousarray(wb.pos[:, perm]))
    rep2 = run_case(wb2, precision, 1.0, 0.1, method)
    assert list(rep2["stats"]["n_cells"]) == [6, 3, 4]
    assert rep2["n_pairs_cut"] == rep["n_pairs_cut"]


@pytest.mark.gpu
@pytest.mark.parametrize("precision,method", [("f32", "rf"), ("f32", "ewald"), ("mixed", "rf"), ("f64", "ewald")])
def test_short_cutoff_many_cells(precision, method):
    """configs[1]'s water box with r_c = 0.45 nm, skin 0.05 nm: 8 cells per axis of ~16 atoms each, two units per cell, rows
    of ~60 entries (the smallest row capacity the builder uses)."""
    wb = wl.make_config(1)
    rep = run_case(wb, precision, 0.45, 0.05, method)
    assert rep["stats"]["pbc_mode"] == 0 and min(rep["stats"]["n_cells"]) >= 8


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_dense_fluid_with_rows_beyond_the_packed_kernels_buffers(precision):
    """Point particles at four times water's atom density (400 nm^-3): ~1,600 list entries per unit, so the row capacity
    grows past what the packed kernel can stage in shared memory and the fp32 call runs on the generic kernel; cells hold
    ~580 atoms (the in-cell sorter's multi-pass path)."""
    import dataclasses

    rng = np.random.default_rng(404)
    n_side, edge = 25, 3.4
    a = edge / n_side
    sites = np.stack(np.meshgrid(*[np.arange(n_side)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)
    n = sites.shape[0]
    pos = (((sites + 0.5) * a + rng.uniform(-0.03, 0.03, size=(n, 3))) % edge).astype(np.float32)
    charge = rng.choice(np.array([-0.3, 0.0, 0.3]), size=n)
    charge -= charge.mean()
    base = wl.make_water_box(2, 5.0, 3)
    wb = dataclasses.replace(base, box=np.array([np.float32(edge)] * 3, dtype=np.float64), pos=pos, charge=charge.astype(np.float32),
                             type=rng.integers(0, 2, size=n).astype(np.int32), sigma=np.array([0.10, 0.08]),
                             epsilon=np.array([0.4, 0.0]), excl_pairs=np.zeros((0, 2), np.int32), mass=np.ones(n))
    rep = run_case(wb, precision, 1.0, 0.1, "rf")
    assert rep["stats"]["row_capacity"] > 1500 and rep["stats"]["pbc_mode"] == 0


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_one_list_handle_rebuilt_for_different_systems(precision):
    """dimos_nl_build with an existing handle takes ANY new system: another atom count, box, cutoff, cell grid (one cell
    with per-pair minimum image <-> 3 x 4 x 6 cells), exclusion list (none, water's, random) and type count.  Nothing of the
    previous system may survive in the handle's buffers: after every rebuild the pair set, forces, energies and virial are
    compared with the oracle, and the sequence returns to the first system at the end."""
    import dataclasses

    water216, water3k = wl.make_config(0), wl.make_config(1)
    ortho = _ortho_mixture_box((12, 16, 23), 0.2875, 77)
    gas = dataclasses.replace(ortho, pos=ortho.pos[::9].copy(), charge=(ortho.charge[::9] - ortho.charge[::9].mean()).astype(np.float32),
                              type=ortho.type[::9].copy(), excl_pairs=np.zeros((0, 2), np.int32), mass=ortho.mass[::9].copy())
    cases = [(water3k, 1.0, 0.1, "rf"), (water216, 0.9, 0.1, "rf"), (ortho, 1.0, 0.1, "ewald"), (gas, 0.8, 0.3, "rf"),
             (water3k, 0.7, 0.05, "ewald"), (water216, 0.9, 0.1, "rf")]
    ctx = dimos.Context(0, precision)
    nl = None
    try:
        for k, (wb, r_cut, skin, method) in enumerate(cases):
            db = DeviceBox(wb, precision)
            nl = dimos.dimos_nl_build(ctx, db.pos, db.box, r_cut, skin, db.excl if wb.excl_pairs.shape[0] else None, nl=nl)
            assert torch.equal(nl.pos_at_build, db.pos)
            pos64 = db.pos.double().cpu().numpy()
            gp = dimos.dimos_nl_export_pairs(ctx, nl).cpu().numpy()
            check_neighbor_set(gp, pos64, db.box, r_cut + skin, wb.excl_pairs)
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj, method=method)
            torch.cuda.synchronize()
            orc = oracle.nonbonded(pos64, db.charge.double().cpu().numpy(), wb.type, db.lj_np, db.box, r_cut, method=METHOD[method],
                                   excl_pairs=wb.excl_pairs, band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, precision)
            assert nl.stats()["n_atoms"] == wb.n_atoms, k
    finally:
        ctx.close()


@pytest.mark.gpu
def test_exceptions_are_revalidated_when_the_handle_is_rebuilt_for_another_system():
    """The 1-4 exceptions stored in a list index atoms and must be excluded pairs.  Rebuilding the handle for fewer atoms
    (indices out of range) or with an exclusion list that lacks them (they would be counted twice) must not use them:
    the build removes them and returns DIMOS_EINVAL; the next build succeeds and the forces are those without exceptions."""
    big, small = wl.make_config(1), wl.make_config(0)
    dbig, dsmall = DeviceBox(big, "f32"), DeviceBox(small, "f32")
    dev = dbig.pos.device
    exc = torch.from_numpy(big.excl_pairs[-30:].copy()).to(dev)  # pairs of the last molecules: beyond the small system's N
    scale = torch.full((30, 2), 0.5, dtype=torch.float64, device=dev)
    ctx = dimos.Context(0, "f32")
    try:
        nl = dimos.dimos_nl_build(ctx, dbig.pos, dbig.box, 1.0, 0.1, dbig.excl)
        dimos.dimos_nl_set_exceptions(ctx, nl, exc, scale)
        nl = dimos.dimos_nl_build(ctx, dbig.pos, dbig.box, 1.0, 0.1, dbig.excl, nl=nl)  # same system: they stay
        with pytest.raises(dimos.DimosError, match="exceptions do not fit"):
            dimos.dimos_nl_build(ctx, dsmall.pos, dsmall.box, 0.9, 0.1, dsmall.excl, nl=nl)
        nl = dimos.dimos_nl_build(ctx, dsmall.pos, dsmall.box, 0.9, 0.1, dsmall.excl, nl=nl)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, dsmall.pos, dsmall.charge, dsmall.type, dsmall.lj)
        orc = oracle.nonbonded(dsmall.pos.double().cpu().numpy(), small.charge, small.type, dsmall.lj_np, dsmall.box, 0.9,
                               excl_pairs=small.excl_pairs, band=BAND)
        check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32")
        # same atoms, but an exclusion list without the exception pairs
        nl = dimos.dimos_nl_build(ctx, dbig.pos, dbig.box, 1.0, 0.1, dbig.excl, nl=nl)
        dimos.dimos_nl_set_exceptions(ctx, nl, exc, scale)
        fewer = torch.from_numpy(big.excl_pairs[:-30].copy()).to(dev)
        with pytest.raises(dimos.DimosError, match="exceptions do not fit"):
            dimos.dimos_nl_build(ctx, dbig.pos, dbig.box, 1.0, 0.1, fewer, nl=nl)
        nl = dimos.dimos_nl_build(ctx, dbig.pos, dbig.box, 1.0, 0.1, dbig.excl, nl=nl)
        F, E, W = dimos.dimos_nonbonded(ctx, nl, dbig.pos, dbig.charge, dbig.type, dbig.lj)
        orc = oracle.nonbonded(dbig.pos.double().cpu().numpy(), big.charge, big.type, dbig.lj_np, dbig.box, 1.0,
                               excl_pairs=big.excl_pairs, band=BAND)
        check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, "f32")
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f32", "mixed", "f64"])
@pytest.mark.parametrize("kind", ["pure_lj", "pure_coulomb", "nothing"])
def test_systems_without_charges_or_without_lj(precision, kind):
    """An argon-like fluid (no charges: every row is in the LJ phase, E_coul = 0 exactly), point charges without any LJ
    parameters (every row in the LJ-free phase after the first call's hint, E_lj = 0 exactly) and a system with neither
    (all outputs exactly zero).  Two force calls with a rebuild in between, so that the second list is filed by the hint."""
    import dataclasses

    wb = _mixture_box(16, 4.6, 11)
    n = wb.n_atoms
    if kind == "pure_lj":
        wb = dataclasses.replace(wb, charge=np.zeros(n, np.float32), type=np.zeros(n, np.int32), sigma=np.array([0.26]), epsilon=np.array([0.9]))
    elif kind == "pure_coulomb":
        wb = dataclasses.replace(wb, sigma=np.array([0.3, 0.2, 0.0]), epsilon=np.zeros(3))
    else:
        wb = dataclasses.replace(wb, charge=np.zeros(n, np.float32), sigma=np.zeros(3), epsilon=np.zeros(3))
    db = DeviceBox(wb, precision)
    ctx = dimos.Context(0, precision)
    try:
        nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl)
        orc = oracle.nonbonded(db.pos.double().cpu().numpy(), wb.charge, wb.type, db.lj_np, db.box, 1.0, excl_pairs=wb.excl_pairs, band=BAND)
        for rep in range(2):
            F, E, W = dimos.dimos_nonbonded(ctx, nl, db.pos, db.charge, db.type, db.lj)
            F, E, W = F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy()
            if kind == "nothing":
                assert not F.any() and not E.any() and not W.any()
            else:
                check_nonbonded(F, E, W, orc, precision)
                assert E[2 if kind == "pure_lj" else 1] == 0.0  # E = (total, LJ, Coulomb, exclusion correction)
            nl = dimos.dimos_nl_build(ctx, db.pos, db.box, 1.0, 0.1, db.excl, nl=nl)
    finally:
        ctx.close()


@pytest.mark.gpu
def test_two_contexts_and_two_lists_interleaved():
    """Two contexts of different precision on one device, and two lists in one of them, used in alternation on two streams:
    a context's workspace, a list's buffers and the per-call reduction state belong to their owner only."""
    a, b = wl.make_config(1), _mixture_box(16, 4.6, 5)
    da32, db32, da64 = DeviceBox(a, "f32"), DeviceBox(b, "f32"), DeviceBox(a, "f64")
    c32, c64 = dimos.Context(0, "f32"), dimos.Context(0, "f64")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    try:
        with torch.cuda.stream(s1):
            nl_a = dimos.dimos_nl_build(c32, da32.pos, da32.box, 1.0, 0.1, da32.excl)
        with torch.cuda.stream(s2):
            nl_b = dimos.dimos_nl_build(c32, db32.pos, db32.box, 1.0, 0.1, db32.excl)
            nl_c = dimos.dimos_nl_build(c64, da64.pos, da64.box, 1.0, 0.1, da64.excl)
        torch.cuda.synchronize()
        out = {}
        for rep in range(3):
            with torch.cuda.stream(s1):
                out["a"] = dimos.dimos_nonbonded(c32, nl_a, da32.pos, da32.charge, da32.type, da32.lj)
            with torch.cuda.stream(s2):
                out["c"] = dimos.dimos_nonbonded(c64, nl_c, da64.pos, da64.charge, da64.type, da64.lj, method="ewald")
            with torch.cuda.stream(s1):
                out["b"] = dimos.dimos_nonbonded(c32, nl_b, db32.pos, db32.charge, db32.type, db32.lj, method="ewald")
        torch.cuda.synchronize()
        for key, dbx, wb, prec, method in (("a", da32, a, "f32", "rf"), ("b", db32, b, "f32", "ewald"), ("c", da64, a, "f64", "ewald")):
            F, E, W = out[key]
            orc = oracle.nonbonded(dbx.pos.double().cpu().numpy(), dbx.charge.double().cpu().numpy(), wb.type, dbx.lj_np, dbx.box, 1.0,
                                   method=METHOD[method], excl_pairs=wb.excl_pairs, band=BAND)
            check_nonbonded(F.cpu().numpy(), E.cpu().numpy(), W.cpu().numpy(), orc, prec)
    finally:
        c32.close()
        c64.close()


@pytest.mark.gpu
def test_list_beyond_two_to_the_31_entries_f32():
    """12.6 million atoms (4.2 million waters, edge 50.1 nm): 1.61 million units x a row capacity of 1,344 = 2.17e9 entry
    slots, beyond the range of a 32-bit index.  Every atom's force, the energies, the virial and the in-cutoff pair count
    (2.64e9) against the oracle's cell list (~35 s on 16 cores)."""
    wb = wl.make_scaled(4200000, seed=wl.SEED_BASE + 99, method="rf")
    rep = run_case(wb, "f32", 1.0, 0.1, "rf", check_set=False, on_device=True)
    assert rep["stats"]["n_units"] * rep["stats"]["row_capacity"] > 2**31
    assert rep["n_pairs_cut"] > 2.6e9
