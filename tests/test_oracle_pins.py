"""Pins for the CPU fp64 oracle (oracle/dimos_oracle.c): closed forms, textbook points, invariants,
finite differences, brute force vs cell list vs scipy.  None of these re-type the oracle's own
expression for a quantity and compare it with itself: each checks the oracle against something the
paper or the mathematics fixes independently (SURVEY.md §8(c) "What pins each part")."""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2503_20541_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
KE = wl.COULOMB_CONST
Q = {"O": wl.Q_O, "H": wl.Q_H}
TYPE = {"O": 0, "H": 1}
BIGBOX = np.array([50.0, 50.0, 50.0])


def lj_table():
    return oracle.lorentz_berthelot([wl.SIGMA_O, 0.0], [wl.EPS_O, 0.0])


def two_particles(kind_a, kind_b, r, r_cut, method=oracle.METHOD_RF, excluded=False, direction=None, **kw):
    """Energy components and radial force on atom 0 along +d for an isolated pair in a huge box."""
    if direction is None:
        direction = np.array([0.3, -0.5, 0.81])
    u = direction / np.linalg.norm(direction)
    pos = np.array([[10.0, 11.0, 12.0] + r * u, [10.0, 11.0, 12.0]])
    excl = np.array([[0, 1]], dtype=np.int32) if excluded else None
    res = oracle.nonbonded(pos, [Q[kind_a], Q[kind_b]], [TYPE[kind_a], TYPE[kind_b]], lj_table(), BIGBOX, r_cut,
                           method=method, excl_pairs=excl, algorithm="bruteforce", **kw)
    f_radial = float(res.F[0] @ u)
    # transverse components must vanish and Newton III must hold
    assert np.allclose(res.F[0] - f_radial * u, 0.0, atol=1e-9 * max(1.0, abs(f_radial)))
    assert np.allclose(res.F[0] + res.F[1], 0.0, atol=1e-9 * max(1.0, abs(f_radial)))
    return res, f_radial


# --- golden closed-form values (SURVEY.md §8(c), 30-digit mpmath, independent of this repo) --------------
def _golden_rows():
    rows = []
    with open(os.path.join(GOLDEN, "two_particle_closed_forms.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            kind, pair, r, rc, qty, val = line.split()
            rows.append((kind, pair, float(r), float(rc), qty, float(val)))
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"{r[0]}-{r[1]}-{r[2]}-{r[4]}")
def test_two_particle_golden(row):
    kind, pair, r, rc, qty, val = row
    method = oracle.METHOD_RF if kind == "rf" else oracle.METHOD_EWALD_REAL
    res, f = two_particles(pair[0], pair[1], r, rc, method=method, excluded=(kind == "excl"))
    got = {
        "U": res.E[0], "U_LJ": res.E[1], "U_RF": res.E[2], "U_COUL": res.E[2], "f": f, "r_dot_f": r * f,
    }[qty]
    if kind == "excl":
        assert res.E[1] == 0.0 and res.E[2] == 0.0  # excluded pair: no LJ, no pair Coulomb
        assert res.E[3] == res.E[0]
    assert got == pytest.approx(val, rel=2e-13, abs=1e-15)


# --- textbook points of Eq. (4) ---------------------------------------------------------------------------
def test_lj_zero_crossing_and_minimum():
    tab = lj_table()
    pos = lambda r: np.array([[5.0 + r, 5.0, 5.0], [5.0, 5.0, 5.0]])
    zero = [0.0, 0.0]
    r0 = wl.SIGMA_O
    res = oracle.nonbonded(pos(r0), zero, [0, 0], tab, BIGBOX, 1.0, algorithm="bruteforce")
    assert abs(res.E[1]) < 1e-12 and res.E[2] == 0.0  # U_LJ(sigma) = 0
    rmin = 2.0 ** (1.0 / 6.0) * wl.SIGMA_O
    res = oracle.nonbonded(pos(rmin), zero, [0, 0], tab, BIGBOX, 1.0, algorithm="bruteforce")
    assert res.E[1] == pytest.approx(-wl.EPS_O, rel=1e-14)  # well depth -eps at 2^(1/6) sigma
    assert np.abs(res.F).max() < 1e-11  # force vanishes at the minimum
    # repulsive inside the minimum, attractive outside
    inside = oracle.nonbonded(pos(0.9 * rmin), zero, [0, 0], tab, BIGBOX, 1.0, algorithm="bruteforce")
    outside = oracle.nonbonded(pos(1.1 * rmin), zero, [0, 0], tab, BIGBOX, 1.0, algorithm="bruteforce")
    assert inside.F[0, 0] > 0 and outside.F[0, 0] < 0


def test_lorentz_berthelot_eq5():
    tab = oracle.lorentz_berthelot([0.3, 0.1, 0.25], [0.5, 2.0, 0.0])
    assert tab[0, 1, 0] == pytest.approx(0.2) and tab[1, 0, 0] == pytest.approx(0.2)
    assert tab[0, 1, 1] == pytest.approx(1.0) and tab[1, 0, 1] == pytest.approx(1.0)
    assert tab[0, 2, 1] == 0.0 and tab[2, 2, 1] == 0.0  # eps = 0 type has no LJ with anything
    assert tab[2, 2, 0] == pytest.approx(0.25)
    water = lj_table()
    assert water[0, 0, 0] == wl.SIGMA_O and water[0, 0, 1] == pytest.approx(wl.EPS_O)
    assert water[0, 1, 1] == 0.0 and water[1, 1, 1] == 0.0  # LJ on O only (configs[0])


# --- reaction field, Eq. (8) ------------------------------------------------------------------------------
@pytest.mark.parametrize("eps_rf,rc", [(78.5, 0.9), (78.5, 1.0), (2.0, 1.3), (1.0, 0.8)])
def test_rf_energy_vanishes_at_cutoff_and_force_limit(eps_rf, rc):
    # U_RFA(r_c) = 0 for any eps_rf, r_c (only holds with reading C-1); force limit 3 k_e qq / ((2eps+1) rc^2)
    r = rc * (1.0 - 1e-12)
    res, f = two_particles("H", "H", r, rc, eps_rf=eps_rf)
    assert abs(res.E[2]) < 1e-8
    assert f == pytest.approx(3.0 * KE * wl.Q_H**2 / ((2 * eps_rf + 1) * rc * rc), rel=1e-9)
    # just outside the cutoff: nothing at all
    res, f = two_particles("H", "H", rc * (1 + 1e-12), rc, eps_rf=eps_rf)
    assert res.E[0] == 0.0 and f == 0.0 and res.n_pairs == 0


# --- the cutoff-band force allowance of reading C-10 (the `allow` output) ------------------------------------
# SURVEY.md §8(c) C-10 prints the values: at r_c = 1.0, eps_rf = 78.5 the RF force jump at the cutoff is
# f(r_c) = 3 k_e q_i q_j / ((2 eps_rf + 1) r_c^2) = 1.835 (O-O), 0.917 (O-H), 0.459 (H-H) kJ mol^-1 nm^-1.
C10_JUMP = {("O", "O"): 1.835, ("O", "H"): 0.917, ("H", "H"): 0.459}


@pytest.mark.parametrize("kinds", sorted(C10_JUMP))
@pytest.mark.parametrize("offset,inside_band", [(-5e-6, True), (5e-6, True), (-2e-5, False), (2e-5, False)])
def test_allow_is_the_rf_force_jump_inside_the_band_and_zero_outside(kinds, offset, inside_band):
    """allow_i = sum over pairs with |r - r_c| < band of |f_ij| (reading C-10): for one pair at r_c + offset both atoms get
    the RF force jump f(r_c) when |offset| < band = 1e-5 and exactly 0 otherwise, on either side of the cutoff."""
    a, b = kinds
    rc = 1.0
    res, f = two_particles(a, b, rc + offset, rc, band=1e-5)
    closed = 3.0 * KE * abs(Q[a] * Q[b]) / ((2 * 78.5 + 1) * rc * rc)
    assert closed == pytest.approx(C10_JUMP[kinds], abs=5e-4)  # the survey's printed value (3 decimals)
    if inside_band:
        # f_RF(r) = k_e qq (1/r^2 - 2 k_rf r) is small at r_c because the two terms nearly cancel (1 - 2 k_rf = 0.019), so
        # d ln f / dr = -(2 + 2 k_rf) / (1 - 2 k_rf) = -157 per nm: |offset| = 5e-6 moves it by 7.8e-4 relative; LJ adds
        # its own 0.015 for O-O (SURVEY C-10)
        lj = 0.016 if kinds == ("O", "O") else 0.0
        assert res.allow[0] == pytest.approx(closed, abs=lj + 160 * abs(offset) * closed)
        assert res.allow[1] == res.allow[0]
    else:
        assert res.allow[0] == 0.0 and res.allow[1] == 0.0
    # the allowance never changes what is computed: forces only from the in-cutoff side
    assert (f != 0.0) == (offset < 0)


def test_allow_is_none_without_band_and_sparse_with_it():
    """band = 0 disables the allowance; with band = 1e-5 only atoms owning a pair within the band get a non-zero value
    (SURVEY C-10 expects ~2.8 % of atoms; a band 100x too wide, or an allowance summed over all pairs, fails here), and
    each value equals the sum of |f_ij| over exactly those pairs (recounted here by brute force in numpy)."""
    wb = wl.make_config(1)  # 9,000 atoms
    tab = lj_table()
    rc, band = 1.0, 1e-5
    res0 = oracle.nonbonded(wb.pos, wb.charge, wb.type, tab, wb.box, rc, excl_pairs=wb.excl_pairs, band=0.0)
    assert res0.allow is None
    res = oracle.nonbonded(wb.pos, wb.charge, wb.type, tab, wb.box, rc, excl_pairs=wb.excl_pairs, band=band)
    assert np.array_equal(res.F, res0.F) and np.array_equal(res.E, res0.E)
    n = wb.n_atoms
    frac = (res.allow > 0).mean()
    assert 0.0 < frac < 0.05, frac
    # independent recount: pairs within the band from scipy's periodic k-d tree, |f| from the closed RF form
    from scipy.spatial import cKDTree

    pos = wb.pos.astype(np.float64)
    tree = cKDTree(pos, boxsize=wb.box)
    outer = tree.query_pairs(rc + band, output_type="ndarray")
    d = pos[outer[:, 0]] - pos[outer[:, 1]]
    d -= wb.box * np.rint(d / wb.box)
    r = np.sqrt((d * d).sum(1))
    sel = np.abs(r - rc) < band
    i, j, r = outer[sel, 0], outer[sel, 1], r[sel]
    keep = (i // 3) != (j // 3)  # workloads.py: atoms 3m..3m+2 form one molecule and exclude one another
    i, j, r = i[keep], j[keep], r[keep]
    assert len(i) > 20 and len(np.unique(np.concatenate([i, j]))) == (res.allow > 0).sum()
    k_rf = (78.5 - 1) / ((2 * 78.5 + 1) * rc**3)
    qq = KE * wb.charge[i].astype(np.float64) * wb.charge[j].astype(np.float64)
    f_c = qq * (1.0 / r**3 - 2 * k_rf) * r
    both_o = (wb.type[i] == 0) & (wb.type[j] == 0)
    s6 = (wl.SIGMA_O / r) ** 6
    f_lj = np.where(both_o, 24 * wl.EPS_O * (2 * s6 * s6 - s6) / r, 0.0)
    want = np.zeros(n)
    np.add.at(want, i, np.abs(f_c + f_lj))
    np.add.at(want, j, np.abs(f_c + f_lj))
    assert np.allclose(res.allow, want, rtol=1e-9, atol=1e-12)


def test_rf_with_unit_dielectric_is_shifted_coulomb():
    # eps_rf = 1 => k_rf = 0, c_rf = 1/r_c: the textbook shifted Coulomb potential k_e qq (1/r - 1/r_c)
    res, f = two_particles("H", "H", 0.5, 2.0, eps_rf=1.0)
    assert res.E[2] == pytest.approx(KE * wl.Q_H**2 * (1 / 0.5 - 1 / 2.0), rel=1e-14)
    assert f == pytest.approx(KE * wl.Q_H**2 / 0.25, rel=1e-14)  # pure Coulomb force


def test_coulomb_constant_enters_linearly():
    a, _ = two_particles("O", "H", 0.4, 1.0, coulomb_const=1.0)
    b, _ = two_particles("O", "H", 0.4, 1.0, coulomb_const=KE)
    assert b.E[2] == pytest.approx(KE * a.E[2], rel=1e-14)
    assert b.E[1] == a.E[1]


# --- Ewald real space + exclusion correction --------------------------------------------------------------
@pytest.mark.parametrize("r", [0.09572, 0.2, 0.55, 0.97])
def test_ewald_real_plus_excluded_complement_is_plain_coulomb(r):
    # erfc + erf = 1: [k qq erfc(ar)/r] - [-k qq erf(ar)/r] = k qq / r, same for the forces
    real, f_real = two_particles("O", "H", r, 1.0, method=oracle.METHOD_EWALD_REAL)
    corr, f_corr = two_particles("O", "H", r, 1.0, method=oracle.METHOD_EWALD_REAL, excluded=True)
    qq = wl.Q_O * wl.Q_H
    assert real.E[2] - corr.E[3] == pytest.approx(KE * qq / r, rel=1e-13)
    assert f_real - f_corr == pytest.approx(KE * qq / r**2, rel=1e-12)


def test_ewald_exclusion_correction_small_r_limit_and_no_cutoff():
    alpha = 3.12
    corr, _ = two_particles("H", "H", 1e-7, 1.0, method=oracle.METHOD_EWALD_REAL, excluded=True, alpha=alpha)
    assert corr.E[3] == pytest.approx(-2 * alpha * KE * wl.Q_H**2 / math.sqrt(math.pi), rel=1e-9)
    # correction applies to excluded pairs beyond r_cut too (reading C-15)
    far, _ = two_particles("H", "H", 1.7, 1.0, method=oracle.METHOD_EWALD_REAL, excluded=True, alpha=alpha)
    assert far.E[3] == pytest.approx(-KE * wl.Q_H**2 * math.erf(alpha * 1.7) / 1.7, rel=1e-13)
    # alpha -> 0 turns the real-space term into plain Coulomb
    plain, f = two_particles("H", "H", 0.4, 1.0, method=oracle.METHOD_EWALD_REAL, alpha=1e-9)
    assert plain.E[2] == pytest.approx(KE * wl.Q_H**2 / 0.4, rel=1e-8)


# --- small periodic systems -------------------------------------------------------------------------------
def small_box(m=24, edge=2.2, seed=7):
    return wl.make_water_box(m, edge, seed)


def energy(pos, wb, box=None, method=oracle.METHOD_RF, r_cut=1.0, algorithm="bruteforce"):
    box = wb.box if box is None else box
    return oracle.nonbonded(pos, wb.charge, wb.type, lj_table(), box, r_cut, method=method,
                            excl_pairs=wb.excl_pairs, algorithm=algorithm)


def _no_pair_near_cutoff(pos, box, r_cut, margin):
    inner = oracle.neighbor_pairs(pos, box, r_cut - margin, None, "bruteforce")
    outer = oracle.neighbor_pairs(pos, box, r_cut + margin, None, "bruteforce")
    return len(inner) == len(outer)


@pytest.mark.parametrize("method", [oracle.METHOD_RF, oracle.METHOD_EWALD_REAL])
def test_forces_are_minus_finite_difference_gradient(method):
    wb = small_box()
    pos = wb.pos.astype(np.float64)
    assert _no_pair_near_cutoff(pos, wb.box, 1.0, 1e-4)
    res = energy(pos, wb, method=method)
    h = 1e-6
    rng = np.random.default_rng(3)
    for i in rng.choice(wb.n_atoms, size=10, replace=False):
        for a in range(3):
            p, m = pos.copy(), pos.copy()
            p[i, a] += h
            m[i, a] -= h
            fd = -(energy(p, wb, method=method).E[0] - energy(m, wb, method=method).E[0]) / (2 * h)
            assert res.F[i, a] == pytest.approx(fd, rel=2e-6, abs=2e-4)


@pytest.mark.parametrize("method", [oracle.METHOD_RF, oracle.METHOD_EWALD_REAL])
def test_newton_third_law_and_virial_symmetry(method):
    wb = small_box(m=40, edge=2.4, seed=11)
    res = energy(wb.pos, wb, method=method)
    assert np.abs(res.F.sum(axis=0)).max() < 1e-9
    assert np.abs(res.W - res.W.T).max() < 1e-9
    assert res.E[0] == pytest.approx(res.E[1] + res.E[2] + res.E[3], rel=1e-15)


@pytest.mark.parametrize("method", [oracle.METHOD_RF, oracle.METHOD_EWALD_REAL])
def test_virial_is_minus_strain_derivative_of_energy(method):
    # W_aa = -dE/d(eps_aa) under x_a -> (1+eps) x_a, L_a -> (1+eps) L_a with r_c fixed; tr W = -dE/dlambda
    wb = small_box(m=30, edge=2.3, seed=5)
    pos = wb.pos.astype(np.float64)
    assert _no_pair_near_cutoff(pos, wb.box, 1.0, 1e-4)
    res = energy(pos, wb, method=method)
    h = 1e-7
    for a in range(3):
        def scaled(s):
            p, b = pos.copy(), wb.box.copy()
            p[:, a] *= s
            b[a] *= s
            return energy(p, wb, box=b, method=method).E[0]
        fd = -(scaled(1 + h) - scaled(1 - h)) / (2 * h)
        assert res.W[a, a] == pytest.approx(fd, rel=1e-5, abs=1e-3)
    fd_iso = -(energy(pos * (1 + h), wb, box=wb.box * (1 + h), method=method).E[0]
               - energy(pos * (1 - h), wb, box=wb.box * (1 - h), method=method).E[0]) / (2 * h)
    assert np.trace(res.W) == pytest.approx(fd_iso, rel=1e-5, abs=1e-3)


def test_translation_and_periodic_image_invariance():
    wb = small_box()
    pos = wb.pos.astype(np.float64)
    ref = energy(pos, wb)
    shift = np.array([0.37, -5.21, 13.9])  # arbitrary, larger than the box in two components
    moved = energy(pos + shift, wb)
    assert moved.E[0] == pytest.approx(ref.E[0], rel=1e-11)
    assert np.allclose(moved.F, ref.F, rtol=0, atol=1e-7)
    assert moved.n_pairs == ref.n_pairs
    img = pos.copy()
    img[5] += np.array([wb.box[0], 0.0, -2 * wb.box[2]])
    imaged = energy(img, wb)
    assert imaged.E[0] == pytest.approx(ref.E[0], rel=1e-12)
    assert np.allclose(imaged.F, ref.F, rtol=0, atol=1e-8)
    # neighbour set unchanged as well
    a = oracle.neighbor_pairs(pos, wb.box, 1.1, wb.excl_pairs, "bruteforce")
    b = oracle.neighbor_pairs(img, wb.box, 1.1, wb.excl_pairs, "bruteforce")
    assert np.array_equal(a, b)


def test_exclusions_single_and_double_water():
    one = wl.make_water_box(1, 3.0, 1)
    res = energy(one.pos, one)
    assert res.n_pairs == 0 and res.E[0] == 0.0 and np.all(res.F == 0.0)
    assert len(oracle.neighbor_pairs(one.pos, one.box, 1.1, one.excl_pairs, "bruteforce")) == 0
    # without the exclusion list the three intramolecular pairs appear
    assert len(oracle.neighbor_pairs(one.pos, one.box, 1.1, None, "bruteforce")) == 3
    two = wl.make_water_box(8, 0.9 * 2, 2)  # 2x2x2 lattice sites, all 8 used -> pick the first two molecules
    pos = two.pos[:6].astype(np.float64)
    pos[3:6] = pos[0:3] + np.array([0.3, 0.05, -0.02])
    pairs = oracle.neighbor_pairs(pos, np.array([5.0, 5.0, 5.0]), 1.1, two.excl_pairs[:6], "bruteforce")
    assert len(pairs) == 9 and all(i < 3 <= j for i, j in pairs)  # exactly the 9 intermolecular pairs
    res = oracle.nonbonded(pos, two.charge[:6], two.type[:6], lj_table(), [5.0, 5.0, 5.0], 1.0,
                           excl_pairs=two.excl_pairs[:6], algorithm="bruteforce")
    assert res.n_pairs == 9


# --- the two enumerations agree; the set agrees with scipy ------------------------------------------------
@pytest.mark.parametrize("case", ["config0", "config1", "slab_n2", "ewald_small"])
def test_celllist_equals_bruteforce(case):
    if case == "config0":  # degenerate 1x1x1 grid, r_nl > L/2
        wb, rc, skin, method = wl.make_config(0), 0.9, 0.1, oracle.METHOD_RF
        box = wb.box
    elif case == "config1":
        wb, rc, skin, method = wl.make_config(1), 1.0, 0.1, oracle.METHOD_RF
        box = wb.box
    elif case == "slab_n2":  # 2 cells along x and y, 3 along z: stencil de-duplication
        wb, rc, skin, method = wl.make_water_box(150, 2.5, 21), 1.0, 0.1, oracle.METHOD_RF
        box = np.array([2.5, 2.3, 3.4])
    else:
        wb, rc, skin, method = wl.make_water_box(100, 2.2, 4), 1.0, 0.1, oracle.METHOD_EWALD_REAL
        box = wb.box
    tab = lj_table()
    kw = dict(method=method, excl_pairs=wb.excl_pairs, band=1e-5)
    b = oracle.nonbonded(wb.pos, wb.charge, wb.type, tab, box, rc, algorithm="bruteforce", **kw)
    c = oracle.nonbonded(wb.pos, wb.charge, wb.type, tab, box, rc, algorithm="celllist", **kw)
    assert b.n_pairs == c.n_pairs
    scale = np.sqrt((b.F**2).sum(axis=1).mean())
    assert np.abs(b.F - c.F).max() < 1e-12 * scale
    assert np.allclose(b.E, c.E, rtol=1e-12, atol=1e-9)
    assert np.allclose(b.W, c.W, rtol=1e-12, atol=1e-8)
    assert np.array_equal(b.allow, c.allow)
    pb = oracle.neighbor_pairs(wb.pos, box, rc + skin, wb.excl_pairs, "bruteforce")
    pc = oracle.neighbor_pairs(wb.pos, box, rc + skin, wb.excl_pairs, "celllist")
    assert np.array_equal(pb, pc)


def test_neighbor_set_matches_scipy_kdtree():
    from scipy.spatial import cKDTree

    wb = wl.make_config(1)  # 9,000 atoms
    r_nl = 1.1
    pos = wb.pos.astype(np.float64)
    tree = cKDTree(pos, boxsize=wb.box)
    kd = tree.query_pairs(r_nl, output_type="ndarray")
    kd = np.sort(kd, axis=1)
    n = wb.n_atoms
    key = kd[:, 0].astype(np.int64) * n + kd[:, 1]
    excl_key = wb.excl_pairs[:, 0].astype(np.int64) * n + wb.excl_pairs[:, 1]
    key = np.setdiff1d(key, excl_key)
    # scipy uses r <= r_nl, the oracle r < r_nl: remove ties (none expected) by checking sizes
    mine = oracle.neighbor_pairs(pos, wb.box, r_nl, wb.excl_pairs, "celllist")
    mine_key = mine[:, 0].astype(np.int64) * n + mine[:, 1]
    assert np.array_equal(np.sort(key), mine_key)  # oracle output is lexicographically sorted already
    assert np.all(np.diff(mine_key) > 0)


def test_config0_matches_surveyors_independent_numbers():
    vals = {}
    with open(os.path.join(GOLDEN, "config0_magnitudes.txt")) as fh:
        for line in fh:
            if not line.startswith("#") and line.strip():
                k, v = line.split()
                vals[k] = float(v)
    wb = wl.make_config(0)
    res = oracle.nonbonded(wb.pos, wb.charge, wb.type, lj_table(), wb.box, 0.9, excl_pairs=wb.excl_pairs,
                           algorithm="bruteforce")
    assert res.n_pairs == int(vals["pairs_lt_rcut"])
    assert len(oracle.neighbor_pairs(wb.pos, wb.box, 1.0, wb.excl_pairs, "bruteforce")) == int(vals["pairs_lt_rnl"])
    assert res.E[0] == pytest.approx(vals["E_total_approx"], abs=0.6)
    assert np.sqrt((res.F**2).sum(axis=1).mean()) == pytest.approx(vals["rmsF_approx"], abs=0.6)


# --- rebuild trigger, PAPER.md:175 ------------------------------------------------------------------------
def test_needs_rebuild_definition_and_strictness():
    ref = np.zeros((5, 3))
    pos = ref.copy()
    skin = 0.1
    assert oracle.needs_rebuild(pos, ref, skin) == (False, 0.0)
    pos[3] = [0.03, 0.04, 0.0]  # |dr| = 0.05 = skin/2 exactly: strict ">" => no rebuild
    flag, m = oracle.needs_rebuild(pos, ref, skin)
    assert m == pytest.approx(0.05) and flag is False
    pos[3] = [0.03, 0.04, 0.001]
    assert oracle.needs_rebuild(pos, ref, skin)[0] is True
    # Euclidean norm, not max-norm: every component is < skin/2 but |dr| = 0.0520 > 0.05
    pos[3] = [0.03, 0.03, 0.03]
    assert oracle.needs_rebuild(pos, ref, skin)[0] is True
    pos[3] = [0.028, 0.028, 0.028]  # |dr| = 0.0485 < 0.05
    assert oracle.needs_rebuild(pos, ref, skin)[0] is False
    # raw coordinates: a jump by a whole box length counts as displacement (caller must not re-wrap, §8(b))
    pos[3] = [2.0, 0.0, 0.0]
    assert oracle.needs_rebuild(pos, ref, skin) == (True, 2.0)


def test_verlet_list_validity_invariant():
    # a list built with radius r_c + r_g holds every pair within r_c for as long as
    # no atom has moved more than r_g/2.
    wb = small_box(m=60, edge=2.6, seed=9)
    rc, skin = 1.0, 0.1
    pos0 = wb.pos.astype(np.float64)
    listed = oracle.neighbor_pairs(pos0, wb.box, rc + skin, wb.excl_pairs, "bruteforce")
    n = wb.n_atoms
    listed_key = set((listed[:, 0].astype(np.int64) * n + listed[:, 1]).tolist())
    rng = np.random.default_rng(0)
    step = rng.standard_normal(pos0.shape)
    step *= (0.5 * skin * 0.999) / np.linalg.norm(step, axis=1, keepdims=True)  # every atom moves just under skin/2
    pos1 = pos0 + step
    assert oracle.needs_rebuild(pos1, pos0, skin)[0] is False
    now = oracle.neighbor_pairs(pos1, wb.box, rc, wb.excl_pairs, "bruteforce")
    now_key = set((now[:, 0].astype(np.int64) * n + now[:, 1]).tolist())
    assert now_key <= listed_key


# --- LJ switching function, Eq. (6) ---------------------------------------------------------
def test_lj_switch_special_values():
    """S(x) = 1 - 6x^5 + 15x^4 - 10x^3 with x = (r - r_s)/(r_c - r_s): S = 1 below r_s, S(1/2) = 1/2 exactly with
    S'(1/2) = -15/8, S(1) = S'(1) = 0.  Checked against the plain potential, which the closed forms above pin."""
    rs, rc = 0.8, 1.0
    for r in (0.35, 0.6, 0.7999):  # below r_s: identical to the unswitched potential
        a, fa = two_particles("O", "O", r, rc, r_switch=rs)
        b, fb = two_particles("O", "O", r, rc)
        assert a.E[1] == b.E[1] and fa == fb
    plain, f_plain = two_particles("O", "O", 0.9, rc)
    sw, f_sw = two_particles("O", "O", 0.9, rc, r_switch=rs)
    assert sw.E[1] == pytest.approx(0.5 * plain.E[1], rel=1e-14)
    assert sw.E[2] == plain.E[2]  # Coulomb untouched
    # the neutral LJ-only pair isolates the LJ force: F = S F_LJ - S'(x)/(r_c - r_s) U_LJ = F_LJ/2 + (15/8)/0.2 U_LJ
    z_plain, fz_plain = _lj_only_pair(0.9, rc, 0.0)
    z_sw, fz_sw = _lj_only_pair(0.9, rc, rs)
    assert fz_sw == pytest.approx(0.5 * fz_plain + (15.0 / 8.0) / (rc - rs) * z_plain.E[1], rel=1e-13)
    assert f_sw - f_plain == pytest.approx(fz_sw - fz_plain, rel=1e-9)  # and the charged pair differs by the same amount
    # at the cutoff both the energy and the force vanish like (1 - x)^3 and (1 - x)^2
    near, f_near = _lj_only_pair(rc - 1e-7, rc, rs)
    assert abs(near.E[1]) < 1e-18 and abs(f_near) < 1e-12


def _lj_only_pair(r, r_cut, r_switch):
    u = np.array([0.6, 0.0, 0.8])
    pos = np.array([[10.0, 11.0, 12.0] + r * u, [10.0, 11.0, 12.0]])
    res = oracle.nonbonded(pos, [0.0, 0.0], [0, 0], lj_table(), BIGBOX, r_cut, algorithm="bruteforce", r_switch=r_switch)
    return res, float(res.F[0] @ u)


def test_lj_switch_forces_are_minus_gradient_and_continuous():
    """Finite-difference gradient through the whole switching interval, and continuity of U and F at r_s."""
    rs, rc = 0.75, 1.0
    h = 1e-6
    for r in np.linspace(0.70, 0.999, 14):
        e = lambda rr: _lj_only_pair(rr, rc, rs)[0].E[1]
        f = _lj_only_pair(r, rc, rs)[1]
        assert f == pytest.approx(-(e(r + h) - e(r - h)) / (2 * h), rel=5e-6, abs=1e-9)
    lo, f_lo = _lj_only_pair(rs - 1e-9, rc, rs)
    hi, f_hi = _lj_only_pair(rs + 1e-9, rc, rs)
    assert hi.E[1] == pytest.approx(lo.E[1], rel=1e-7) and f_hi == pytest.approx(f_lo, rel=1e-6)


def test_lj_switch_many_body_cell_list_equals_bruteforce():
    wb = small_box()
    lj = lj_table()
    a = oracle.nonbonded(wb.pos, wb.charge, wb.type, lj, wb.box, 1.0, excl_pairs=wb.excl_pairs, algorithm="bruteforce", r_switch=0.8)
    b = oracle.nonbonded(wb.pos, wb.charge, wb.type, lj, wb.box, 1.0, excl_pairs=wb.excl_pairs, algorithm="celllist", r_switch=0.8)
    c = oracle.nonbonded(wb.pos, wb.charge, wb.type, lj, wb.box, 1.0, excl_pairs=wb.excl_pairs, algorithm="celllist")
    assert np.abs(a.F - b.F).max() < 1e-9 and a.E[1] == pytest.approx(b.E[1], rel=1e-13)
    assert a.E[1] != c.E[1] and a.E[2] == pytest.approx(c.E[2], rel=1e-13)


# --- 1-4 exceptions (reading C-21) -----------------------------------------------------------------
def _exception_pair(kind_a, kind_b, r, s_c, s_lj, method=oracle.METHOD_RF):
    u = np.array([0.48, -0.6, 0.64])
    pos = np.array([[10.0, 11.0, 12.0] + r * u, [10.0, 11.0, 12.0]])
    pair = np.array([[0, 1]], dtype=np.int32)
    res = oracle.nonbonded(pos, [Q[kind_a], Q[kind_b]], [TYPE[kind_a], TYPE[kind_b]], lj_table(), BIGBOX, 1.0, method=method,
                           excl_pairs=pair, exceptions=(pair, np.array([[s_c, s_lj]])), algorithm="bruteforce")
    return res, float(res.F[0] @ u)


def test_exception_is_scaled_bare_lj_plus_bare_coulomb():
    """An exception pair contributes s_lj U_LJ (Eq. 4) + s_c k_e q q / r (Eq. 7) and nothing else.  The LJ part is
    checked against the pinned pair potential; the bare Coulomb part through erfc + erf = 1: the Ewald real-space term
    of the free pair minus the exclusion correction of the excluded pair IS k_e q q / r (and likewise the forces)."""
    r = 0.31
    free, f_free = two_particles("O", "O", r, 1.0)                                    # LJ + RF, pinned above
    ew, f_ew = two_particles("O", "O", r, 1.0, method=oracle.METHOD_EWALD_REAL)       # LJ + erfc/r
    corr, f_corr = two_particles("O", "O", r, 1.0, method=oracle.METHOD_EWALD_REAL, excluded=True)  # -erf/r
    bare_e, bare_f = ew.E[2] - corr.E[3], (f_ew - f_corr)                              # includes the LJ force once
    lj_e = free.E[1]
    z, f_lj = _lj_only_pair(r, 1.0, 0.0)
    for s_c, s_lj in ((1.0, 1.0), (0.5, 0.5), (0.8333, 0.5), (0.0, 1.0), (1.0, 0.0)):
        res, f = _exception_pair("O", "O", r, s_c, s_lj)
        assert res.E[1] == pytest.approx(s_lj * lj_e, rel=1e-11, abs=1e-15)  # r is rebuilt from rounded coordinates
        assert res.E[2] == pytest.approx(s_c * bare_e, rel=1e-12, abs=1e-12)
        assert res.E[3] == 0.0 and res.E[0] == pytest.approx(res.E[1] + res.E[2], rel=1e-15)
        assert f == pytest.approx(s_lj * f_lj + s_c * (bare_f - f_lj), rel=1e-11, abs=1e-9)
    # under Ewald the pair is still an excluded pair: its -erf correction stays, the exception is added on top
    res, _ = _exception_pair("O", "H", 0.2, 0.5, 0.0, method=oracle.METHOD_EWALD_REAL)
    only_corr, _ = two_particles("O", "H", 0.2, 1.0, method=oracle.METHOD_EWALD_REAL, excluded=True)
    assert res.E[3] == pytest.approx(only_corr.E[3], rel=1e-12) and res.E[2] != 0.0


def test_exception_forces_are_minus_gradient_and_newton():
    wb = small_box(m=20, edge=2.3, seed=8)
    pos = wb.pos.astype(np.float64)
    exc = wb.excl_pairs[::3].copy()  # a third of the intramolecular pairs become scaled exceptions
    scale = np.tile(np.array([[0.8333, 0.5]]), (exc.shape[0], 1))
    lj = oracle.lorentz_berthelot([wl.SIGMA_O, 0.1], [wl.EPS_O, 0.2])  # LJ on H too, so the LJ scale acts on O-H pairs

    def en(p):
        return oracle.nonbonded(p, wb.charge, wb.type, lj, wb.box, 1.0, excl_pairs=wb.excl_pairs, exceptions=(exc, scale),
                                algorithm="bruteforce")

    res = en(pos)
    base = oracle.nonbonded(pos, wb.charge, wb.type, lj, wb.box, 1.0, excl_pairs=wb.excl_pairs, algorithm="bruteforce")
    assert res.E[0] != base.E[0]
    assert np.abs(res.F.sum(axis=0)).max() < 1e-9 and np.abs(res.W - res.W.T).max() < 1e-9
    h = 1e-6
    for i in (int(exc[0, 0]), int(exc[1, 1]), int(exc[-1, 0])):
        for a in range(3):
            p, m = pos.copy(), pos.copy()
            p[i, a] += h
            m[i, a] -= h
            assert res.F[i, a] == pytest.approx(-(en(p).E[0] - en(m).E[0]) / (2 * h), rel=2e-6, abs=2e-4)
    with pytest.raises(ValueError):  # an exception must also be an exclusion
        oracle.nonbonded(pos, wb.charge, wb.type, lj, wb.box, 1.0, excl_pairs=wb.excl_pairs[1:],
                         exceptions=(wb.excl_pairs[:1], np.array([[1.0, 1.0]])), algorithm="bruteforce")


# --- velocity Verlet, steps 1, 2, 5 of PAPER.md:281-292 -----------------------------------------------------------
def _vv_run(x, v, force_fn, inv_m, dt, n):
    f = force_fn(x)
    for _ in range(n):
        x, v = oracle.vv_kick_drift(x, v, f, inv_m, dt)
        f = force_fn(x)
        v = oracle.vv_kick(v, f, inv_m, dt)
    return x, v


def test_velocity_verlet_is_exact_for_a_constant_force():
    """x(t) = x0 + v0 t + F t^2 / (2 m), v(t) = v0 + F t / m: velocity Verlet reproduces it exactly; the units need no
    conversion factor (kJ mol^-1 nm^-1 / amu = nm ps^-2)."""
    x0 = np.array([[0.1, -0.2, 0.3], [1.0, 2.0, 3.0]])
    v0 = np.array([[0.5, 0.0, -1.0], [0.0, 0.25, 0.0]])
    F = np.array([[10.0, -4.0, 2.5], [-3.0, 0.0, 8.0]])
    m = np.array([15.9994, 1.008])
    dt, n = 0.002, 50
    x, v = _vv_run(x0, v0, lambda _x: F, 1.0 / m, dt, n)
    t = n * dt
    assert np.allclose(x, x0 + v0 * t + 0.5 * F / m[:, None] * t * t, rtol=0, atol=1e-13)
    assert np.allclose(v, v0 + F / m[:, None] * t, rtol=0, atol=1e-13)


def test_velocity_verlet_harmonic_oscillator_closed_form_and_reversibility():
    """For F = -k x velocity Verlet is the exact flow of a shadow oscillator: x_n = x_0 cos(n phi) with
    cos(phi) = 1 - (omega dt)^2 / 2 (v_0 = 0).  Negating the velocities retraces the trajectory."""
    k, m, dt, n = 300.0, 2.0, 0.004, 137
    w2 = k / m
    x0 = np.array([[0.7, 0.0, 0.0]])
    v0 = np.zeros((1, 3))
    x, v = _vv_run(x0, v0, lambda xx: -k * xx, np.array([1.0 / m]), dt, n)
    phi = np.arccos(1.0 - 0.5 * w2 * dt * dt)
    assert x[0, 0] == pytest.approx(0.7 * np.cos(n * phi), abs=1e-12)
    xb, vb = _vv_run(x, -v, lambda xx: -k * xx, np.array([1.0 / m]), dt, n)
    assert np.allclose(xb, x0, atol=1e-12) and np.allclose(vb, -v0, atol=1e-12)


# --- edge list with distance vectors and shifts ------------------------------------------------
def test_edge_vectors_identities():
    """d = r_a - r_b - shift L with every component of d in [-L/2, L/2]; |d| < r_list for listed pairs; zero shifts when
    the atoms sit far from the faces of a huge box; a pair across a face gets shift -1/+1 and the short vector."""
    wb = small_box()
    pairs = oracle.neighbor_pairs(wb.pos, wb.box, 0.9, wb.excl_pairs, "bruteforce")
    d, s = oracle.edge_vectors(wb.pos, wb.box, pairs)
    pos = wb.pos.astype(np.float64)
    assert np.allclose(d, pos[pairs[:, 0]] - pos[pairs[:, 1]] - s * wb.box, atol=1e-15)
    assert np.all(np.abs(d) <= 0.5 * wb.box + 1e-12) and np.all(np.sqrt((d * d).sum(1)) < 0.9)
    two = np.array([[0.05, 1.0, 1.0], [2.95, 1.0, 1.0]])
    d2, s2 = oracle.edge_vectors(two, [3.0, 3.0, 3.0], [[0, 1]])
    assert np.allclose(d2, [[0.1, 0.0, 0.0]]) and s2.tolist() == [[-1, 0, 0]]
    d3, s3 = oracle.edge_vectors([[10.0, 11.0, 12.0], [10.3, 11.0, 12.4]], BIGBOX, [[0, 1]])
    assert s3.tolist() == [[0, 0, 0]] and np.allclose(d3, [[-0.3, 0.0, -0.4]])


# --- non-periodic systems by embedding into a virtual box ------------------------------------------
def test_virtual_box_embedding_equals_open_boundaries():
    """A periodic box of edge extent + r_c + 2 skin around an isolated cluster gives the same pair set, energy and
    forces as a box so large that periodicity cannot matter: the images are farther away than r_c + skin."""
    wb = small_box(m=30, edge=2.3, seed=21)
    pos = wb.pos.astype(np.float64) + np.array([-0.4, 7.0, 3.3])  # anywhere, partly negative
    ext = pos.max(0) - pos.min(0)
    rc, skin = 0.9, 0.1
    vbox = ext + rc + 2 * skin
    huge = 20.0 * vbox
    a = oracle.nonbonded(pos, wb.charge, wb.type, lj_table(), vbox, rc, excl_pairs=wb.excl_pairs, algorithm="bruteforce")
    b = oracle.nonbonded(pos, wb.charge, wb.type, lj_table(), huge, rc, excl_pairs=wb.excl_pairs, algorithm="bruteforce")
    assert a.n_pairs == b.n_pairs and np.abs(a.F - b.F).max() < 1e-9 and a.E[0] == pytest.approx(b.E[0], rel=1e-12)
    pa = oracle.neighbor_pairs(pos, vbox, rc + skin, wb.excl_pairs, "celllist")
    pb = oracle.neighbor_pairs(pos, huge, rc + skin, wb.excl_pairs, "bruteforce")
    assert np.array_equal(pa, pb)
    # one skin less and a pair across the seam can enter the list: the margin is needed
    tight = ext + 0.5 * (rc + skin)
    assert oracle.neighbor_pairs(pos, np.maximum(tight, 2 * rc + 1e-3), rc + skin, wb.excl_pairs, "bruteforce").shape[0] >= pb.shape[0]


# --- long-range dispersion correction (reading C-22) ------------------------------------------------
def test_dispersion_correction_textbook_tail_and_switch_limits():
    """Plain truncation: the textbook tail 8 pi N^2 eps / V [sigma^12 / (9 r_c^9) - sigma^6 / (3 r_c^3)] for one species.
    With the switch the correction lies between the plain values at r_s and at r_c and tends to the plain value as
    r_s -> r_c; it is extensive (doubling the box at constant density doubles it)."""
    n_o, vol = 1000.0, 30.0
    types = np.zeros(int(n_o), dtype=np.int32)
    box = np.array([vol ** (1 / 3)] * 3)
    tab = lj_table()
    s, e, rc = wl.SIGMA_O, wl.EPS_O, 1.0
    textbook = 8.0 * np.pi * n_o * n_o * e / vol * (s ** 12 / (9 * rc ** 9) - s ** 6 / (3 * rc ** 3))
    got, w = oracle.dispersion_correction(types, tab, box, rc)
    assert got == pytest.approx(textbook, rel=1e-12) and np.allclose(w, got * np.eye(3))
    at_rs = oracle.dispersion_correction(types, tab, box, 0.8)[0]
    sw = oracle.dispersion_correction(types, tab, box, rc, r_switch=0.8)[0]
    assert at_rs < sw < got < 0.0  # attractive tail; more of it is missing the earlier the potential is cut
    assert oracle.dispersion_correction(types, tab, box, rc, r_switch=rc - 1e-7)[0] == pytest.approx(got, rel=1e-6)
    big = oracle.dispersion_correction(np.zeros(2000, dtype=np.int32), tab, box * 2 ** (1 / 3), rc)[0]
    assert big == pytest.approx(2 * got, rel=1e-12)
    # hydrogens (epsilon = 0) do not contribute
    mixed = oracle.dispersion_correction(np.concatenate([types, np.ones(2000, dtype=np.int32)]), tab, box, rc)[0]
    assert mixed == pytest.approx(got, rel=1e-14)


# --- rigid-water position constraints (step 3 of PAPER.md:281-292; SETTLE) ---------------------------
def test_shake_water_satisfies_constraints_and_conserves_momentum():
    """The constrained positions have the rigid geometry to 1e-12; the correction is a sum of pair displacements weighted
    by inverse mass, so it leaves every molecule's centre of mass where the unconstrained step put it; an already rigid
    configuration is left untouched; a rigid translation + small rotation of the old molecule is reproduced."""
    wb = small_box(m=40, edge=2.4, seed=4)
    d_hh = 2.0 * wl.R_OH * np.sin(np.radians(wl.ANGLE_HOH_DEG) / 2.0)
    x0 = wb.pos.astype(np.float64)
    x0 = oracle.shake_water(x0, x0, wb.mass, wl.R_OH, d_hh)  # the workload stores fp32: make it rigid in fp64 first
    rng = np.random.default_rng(1)
    x1 = x0 + rng.normal(0.0, 0.004, size=x0.shape)  # an unconstrained step of a few pm
    xc = oracle.shake_water(x0, x1, wb.mass, wl.R_OH, d_hh)
    m = xc.reshape(-1, 3, 3)
    for i, j, d in ((0, 1, wl.R_OH), (0, 2, wl.R_OH), (1, 2, d_hh)):
        assert np.abs(np.linalg.norm(m[:, i] - m[:, j], axis=1) - d).max() < 1e-12
    w = wb.mass.reshape(-1, 3, 1)
    com = lambda p: (p.reshape(-1, 3, 3) * w).sum(1) / w.sum(1)
    assert np.abs(com(xc) - com(x1)).max() < 1e-13
    assert np.abs(oracle.shake_water(x0, x0, wb.mass, wl.R_OH, d_hh) - x0).max() < 1e-13
    shift = x0 + np.array([0.01, -0.02, 0.005])
    assert np.abs(oracle.shake_water(x0, shift, wb.mass, wl.R_OH, d_hh) - shift).max() < 1e-12


def test_shake_water_runs_to_convergence_for_a_nearly_linear_molecule():
    """A 170-degree triangle makes the three bond vectors almost dependent: the sweeps need thousands of iterations (water
    needs ~30).  The answer must still satisfy the constraints to 1e-13, keep every centre of mass, not move when the cap is
    raised further -- and a cap that is too small must raise instead of returning the unconverged positions (which are
    8e-6 nm off here, the size of an fp32 parity bar)."""
    d_oh, m_c, m_e = 0.11, 12.0, 3.0
    d_ee = 2.0 * d_oh * np.sin(np.radians(170.0) / 2.0)
    rng = np.random.default_rng(9)
    h = np.radians(85.0)
    tri = np.array([[0.0, 0.0, 0.0], [d_oh * np.sin(h), 0.0, d_oh * np.cos(h)], [-d_oh * np.sin(h), 0.0, d_oh * np.cos(h)]])
    n = 50
    x0 = (tri[None] + rng.uniform(0.0, 6.0, size=(n, 1, 3))).reshape(-1, 3)
    mass = np.tile([m_c, m_e, m_e], n)
    x1 = x0 + 0.001 * rng.normal(0.0, 1.5, size=x0.shape) / np.sqrt(mass)[:, None]
    xc = oracle.shake_water(x0, x1, mass, d_oh, d_ee)
    m = xc.reshape(-1, 3, 3)
    for i, j, d in ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_ee)):
        assert np.abs(np.linalg.norm(m[:, i] - m[:, j], axis=1) - d).max() < 1e-13
    w = mass.reshape(-1, 3, 1)
    com = lambda p: (p.reshape(-1, 3, 3) * w).sum(1) / w.sum(1)
    assert np.abs(com(xc) - com(x1)).max() < 1e-13
    assert np.abs(oracle.shake_water(x0, x1, mass, d_oh, d_ee, max_iter=400000) - xc).max() == 0.0
    with pytest.raises(RuntimeError, match="not converged"):
        oracle.shake_water(x0, x1, mass, d_oh, d_ee, max_iter=500)
    v = rng.normal(0.0, 1.0, size=x0.shape) / np.sqrt(mass)[:, None]
    vc = oracle.rattle_water_velocities(xc, v, mass).reshape(-1, 3, 3)
    for i, j in ((0, 1), (0, 2), (1, 2)):
        assert np.abs(((vc[:, i] - vc[:, j]) * (m[:, i] - m[:, j])).sum(1)).max() < 1e-14
    with pytest.raises(RuntimeError, match="not converged"):
        oracle.rattle_water_velocities(xc, v, mass, max_iter=20)


def test_rattle_water_velocities_pins():
    """Step 6: after the velocity constraint no bond length changes to first order (v_ij . r_ij = 0);
    the impulses are internal and central, so each molecule keeps its linear and angular momentum; a rigid-body velocity
    field v = V + omega x r already satisfies the constraints and is returned unchanged; and the result is the projection
    that removes exactly the three internal degrees of freedom: kinetic energy never increases."""
    wb = small_box(m=40, edge=2.4, seed=5)
    x = wb.pos.astype(np.float64)
    mass = wb.mass.astype(np.float64)
    rng = np.random.default_rng(2)
    v = rng.normal(0.0, 1.0, size=x.shape) / np.sqrt(mass)[:, None]
    vc = oracle.rattle_water_velocities(x, v, mass)
    X, V, VC, M = x.reshape(-1, 3, 3), v.reshape(-1, 3, 3), vc.reshape(-1, 3, 3), mass.reshape(-1, 3, 1)
    for i, j in ((0, 1), (0, 2), (1, 2)):
        assert np.abs(((VC[:, i] - VC[:, j]) * (X[:, i] - X[:, j])).sum(1)).max() < 1e-15
    assert np.abs((M * VC).sum(1) - (M * V).sum(1)).max() < 1e-13
    assert np.abs((M * np.cross(X, VC)).sum(1) - (M * np.cross(X, V)).sum(1)).max() < 1e-13
    assert (M * VC * VC).sum() < (M * V * V).sum()
    com = (M * X).sum(1, keepdims=True) / M.sum(1, keepdims=True)
    omega = rng.normal(0.0, 3.0, size=(X.shape[0], 1, 3))
    rigid = rng.normal(0.0, 0.5, size=(X.shape[0], 1, 3)) + np.cross(omega, X - com)
    assert np.abs(oracle.rattle_water_velocities(x, rigid.reshape(-1, 3), mass) - rigid.reshape(-1, 3)).max() < 1e-14
    # 9 velocity components - 3 constraints: the removed part is 3-dimensional per molecule and mass-orthogonal to the rest
    assert np.abs((M * (V - VC) * VC).sum((1, 2))).max() < 1e-13


def test_berendsen_thermostat_pins():
    """Step 7 (Berendsen rescaling).  The rescaled temperature obeys the linear relaxation
    T' = T + (dt/tau)(T0 - T) exactly, so n applications give T0 + (T - T0)(1 - dt/tau)^n; dt = tau lands on T0 in one
    step; T = T0 is a fixed point; one atom of mass m and speed v has K = m v^2 / 2; velocities drawn from the
    Maxwell-Boltzmann distribution at T0 (sigma^2 = k_B T0 / m per component) measure T0 within 4 standard errors; and k_B
    is R = N_A k (both exact SI constants)."""
    assert oracle.K_B == pytest.approx(6.02214076e23 * 1.380649e-23 * 1e-3, rel=1e-12)
    assert oracle.kinetic_energy([[3.0, 4.0, 12.0]], [2.0]) == pytest.approx(169.0, rel=1e-15)
    rng = np.random.default_rng(3)
    n = 20000
    mass = rng.choice(np.array([15.9994, 1.008]), size=n)
    T0 = 300.0
    v = rng.normal(size=(n, 3)) * np.sqrt(oracle.K_B * T0 / mass)[:, None]
    n_dof = 3 * n
    T = 2.0 * oracle.kinetic_energy(v, mass) / (n_dof * oracle.K_B)
    assert abs(T - T0) < 4.0 * T0 * np.sqrt(2.0 / n_dof)
    hot = v * 1.3
    Th = 2.0 * oracle.kinetic_energy(hot, mass) / (n_dof * oracle.K_B)
    cur, dt, tau = hot, 0.002, 0.1
    for k in range(1, 6):
        cur, T_before = oracle.berendsen(cur, mass, n_dof, T0, tau, dt)
        T_after = 2.0 * oracle.kinetic_energy(cur, mass) / (n_dof * oracle.K_B)
        assert T_after == pytest.approx(T0 + (Th - T0) * (1.0 - dt / tau) ** k, rel=1e-12)
    one, _ = oracle.berendsen(hot, mass, n_dof, T0, 0.05, 0.05)
    assert 2.0 * oracle.kinetic_energy(one, mass) / (n_dof * oracle.K_B) == pytest.approx(T0, rel=1e-13)
    same, T_same = oracle.berendsen(v, mass, n_dof, T, tau, dt)
    assert np.array_equal(same, v) and T_same == T


def test_langevin_ou_pins():
    """Reading C-26: the exact Ornstein-Uhlenbeck velocity update.  Pins that do not re-type it: without
    noise the velocity decays by exactly e^(-gamma t) over any number of steps (the velocity autocorrelation of free
    Langevin dynamics); gamma = 0 leaves v unchanged and gamma -> infinity replaces it by a Maxwell-Boltzmann sample; the
    Maxwell-Boltzmann distribution is stationary (variance k_B T / m kept exactly in expectation, checked by sampling);
    from rest <v^2> relaxes as (k_B T / m)(1 - e^(-2 gamma t)); and <v(0) v(t)> over a sampled ensemble is e^(-gamma t)."""
    rng = np.random.default_rng(12)
    n = 200000
    mass = np.where(np.arange(n) % 3 == 0, 15.9994, 1.008)
    T, gamma, dt = 300.0, 5.0, 0.002
    kT_m = oracle.K_B * T / mass[:, None]
    v0 = rng.normal(size=(n, 3)) * np.sqrt(kT_m)
    zero = np.zeros((n, 3))
    v = v0.copy()
    for _ in range(25):
        v = oracle.langevin_ou(v, mass, zero, gamma, dt, T)
    assert np.allclose(v, v0 * math.exp(-gamma * 25 * dt), rtol=1e-13, atol=0)
    assert np.array_equal(oracle.langevin_ou(v0, mass, rng.normal(size=(n, 3)), 0.0, dt, T), v0)
    xi = rng.normal(size=(n, 3))
    assert np.allclose(oracle.langevin_ou(v0, mass, xi, 1e6, dt, T), np.sqrt(kT_m) * xi, rtol=1e-12, atol=1e-300)
    # stationarity and relaxation from rest, in units of k_B T / m (standard error of the variance estimate ~ sqrt(2/3n))
    v1 = oracle.langevin_ou(v0, mass, rng.normal(size=(n, 3)), gamma, dt, T)
    assert ((v1**2) / kT_m).mean() == pytest.approx(1.0, abs=6 * math.sqrt(2.0 / (3 * n)))
    v = zero.copy()
    for k in range(1, 41):
        v = oracle.langevin_ou(v, mass, rng.normal(size=(n, 3)), gamma, dt, T)
        if k in (5, 20, 40):
            assert ((v**2) / kT_m).mean() == pytest.approx(1.0 - math.exp(-2 * gamma * k * dt), abs=8 * math.sqrt(2.0 / (3 * n)))
    # velocity autocorrelation over the ensemble
    v = v0.copy()
    for k in range(1, 31):
        v = oracle.langevin_ou(v, mass, rng.normal(size=(n, 3)), gamma, dt, T)
        if k in (10, 30):
            c = ((v * v0) / kT_m).mean()
            assert c == pytest.approx(math.exp(-gamma * k * dt), abs=8 / math.sqrt(3 * n))


def test_count_pairs_equals_the_length_of_the_pair_list_and_a_kd_tree_count():
    """oracle.count_pairs (the count-only call that brackets the metric's numerator at the full-size configs) against
    (a) the length of the pair list both algorithms return and (b) scipy's periodic k-d tree minus the excluded pairs in
    range, on configs[1] (4 cells per axis), a single-cell box and a non-cubic box, with and without exclusions."""
    from scipy.spatial import cKDTree

    cases = [(wl.make_config(1), None, 1.0), (wl.make_config(1), None, 0.37), (small_box(m=40, edge=2.4, seed=4), None, 1.1),
             (small_box(m=60, edge=2.6, seed=9), np.array([2.6, 3.1, 2.9]), 1.2)]
    for wb, box, r in cases:
        box = wb.box if box is None else box
        pos = wb.pos.astype(np.float64)
        for excl in (wb.excl_pairs, None):
            n_list = len(oracle.neighbor_pairs(pos, box, r, excl, "celllist"))
            assert oracle.count_pairs(pos, box, r, excl) == n_list
            assert oracle.count_pairs(pos, box, r, excl, algorithm="bruteforce") == n_list
            if r <= 0.5 * box.min():  # scipy's periodic tree needs r < L/2
                pairs = cKDTree(pos % box, boxsize=box).query_pairs(r, output_type="ndarray")
                d = pos[pairs[:, 0]] - pos[pairs[:, 1]]
                d -= box * np.rint(d / box)
                inside = (d * d).sum(1) < r * r  # the tree's test is <=; the oracle's is strict (reading C-4)
                n_tree = int(inside.sum())
                if excl is not None:
                    i, j = excl[:, 0], excl[:, 1]
                    de = pos[i] - pos[j]
                    de -= box * np.rint(de / box)
                    n_tree -= int(((de * de).sum(1) < r * r).sum())
                assert n_list == n_tree, (r, n_list, n_tree)
