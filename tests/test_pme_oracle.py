"""Pins for oracle/pme_oracle.py (reciprocal-space Ewald, Eq. 11-12, and smooth PME).  Each test checks
the oracle against something fixed outside it: the Madelung constant of rock salt, the independence of the Ewald total of
alpha ("for any choice of alpha above formulas are correct"), finite differences, invariances, textbook
B-spline values, and the convergence of the mesh method to the plain sum."""
import math

import numpy as np
import pytest

import oracle
from oracle import pme_oracle as pme

KE = pme.COULOMB_CONST
MADELUNG_NACL = 1.747564594633182  # rock salt, referred to the nearest-neighbour distance (textbook constant)


def rock_salt(cells: int, a: float = 1.0):
    """cells^3 conventional cells of edge a: ions on a simple cubic lattice of spacing a/2 with alternating charge."""
    n = 2 * cells
    g = np.arange(n)
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    pos = np.stack([x, y, z], axis=-1).reshape(-1, 3) * (a / 2)
    q = np.where((x + y + z).reshape(-1) % 2 == 0, 1.0, -1.0)
    return pos.astype(np.float64), q, np.full(3, cells * a)


def real_space(pos, q, box, alpha, r_cut):
    """Real-space Ewald energy and forces from the pinned pair oracle (dimos_oracle.c, Eq. 10, nearest image)."""
    n = len(q)
    lj = np.zeros((1, 1, 2))
    res = oracle.nonbonded(pos, q, np.zeros(n, np.int32), lj, box, r_cut, method=oracle.METHOD_EWALD_REAL, alpha=alpha,
                           algorithm="bruteforce")
    return res.E[0], res.F, res.W


def random_neutral(n_pairs, edge, seed):
    rng = np.random.default_rng(seed)
    pos = rng.uniform(0, edge, size=(2 * n_pairs, 3))
    q = np.concatenate([rng.uniform(0.3, 1.0, n_pairs), np.zeros(n_pairs)])
    q[n_pairs:] = -q[:n_pairs][rng.permutation(n_pairs)]
    return pos, q, np.array([edge, edge * 1.1, edge * 0.9])


def test_madelung_constant_of_rock_salt():
    """E_total = real + reciprocal + self = -(N/2) M k_e q^2 / r0 for NaCl: pins Eq. 11 (with the charges restored),
    Eq. 12, their prefactors and signs, and the real-space term's erfc together."""
    pos, q, box = rock_salt(2)  # 64 ions, L = 2, nearest-neighbour distance 0.5
    # move every ion off the exact lattice-symmetric cutoff shell: r_cut = L/2 = 1.0 coincides with lattice distances,
    # so use a slightly smaller cutoff; alpha large enough that erfc(alpha r_cut) ~ 1e-15
    alpha, r_cut = 6.2, 0.97
    e_real, _, _ = real_space(pos, q, box, alpha, r_cut)
    e_rec, _, _ = pme.ewald_recip(pos, q, box, alpha, n_max=16)
    e_self = pme.ewald_self(q, alpha)
    want = -0.5 * len(q) * MADELUNG_NACL * KE / 0.5
    assert e_real + e_rec + e_self == pytest.approx(want, rel=1e-9)


def test_ewald_total_is_independent_of_alpha():
    pos, q, box = random_neutral(20, 2.4, 3)
    r_cut = 0.5 * box.min() - 1e-9
    totals, forces = [], []
    for alpha in (5.2, 6.0, 7.0):
        e_real, f_real, _ = real_space(pos, q, box, alpha, r_cut)
        e_rec, f_rec, _ = pme.ewald_recip(pos, q, box, alpha, n_max=int(math.ceil(alpha * box.max() * 2.0)))
        totals.append(e_real + e_rec + pme.ewald_self(q, alpha))
        forces.append(f_real + f_rec)
    assert totals[1] == pytest.approx(totals[0], rel=1e-9) and totals[2] == pytest.approx(totals[0], rel=1e-9)
    scale = np.abs(forces[0]).max()
    assert np.abs(forces[1] - forces[0]).max() < 1e-8 * scale and np.abs(forces[2] - forces[0]).max() < 1e-8 * scale


def test_self_energy_closed_form():
    assert pme.ewald_self([1.0, -2.0, 0.5], 3.0, coulomb_const=2.0) == pytest.approx(-2.0 * 3.0 / math.sqrt(math.pi) * 5.25)


@pytest.mark.parametrize("which", ["ewald", "pme"])
def test_reciprocal_forces_are_minus_gradient_and_sum_to_zero(which):
    pos, q, box = random_neutral(6, 1.9, 11)
    alpha = 3.0
    if which == "ewald":
        fn = lambda p: pme.ewald_recip(p, q, box, alpha, n_max=6)
    else:
        fn = lambda p: pme.pme_recip(p, q, box, alpha, (16, 18, 15), order=5)
    U, F, W = fn(pos)
    h = 1e-5
    rng = np.random.default_rng(0)
    for i, a in zip(rng.integers(0, len(q), 6), rng.integers(0, 3, 6)):
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h
        pm[i, a] -= h
        fd = -(fn(pp)[0] - fn(pm)[0]) / (2 * h)
        assert F[i, a] == pytest.approx(fd, rel=2e-6, abs=1e-6 * np.abs(F).max())
    if which == "ewald":  # exact translation invariance => momentum conservation; the mesh breaks it at the level of its error
        assert np.abs(F.sum(axis=0)).max() < 1e-10 * np.abs(F).max()
    assert np.allclose(W, W.T, rtol=0, atol=1e-12 * np.abs(W).max())


@pytest.mark.parametrize("which", ["ewald", "pme"])
def test_reciprocal_virial_is_minus_strain_derivative(which):
    """tr W = -dU/dlambda under uniform scaling of positions and box at fixed alpha (reading C-7's convention), and the
    xy component from a simple shear-free anisotropic stretch of one axis."""
    pos, q, box = random_neutral(8, 2.0, 5)
    alpha = 2.8

    def energy(scale):
        s = np.asarray(scale, dtype=np.float64)
        if which == "ewald":
            return pme.ewald_recip(pos * s, q, box * s, alpha, n_max=6)[0]
        return pme.pme_recip(pos * s, q, box * s, alpha, (20, 20, 20), order=5)[0]

    W = (pme.ewald_recip(pos, q, box, alpha, n_max=6) if which == "ewald" else pme.pme_recip(pos, q, box, alpha, (20, 20, 20), 5))[2]
    h = 1e-5
    dU = (energy([1 + h] * 3) - energy([1 - h] * 3)) / (2 * h)
    assert np.trace(W) == pytest.approx(-dU, rel=1e-6)
    for a in range(3):  # stretching one axis only gives the diagonal component
        sp, sm = np.ones(3), np.ones(3)
        sp[a] += h
        sm[a] -= h
        assert W[a, a] == pytest.approx(-(energy(sp) - energy(sm)) / (2 * h), rel=1e-5, abs=1e-7 * abs(np.trace(W)))


def test_translation_and_image_invariance_of_the_plain_sum():
    pos, q, box = random_neutral(10, 2.2, 8)
    U0, F0, _ = pme.ewald_recip(pos, q, box, 3.1, n_max=5)
    shifted = pos + np.array([0.37, -5.1, 12.0])
    shifted[3] += box * np.array([1, -2, 0])
    U1, F1, _ = pme.ewald_recip(shifted, q, box, 3.1, n_max=5)
    assert U1 == pytest.approx(U0, rel=1e-12)
    assert np.abs(F1 - F0).max() < 1e-10 * np.abs(F0).max()


def test_bspline_textbook_values_and_partition_of_unity():
    # M_2 is the hat function; M_4 is the cubic B-spline with knots 0..4: M_4(1) = 1/6, M_4(2) = 2/3, M_4(3) = 1/6
    assert pme.bspline(2, [0.0, 0.5, 1.0, 1.5, 2.0]).tolist() == [0.0, 0.5, 1.0, 0.5, 0.0]
    assert pme.bspline(4, [1.0, 2.0, 3.0]) == pytest.approx([1 / 6, 2 / 3, 1 / 6], rel=1e-15)
    assert pme.bspline(4, [0.5]) == pytest.approx([0.5**3 / 6], rel=1e-15)
    # M_5 at the integers: 1/24, 11/24, 11/24, 1/24 (quartic B-spline)
    assert pme.bspline(5, [1.0, 2.0, 3.0, 4.0]) == pytest.approx([1 / 24, 11 / 24, 11 / 24, 1 / 24], rel=1e-15)
    w = np.linspace(0.0, 0.999, 7)
    for n in (3, 4, 5, 6):
        j = np.arange(n)
        assert np.allclose(pme.bspline(n, w[:, None] + j[None, :]).sum(axis=1), 1.0, atol=1e-14)        # sum_k M_n(u - k) = 1
        assert np.allclose(pme.bspline_derivative(n, w[:, None] + j[None, :]).sum(axis=1), 0.0, atol=1e-14)
        h = 1e-6
        fd = (pme.bspline(n, 1.3 + h) - pme.bspline(n, 1.3 - h)) / (2 * h)
        assert pme.bspline_derivative(n, 1.3) == pytest.approx(fd, rel=1e-8)


def test_pme_converges_to_the_plain_reciprocal_sum():
    """Smooth PME approximates Eq. 11; its error falls with the mesh spacing like h^n (order n = 5) -- the error bound of
    the method -- and at the paper's heuristic mesh it is of the size of the tolerance delta."""
    pos, q, box = random_neutral(15, 2.0, 21)
    alpha = 3.12
    U0, F0, W0 = pme.ewald_recip(pos, q, box, alpha, n_max=10)
    rms = np.sqrt((F0**2).sum(axis=1).mean())
    errs = []
    for K in (12, 24, 48):
        U, F, W = pme.pme_recip(pos, q, box, alpha, (K, K, K), order=5)
        errs.append(np.sqrt(((F - F0) ** 2).sum(axis=1).mean()) / rms)
    assert errs[0] > errs[1] > errs[2]
    assert errs[1] / errs[2] > 12.0  # ~ 2^5 = 32 asymptotically, at least 2^3.6 here
    assert errs[2] < 2e-5
    U, F, W = pme.pme_recip(pos, q, box, alpha, (48, 48, 48), order=5)
    assert U == pytest.approx(U0, rel=1e-5)
    assert np.abs(W - W0).max() < 1e-4 * np.abs(W0).max()
    delta = 2.96e-5  # alpha = 3.12 <-> Eq. 13 at r_c = 1 nm (reading C-13)
    mesh = pme.pme_mesh_size(alpha, box, delta)
    assert mesh == tuple(int(math.ceil(2 * alpha * d / (3 * delta**0.2))) for d in box)
    U, F, W = pme.pme_recip(pos, q, box, alpha, mesh, order=5)
    assert np.sqrt(((F - F0) ** 2).sum(axis=1).mean()) / rms < 5e-4


def test_pme_madelung_constant_through_the_mesh():
    pos, q, box = rock_salt(2)
    rng = np.random.default_rng(1)
    pos = pos + 0.013  # off the mesh nodes, still a perfect crystal
    alpha, r_cut = 6.2, 0.97
    e_real, _, _ = real_space(pos, q, box, alpha, r_cut)
    e_rec, F, _ = pme.pme_recip(pos, q, box, alpha, (64, 64, 64), order=6)
    want = -0.5 * len(q) * MADELUNG_NACL * KE / 0.5
    assert e_real + e_rec + pme.ewald_self(q, alpha) == pytest.approx(want, rel=2e-6)
    assert np.abs(F).max() < 1e-3 * abs(want)  # forces vanish by symmetry up to the mesh error


def test_bspline_moduli_special_values():
    """|b(m)|^2 (Essmann Eq. 4.4): 1 at m = 0 for every order (the weights M_n(k + 1) sum to one); identically 1 for order 2
    (M_2(1) = 1 is the only weight); symmetric under m -> K - m (complex conjugation); never below 1 (|sum w e^{i..}| <= sum w
    = 1 for non-negative weights); for order 4 at m = K/2 the closed value 1 / (M_4(1) - M_4(2) + M_4(3))^2 = 1 / (1/3)^2 = 9;
    and for an odd order the vanishing denominator at 2 m = K is replaced by the neighbours' average (reading C-25)."""
    for n in (2, 3, 4, 5, 6):
        for K in (16, 21, 30):
            mod = pme.bspline_moduli(n, K)
            assert mod[0] == pytest.approx(1.0, rel=1e-14)
            assert np.allclose(mod[1:], mod[1:][::-1], rtol=1e-12)
            assert np.all(mod >= 1.0 - 1e-12)
            if n == 2:
                assert np.allclose(mod, 1.0, rtol=1e-14)
    assert pme.bspline_moduli(4, 16)[8] == pytest.approx(9.0, rel=1e-12)
    mod = pme.bspline_moduli(5, 16)  # odd order, even mesh: sum_k M_5(k + 1) (-1)^k = 1/24 - 11/24 + 11/24 - 1/24 = 0
    den = 1.0 / mod
    assert den[8] == pytest.approx(0.5 * (den[7] + den[9]), rel=1e-12)
