"""CPU fp64 oracle for the reciprocal-space half of Ewald electrostatics.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): plain numpy, no blocking or reordering, shares no code with csrc/.

Two functions and one constant term:

* ewald_recip      -- the plain reciprocal sum, Eq. 11 with reading C-25: the printed formula lost the
                      charges and the imaginary unit; restored it reads
                          U_recip = k_e / (2 pi V) sum_{k != 0} exp(-(pi k / alpha)^2) / k^2 |S(k)|^2,
                          S(k) = sum_j q_j exp(2 pi i k . r_j),   k = (n_x / L_x, n_y / L_y, n_z / L_z),
                      which is 1/2 sum_{i,j} q_i q_j (...) exp(2 pi i k . r_ij) of the paper written with the structure
                      factor.  This is the DEFINITION the mesh method approximates.
* ewald_self       -- Eq. 12: U_self = -k_e alpha / sqrt(pi) sum_i q_i^2.
* pme_recip        -- smooth particle-mesh Ewald ("Following OpenMM, we implement smooth PME [15] ... B-splines
                      based on the recursive definition"), followed step by step in the notation of Essmann et al. 1995:
                      scaled fractional coordinates u = K r / L, cardinal B-spline weights M_n(u - k) by the recursion,
                      charge array Q, its discrete Fourier transform, the array B(m) C(m), the energy
                      1/2 sum_m B C |F(Q)|^2, the convolution theta_rec * Q and the forces -q_i sum_k grad(theta) (theta_rec * Q).

Virial (reading C-7, absent from the paper): W_ab = -dU/d(strain_ab); for both functions
    W_ab = sum_k u(k) [delta_ab - 2 (1 / k^2 + pi^2 / alpha^2) k_a k_b],  u(k) = the energy term of wave vector k,
so that tr W = -dU/dlambda under uniform scaling of positions and box at fixed alpha (pinned in tests/test_pme_oracle.py).

Pins (tests/test_pme_oracle.py): the NaCl Madelung constant through real + reciprocal + self, independence of the total
of alpha, forces = -finite-difference gradient, translation invariance, the virial's strain derivative, B-spline partition
of unity and the textbook M_2 / M_4 values, PME -> plain Ewald as the mesh is refined (the error bound of the method).
"""
from __future__ import annotations

import math

import numpy as np

COULOMB_CONST = 138.935456  # kJ mol^-1 nm e^-2 (reading C-2)


def ewald_self(charge, alpha, coulomb_const=COULOMB_CONST) -> float:
    """Eq. 12."""
    q = np.asarray(charge, dtype=np.float64)
    return float(-coulomb_const * alpha / math.sqrt(math.pi) * np.sum(q * q))


def ewald_recip(pos, charge, box, alpha, n_max, coulomb_const=COULOMB_CONST):
    """Plain reciprocal-space Ewald sum (Eq. 11, reading C-25) over all integer triples |n_a| <= n_max, n != 0.
    Returns (U, F (N,3), W (3,3)).  Cost O(N (2 n_max + 1)^3): small systems only."""
    r = np.asarray(pos, dtype=np.float64)
    q = np.asarray(charge, dtype=np.float64)
    L = np.asarray(box, dtype=np.float64)
    V = float(np.prod(L))
    n = np.arange(-n_max, n_max + 1)
    # e^{2 pi i n x / L} per axis: (N, 2 n_max + 1)
    ph = [np.exp(2j * np.pi * np.outer(r[:, a] / L[a], n)) for a in range(3)]
    U = 0.0
    F = np.zeros_like(r)
    W = np.zeros((3, 3))
    for ix, nx in enumerate(n):
        for iy, ny in enumerate(n):
            exy = ph[0][:, ix] * ph[1][:, iy]  # (N,)
            for iz, nz in enumerate(n):
                if nx == 0 and ny == 0 and nz == 0:
                    continue
                k = np.array([nx / L[0], ny / L[1], nz / L[2]])
                k2 = float(k @ k)
                a_k = math.exp(-(math.pi**2) * k2 / alpha**2) / k2
                e = exy * ph[2][:, iz]          # exp(2 pi i k . r_j)
                S = np.sum(q * e)
                u_k = coulomb_const / (2.0 * math.pi * V) * a_k * (S.real**2 + S.imag**2)
                U += u_k
                # F_j = -dU/dr_j = (2 k_e / V) q_j a(k) k Im(conj(S) e_j)
                F += (2.0 * coulomb_const / V) * a_k * np.outer(q * np.imag(np.conj(S) * e), k)
                W += u_k * (np.eye(3) - 2.0 * (1.0 / k2 + math.pi**2 / alpha**2) * np.outer(k, k))
    return U, F, W


def bspline(n: int, u):
    """Cardinal B-spline M_n(u) by the recursion of Essmann et al. (their Eq. 4.1):
    M_2(u) = 1 - |u - 1| on [0, 2], M_n(u) = u/(n-1) M_{n-1}(u) + (n-u)/(n-1) M_{n-1}(u-1)."""
    u = np.asarray(u, dtype=np.float64)
    if n == 2:
        return np.where((u >= 0.0) & (u <= 2.0), 1.0 - np.abs(u - 1.0), 0.0)
    return u / (n - 1) * bspline(n - 1, u) + (n - u) / (n - 1) * bspline(n - 1, u - 1.0)


def bspline_derivative(n: int, u):
    """dM_n/du = M_{n-1}(u) - M_{n-1}(u - 1) (Essmann Eq. 4.2)."""
    u = np.asarray(u, dtype=np.float64)
    return bspline(n - 1, u) - bspline(n - 1, u - 1.0)


def bspline_moduli(n: int, K: int):
    """|b(m)|^2, m = 0..K-1 (Essmann Eq. 4.4): b(m) = e^{2 pi i (n-1) m / K} / sum_{k=0}^{n-2} M_n(k+1) e^{2 pi i m k / K}.
    Where the sum vanishes (odd n, 2 m = K) the neighbours' average is used, as OpenMM does (reading C-25)."""
    k = np.arange(n - 1)
    mn = bspline(n, k + 1.0)
    m = np.arange(K)
    denom = np.abs(np.exp(2j * np.pi * np.outer(m, k) / K) @ mn) ** 2
    mod = np.empty(K)
    for i in range(K):
        d = denom[i]
        if d < 1e-7:
            d = 0.5 * (denom[(i - 1) % K] + denom[(i + 1) % K])
        mod[i] = 1.0 / d
    return mod


def pme_recip(pos, charge, box, alpha, mesh, order=5, coulomb_const=COULOMB_CONST):
    """Smooth PME reciprocal energy, forces and virial.  mesh = (K1, K2, K3), order = spline order n.
    Returns (U, F (N,3), W (3,3))."""
    r = np.asarray(pos, dtype=np.float64)
    q = np.asarray(charge, dtype=np.float64)
    L = np.asarray(box, dtype=np.float64)
    K = np.asarray(mesh, dtype=np.int64)
    N = r.shape[0]
    V = float(np.prod(L))
    n = int(order)
    # 1. scaled fractional coordinates u in [0, K), their integer part and the n spline weights / derivatives per axis
    frac = r / L
    frac -= np.floor(frac)
    u = frac * K
    fl = np.floor(u).astype(np.int64)
    fl = np.where(fl >= K, K - 1, fl)  # frac rounded to 1.0
    w = u - fl
    j = np.arange(n)
    theta = np.stack([bspline(n, w[:, a:a + 1] + j[None, :]) for a in range(3)], axis=1)              # (N, 3, n)
    dtheta = np.stack([bspline_derivative(n, w[:, a:a + 1] + j[None, :]) for a in range(3)], axis=1)  # (N, 3, n)
    idx = [(fl[:, a:a + 1] - j[None, :]) % K[a] for a in range(3)]                                    # (N, n) each
    # 2. charge array Q(k1, k2, k3) = sum_i q_i M_n(u1 - k1) M_n(u2 - k2) M_n(u3 - k3)
    Q = np.zeros(tuple(K))
    for i in range(N):
        Q[np.ix_(idx[0][i], idx[1][i], idx[2][i])] += q[i] * np.einsum("a,b,c->abc", theta[i, 0], theta[i, 1], theta[i, 2])
    # 3. B(m) C(m), m = (m1'/L1, m2'/L2, m3'/L3) with m' = m for m <= K/2, m - K otherwise
    mp = [np.where(np.arange(K[a]) <= K[a] // 2, np.arange(K[a]), np.arange(K[a]) - K[a]) / L[a] for a in range(3)]
    mx, my, mz = np.meshgrid(mp[0], mp[1], mp[2], indexing="ij")
    m2 = mx * mx + my * my + mz * mz
    m2[0, 0, 0] = 1.0
    C = coulomb_const / (math.pi * V) * np.exp(-(math.pi**2) * m2 / alpha**2) / m2
    C[0, 0, 0] = 0.0
    B = np.einsum("a,b,c->abc", bspline_moduli(n, int(K[0])), bspline_moduli(n, int(K[1])), bspline_moduli(n, int(K[2])))
    BC = B * C
    # 4. energy 1/2 sum_m B C |F(Q)(m)|^2 and the virial from the same terms
    Qh = np.fft.fftn(Q)
    e_m = 0.5 * BC * (Qh.real**2 + Qh.imag**2)
    U = float(e_m.sum())
    fac = 2.0 * (1.0 / m2 + math.pi**2 / alpha**2)
    W = np.zeros((3, 3))
    mv = (mx, my, mz)
    for a in range(3):
        for b in range(3):
            W[a, b] = float(np.sum(e_m * ((1.0 if a == b else 0.0) - fac * mv[a] * mv[b])))
    # 5. convolution (theta_rec * Q)(k) = sum_m B C F(Q)(m) e^{+2 pi i m.k/K} and the forces
    phi = np.fft.ifftn(BC * Qh).real * float(np.prod(K))
    F = np.zeros_like(r)
    for i in range(N):
        p = phi[np.ix_(idx[0][i], idx[1][i], idx[2][i])]
        t0, t1, t2 = theta[i]
        d0, d1, d2 = dtheta[i]
        F[i, 0] = -q[i] * K[0] / L[0] * np.einsum("a,b,c,abc->", d0, t1, t2, p)
        F[i, 1] = -q[i] * K[1] / L[1] * np.einsum("a,b,c,abc->", t0, d1, t2, p)
        F[i, 2] = -q[i] * K[2] / L[2] * np.einsum("a,b,c,abc->", t0, t1, d2, p)
    return U, F, W


def pme_mesh_size(alpha, box, delta):
    """The paper's heuristic: n_mesh = 2 alpha d / (3 delta^(1/5)) per box edge d, rounded up."""
    return tuple(int(math.ceil(2.0 * alpha * float(d) / (3.0 * delta**0.2))) for d in box)
