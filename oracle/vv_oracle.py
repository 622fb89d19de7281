"""The velocity-Verlet loop of PAPER.md:281-292 (section III C 1) written out in numpy fp64: steps 1, 2, 5 (kicks and
drift), steps 3 and 6 for rigid three-site water (SHAKE / RATTLE iterated to convergence, reading C-23), step 7 as the
Berendsen thermostat (reading C-24) and the Langevin update of PAPER.md:309 (reading C-26), plus the long-range dispersion
correction of PAPER.md:202 (reading C-22).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): the product package never imports this.

Units: positions nm, velocities nm/ps, forces kJ mol^-1 nm^-1, masses amu, time ps.  With these units the
acceleration a = F / m is in nm/ps^2 without any conversion factor (1 kJ/mol = 1 amu nm^2 ps^-2).
"""
from __future__ import annotations

import numpy as np


def vv_kick_drift(pos, vel, force, inv_mass, dt):
    """Steps 1 and 2: v(t + dt/2) = v(t) + a(t) dt / 2;  x(t + dt) = x(t) + v(t + dt/2) dt.
    Returns (pos_new, vel_half) as float64 arrays; inputs are promoted to float64."""
    pos = np.asarray(pos, dtype=np.float64)
    vel = np.asarray(vel, dtype=np.float64)
    force = np.asarray(force, dtype=np.float64)
    inv_mass = np.asarray(inv_mass, dtype=np.float64).reshape(-1, 1)
    vel_half = vel + 0.5 * dt * (force * inv_mass)
    pos_new = pos + dt * vel_half
    return pos_new, vel_half


def vv_kick(vel_half, force_new, inv_mass, dt):
    """Step 5: v(t + dt) = v(t + dt/2) + a(t + dt) dt / 2."""
    vel_half = np.asarray(vel_half, dtype=np.float64)
    force_new = np.asarray(force_new, dtype=np.float64)
    inv_mass = np.asarray(inv_mass, dtype=np.float64).reshape(-1, 1)
    return vel_half + 0.5 * dt * (force_new * inv_mass)


def dispersion_correction(type_, lj_table, box, r_cut, r_switch=0.0):
    """Long-range dispersion (LJ tail) correction, PAPER.md:202 ("long-range dispersion corrections that approximate the
    contributions beyond r_c"; no formula given: reading C-22).  Homogeneous fluid beyond the truncation, g(r) = 1:

        E = (2 pi / V) sum_a sum_b N_a N_b  integral_0^inf [1 - S(r)] U_ab(r) r^2 dr

    with U_ab the 12-6 potential of Eq. 4, S(r) = 1 for r < r_s, Eq. 6 for r_s <= r < r_c, 0 beyond r_c (r_switch <= 0 or
    >= r_cut: S = 1 below r_c).  Evaluated by adaptive quadrature of exactly this integrand (scipy QUADPACK).
    Returns (E, W) with W the 3x3 virial in the convention of reading C-7 (tr W = -dE/d lambda at fixed r_c): E scales as
    1/V, so W = E * identity."""
    from scipy import integrate

    type_ = np.asarray(type_, dtype=np.int64)
    lj_table = np.asarray(lj_table, dtype=np.float64)
    nt = lj_table.shape[0]
    counts = np.bincount(type_, minlength=nt).astype(np.float64)
    vol = float(np.prod(np.asarray(box, dtype=np.float64)))
    switched = 0.0 < r_switch < r_cut

    def one_minus_s(r):
        if r >= r_cut:
            return 1.0
        if not switched or r < r_switch:
            return 0.0
        x = (r - r_switch) / (r_cut - r_switch)
        return 1.0 - (1.0 - 6.0 * x ** 5 + 15.0 * x ** 4 - 10.0 * x ** 3)

    total = 0.0
    for a in range(nt):
        for b in range(nt):
            sigma, eps = lj_table[a, b]
            if eps == 0.0 or sigma == 0.0 or counts[a] == 0 or counts[b] == 0:
                continue

            def integrand(r, sigma=sigma, eps=eps):
                sr6 = (sigma / r) ** 6
                return one_minus_s(r) * 4.0 * eps * (sr6 * sr6 - sr6) * r * r

            lo = r_switch if switched else r_cut
            inner = integrate.quad(integrand, lo, r_cut, epsabs=0, epsrel=1e-13)[0] if switched else 0.0
            outer = integrate.quad(integrand, r_cut, np.inf, epsabs=0, epsrel=1e-13)[0]
            total += counts[a] * counts[b] * (inner + outer)
    e = 2.0 * np.pi / vol * total
    return e, e * np.eye(3)


def shake_water(pos_old, pos_new, mass, d_oh, d_hh, tol=1e-14, max_iter=200000):
    """Position constraints of rigid three-site water (step 3 of PAPER.md:281-292; PAPER.md:327 names SETTLE for it), as
    the plain iterative SHAKE procedure run to convergence: for every molecule (atoms 3k, 3k+1, 3k+2 = O, H, H) the new
    positions are corrected along the OLD bond vectors, x_i += g m_i^-1 r_ij_old, x_j -= g m_j^-1 r_ij_old with
    g = (d_ij^2 - |r_ij_new|^2) / (2 (1/m_i + 1/m_j) r_ij_new . r_ij_old), until |r_ij| = d_ij for the three bonds.
    SETTLE solves the same equations in closed form, so a converged SHAKE is its oracle.  Returns the constrained
    positions (fp64); pos_old must satisfy the constraints.  The sweeps converge in ~30 iterations for water's shape and in
    thousands for a nearly linear molecule (the three bond vectors are then almost dependent); a run that has not reached
    `tol` after max_iter sweeps raises instead of returning an unconverged answer."""
    x0 = np.asarray(pos_old, dtype=np.float64).reshape(-1, 3, 3)
    x = np.array(pos_new, dtype=np.float64).reshape(-1, 3, 3)
    im = 1.0 / np.asarray(mass, dtype=np.float64).reshape(-1, 3)
    bonds = ((0, 1, d_oh), (0, 2, d_oh), (1, 2, d_hh))
    best, stalled = np.inf, 0
    for _ in range(max_iter):
        worst = 0.0
        for i, j, d in bonds:
            r_old = x0[:, i] - x0[:, j]
            r_new = x[:, i] - x[:, j]
            diff = d * d - (r_new * r_new).sum(1)
            worst = max(worst, float(np.abs(diff).max()) / (d * d))
            g = diff / (2.0 * (im[:, i] + im[:, j]) * (r_new * r_old).sum(1))
            x[:, i] += (g * im[:, i])[:, None] * r_old
            x[:, j] -= (g * im[:, j])[:, None] * r_old
        # converged: the residual is below tol, or it sits on its rounding floor (no 1 % improvement in 100 sweeps, below
        # 1e-11: an ill-conditioned shape amplifies the rounding of the coordinates past tol)
        if worst < 0.99 * best:
            best, stalled = worst, 0
        else:
            stalled += 1
        if worst < tol or (stalled >= 100 and best < 1e-11):
            break
    else:
        raise RuntimeError(f"shake_water: not converged after {max_iter} sweeps (worst relative residual {worst:.3e})")
    return x.reshape(-1, 3)


def rattle_water_velocities(pos, vel, mass, tol=1e-15, max_iter=200000):
    """Velocity constraints of rigid three-site water (step 6 of PAPER.md:281-292), as the plain iterative RATTLE velocity
    stage run to convergence: for every bond (i, j) of a molecule (atoms 3k, 3k+1, 3k+2) the component of the relative
    velocity along the bond is removed by an impulse along r_ij shared by inverse mass,
    k = (v_ij . r_ij) / (|r_ij|^2 (1/m_i + 1/m_j)),  v_i -= k r_ij / m_i,  v_j += k r_ij / m_j, until v_ij . r_ij = 0 for the
    three bonds.  Returns the constrained velocities (fp64)."""
    x = np.asarray(pos, dtype=np.float64).reshape(-1, 3, 3)
    v = np.array(vel, dtype=np.float64).reshape(-1, 3, 3)
    im = 1.0 / np.asarray(mass, dtype=np.float64).reshape(-1, 3)
    scale = max(float(np.abs(v).max()), 1e-300)
    for _ in range(max_iter):
        worst = 0.0
        for i, j in ((0, 1), (0, 2), (1, 2)):
            r = x[:, i] - x[:, j]
            rv = ((v[:, i] - v[:, j]) * r).sum(1)
            r2 = (r * r).sum(1)
            worst = max(worst, float((np.abs(rv) / np.sqrt(r2)).max()) / scale)
            k = rv / (r2 * (im[:, i] + im[:, j]))
            v[:, i] -= (k * im[:, i])[:, None] * r
            v[:, j] += (k * im[:, j])[:, None] * r
        if worst < tol:
            break
    else:
        raise RuntimeError(f"rattle_water_velocities: not converged after {max_iter} sweeps (worst residual {worst:.3e} of max|v|)")
    return v.reshape(-1, 3)


K_B = 8.314462618e-3  # kJ mol^-1 K^-1 (molar gas constant, CODATA 2018): the units of PAPER.md's MD (nm, ps, amu)


def kinetic_energy(vel, mass):
    """K = 1/2 sum_i m_i |v_i|^2 in kJ/mol (amu nm^2 ps^-2 = kJ/mol), fp64."""
    v = np.asarray(vel, dtype=np.float64)
    return 0.5 * float((np.asarray(mass, dtype=np.float64)[:, None] * v * v).sum())


def berendsen(vel, mass, n_dof, T0, tau, dt):
    """Step 7 of PAPER.md:281-292 with the Berendsen thermostat (a thermostat that rescales the velocities):
    T = 2 K / (n_dof k_B); every velocity is multiplied by lambda = sqrt(1 + (dt / tau) (T0 / T - 1)).
    Returns (scaled velocities fp64, T before scaling)."""
    T = 2.0 * kinetic_energy(vel, mass) / (n_dof * K_B)
    lam = np.sqrt(1.0 + (dt / tau) * (T0 / T - 1.0))
    return np.asarray(vel, dtype=np.float64) * lam, T


def langevin_ou(vel, mass, xi, gamma, dt, T):
    """Langevin dynamics (PAPER.md:309 names it and gives no formula: reading C-26): the friction + noise part of the
    Langevin equation dv = -gamma v dt + sqrt(2 gamma k_B T / m) dW integrated EXACTLY over one time step (the
    Ornstein-Uhlenbeck update, applied where velocity Verlet has its step 7):
        v <- a v + sqrt((1 - a^2) k_B T / m) xi,   a = exp(-gamma dt),
    xi = one standard normal number per velocity component, passed in (both sides of the parity test read the same
    array).  gamma in ps^-1, T in K, masses in amu, velocities in nm/ps.  Returns fp64 velocities."""
    v = np.asarray(vel, dtype=np.float64)
    m = np.asarray(mass, dtype=np.float64)[:, None]
    x = np.asarray(xi, dtype=np.float64)
    a = np.exp(-gamma * dt)
    return a * v + np.sqrt((1.0 - a * a) * K_B * T / m) * x
