"""Velocity-Verlet steps 1, 2 and 5 of PAPER.md:281-292 (section III C 1), written out in numpy fp64.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): the product package never imports this.

Units: positions nm, velocities nm/ps, forces kJ mol^-1 nm^-1, masses amu, time ps.  With these units the
acceleration a = F / m is in nm/ps^2 without any conversion factor (1 kJ/mol = 1 amu nm^2 ps^-2).
Constraints (steps 3, 6) and the thermostat (step 7) are not part of this oracle: the library does not build them.
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
