"""Seeded synthetic water-box inputs (BASELINE.json `configs[0..4]`, SURVEY.md §8(d) recipe).

This module is the ONLY code shared between the CPU oracle's tests and the CUDA path's
tests/bench.  It draws random numbers and lays out rigid 3-site water molecules; it holds none
of the method's arithmetic (no distances, no potentials, no neighbour search).

The paper's workload is a constant-density TIP3P water box (Fig. 1 caption,
PAPER.md:41 §I A); its coordinate files are not available, so these boxes take its shape
(density 33.4 molecules/nm^3, rigid 3-site geometry, charges, LJ on O only) and stand in for it.

Units: nm, ps, amu, e, kJ/mol.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SEED_BASE = 250320541  # arXiv id 2503.20541 -> seed; + config index

# TIP3P-geometry water (BASELINE.json configs[0])
Q_O = -0.834
Q_H = +0.417
R_OH = 0.09572  # nm
ANGLE_HOH_DEG = 104.52
SIGMA_O = 0.315061  # nm
EPS_O = 0.6364  # kJ/mol
MASS_O = 15.9994
MASS_H = 1.008
DENSITY = 33.4  # molecules / nm^3
COULOMB_CONST = 138.935456  # kJ mol^-1 nm e^-2
K_BOLTZ = 0.0083144626  # kJ mol^-1 K^-1


@dataclasses.dataclass(frozen=True)
class ConfigSpec:
    index: int
    name: str
    n_molecules: int
    box_edge: float | None  # None -> from density
    r_cut: float
    skin: float
    method: str  # "rf" | "ewald"
    eps_rf: float = 78.5
    alpha: float = 3.12
    precisions: tuple = ("f32",)


CONFIGS = (
    ConfigSpec(0, "water216", 216, 1.8621, 0.9, 0.1, "rf", precisions=("f64", "f32")),
    ConfigSpec(1, "water3k", 3000, None, 1.0, 0.1, "rf", precisions=("f32",)),
    ConfigSpec(2, "water30k", 30000, None, 1.0, 0.1, "rf", precisions=("f32", "mixed")),
    ConfigSpec(3, "water300k", 300000, None, 1.0, 0.1, "rf", precisions=("f32",)),
    ConfigSpec(4, "water100k_ewald", 100000, None, 1.0, 0.1, "ewald", precisions=("f32", "f64")),
)


@dataclasses.dataclass
class WaterBox:
    """One synthetic periodic water box.  All arrays are host numpy arrays."""

    spec: ConfigSpec
    box: np.ndarray  # (3,) float64, each value exactly fp32-representable
    pos: np.ndarray  # (N,3) float32, wrapped into [0,L)
    charge: np.ndarray  # (N,) float32
    type: np.ndarray  # (N,) int32, 0 = O, 1 = H
    sigma: np.ndarray  # (ntypes,) float64 per-type sigma_i
    epsilon: np.ndarray  # (ntypes,) float64 per-type epsilon_i
    excl_pairs: np.ndarray  # (n_excl,2) int32, i<j, unique, lexicographically sorted
    mass: np.ndarray  # (N,) float64

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])


def box_edge_for(spec: ConfigSpec) -> float:
    """Cubic box edge, rounded to fp32 so both sides hold the identical number."""
    if spec.box_edge is not None:
        edge = spec.box_edge
    else:
        edge = (spec.n_molecules / DENSITY) ** (1.0 / 3.0)
    return float(np.float32(edge))


def _body_frame() -> np.ndarray:
    half = math.radians(ANGLE_HOH_DEG) / 2.0
    s, c = math.sin(half), math.cos(half)
    return np.array(
        [[0.0, 0.0, 0.0], [+R_OH * s, 0.0, R_OH * c], [-R_OH * s, 0.0, R_OH * c]],
        dtype=np.float64,
    )


def _quat_to_matrix(q: np.ndarray) -> np.ndarray:
    """(M,4) unit quaternions (w,x,y,z) -> (M,3,3) rotation matrices."""
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    rot = np.empty((q.shape[0], 3, 3), dtype=np.float64)
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z)
    rot[:, 0, 1] = 2 * (x * y - z * w)
    rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w)
    rot[:, 1, 1] = 1 - 2 * (x * x + z * z)
    rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w)
    rot[:, 2, 1] = 2 * (y * z + x * w)
    rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return rot


def make_water_box(n_molecules: int, edge: float, seed: int, spec: ConfigSpec | None = None) -> WaterBox:
    """Lattice-with-jitter water box (readings C-19/C-20)."""
    rng = np.random.default_rng(seed)
    edge = float(np.float32(edge))
    m = int(n_molecules)
    n_side = int(math.ceil(round(m ** (1.0 / 3.0), 9)))
    while n_side**3 < m:
        n_side += 1
    a = edge / n_side
    # occupy m of n^3 sites chosen by a seeded permutation, kept in ascending site order
    sites = np.sort(rng.permutation(n_side**3)[:m])
    kx = sites // (n_side * n_side)
    ky = (sites // n_side) % n_side
    kz = sites % n_side
    centre = (np.stack([kx, ky, kz], axis=1).astype(np.float64) + 0.5) * a
    centre += rng.uniform(-0.02, 0.02, size=(m, 3))
    quat = rng.standard_normal(size=(m, 4))
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    rot = _quat_to_matrix(quat)
    body = _body_frame()  # (3 sites, 3)
    # centre = oxygen position (C-19); rotate body frame about it
    pos = centre[:, None, :] + np.einsum("mab,sb->msa", rot, body)
    pos = pos.reshape(3 * m, 3)
    pos = pos - edge * np.floor(pos / edge)
    pos32 = pos.astype(np.float32)
    edge32 = np.float32(edge)
    pos32 = np.where(pos32 >= edge32, pos32 - edge32, pos32).astype(np.float32)
    pos32 = np.where(pos32 < 0, np.float32(0.0), pos32).astype(np.float32)

    charge = np.tile(np.array([Q_O, Q_H, Q_H], dtype=np.float32), m)
    typ = np.tile(np.array([0, 1, 1], dtype=np.int32), m)
    mass = np.tile(np.array([MASS_O, MASS_H, MASS_H], dtype=np.float64), m)
    base = 3 * np.arange(m, dtype=np.int32)
    excl = np.stack(
        [
            np.stack([base, base + 1], axis=1),
            np.stack([base, base + 2], axis=1),
            np.stack([base + 1, base + 2], axis=1),
        ],
        axis=1,
    ).reshape(3 * m, 2)
    if spec is None:
        spec = ConfigSpec(-1, f"custom{m}", m, edge, 1.0, 0.1, "rf")
    return WaterBox(
        spec=spec,
        box=np.array([edge, edge, edge], dtype=np.float64),
        pos=np.ascontiguousarray(pos32),
        charge=charge,
        type=typ,
        sigma=np.array([SIGMA_O, 0.0], dtype=np.float64),
        epsilon=np.array([EPS_O, 0.0], dtype=np.float64),
        excl_pairs=np.ascontiguousarray(excl.astype(np.int32)),
        mass=mass,
    )


def make_config(index: int) -> WaterBox:
    spec = CONFIGS[index]
    return make_water_box(spec.n_molecules, box_edge_for(spec), SEED_BASE + index, spec)


def make_scaled(n_molecules: int, seed: int = SEED_BASE + 100, r_cut: float = 1.0, skin: float = 0.1,
                method: str = "rf") -> WaterBox:
    """A constant-density box of arbitrary size (tau(N) sweep, test sizes)."""
    edge = float(np.float32((n_molecules / DENSITY) ** (1.0 / 3.0)))
    spec = ConfigSpec(-1, f"water{n_molecules}", n_molecules, edge, r_cut, skin, method)
    return make_water_box(n_molecules, edge, seed, spec)


def maxwell_boltzmann_velocities(mass: np.ndarray, temperature: float, seed: int) -> np.ndarray:
    """(N,3) float64 velocities in nm/ps, centre-of-mass velocity removed."""
    rng = np.random.default_rng(seed)
    sigma_v = np.sqrt(K_BOLTZ * temperature / mass)
    vel = rng.standard_normal(size=(mass.shape[0], 3)) * sigma_v[:, None]
    vcom = (vel * mass[:, None]).sum(axis=0) / mass.sum()
    return vel - vcom
