"""CPU fp64 oracle for the DIMOS neighbour-list + nonbonded hot path.

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this.
"""
from .dimos_oracle import (  # noqa: F401
    METHOD_EWALD_REAL,
    METHOD_RF,
    NonbondedResult,
    count_pairs,
    edge_vectors,
    lorentz_berthelot,
    needs_rebuild,
    neighbor_pairs,
    nonbonded,
    num_threads,
)
from .vv_oracle import K_B, berendsen, langevin_ou, dispersion_correction, kinetic_energy, rattle_water_velocities, shake_water, vv_kick, vv_kick_drift  # noqa: F401,E402
