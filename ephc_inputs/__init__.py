"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package only *draws inputs* (grids, band energies, phonon energies,
|g|^2 blocks, candidate (k,k+q) pairs, occupations, velocities).  It holds none
of the collision-integral arithmetic: no delta functions, no channel selection,
no k+q index arithmetic, no occupation factors.  Both `oracle/` and
`paper_2511_03683_b200/` receive the same arrays from here and implement the
method independently.
"""
from .configs import (  # noqa: F401
    KB_EV_PER_K,
    Problem,
    CONFIG_NAMES,
    make_problem,
    fermi_dirac,
    bose_einstein,
)
