"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This package holds NO arithmetic of the GMNN method (no radial basis, no moments, no MLP):
only positions, species, masses, velocities and random weight tensors with the shapes and
distributions DESIGN.md section 4 states.  Neither `oracle/` nor `paper_2505_22168_b200/`
imports it; the tests and bench.py hand its arrays to both.
"""
from .inputs import (  # noqa: F401
    Workload,
    ModelSpec,
    make_model,
    make_workload,
    tiny_box,
    ionic_liquid_box,
    li3po4_box,
    cluster,
    triclinic_box,
    splitmix64,
    uniform01,
    normal01,
    KB_EV,
    ACC_CONV,
    FORCE_SCALE,
)
