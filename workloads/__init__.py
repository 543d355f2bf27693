"""Seeded synthetic inputs (scenes, efficiency tables, photons) for the oracle, the
CUDA path, the tests and bench.py.

This package holds *none* of the method's arithmetic (no ray/triangle test, no
Philox, no table lookup, no pixel map): it only produces the arrays both sides
consume.  It imports neither ``oracle`` nor ``paper_2309_12496_b200``.

The recipes are the synthetic stand-ins for the paper's own inputs (Geant4 photon
files, GDML/OBJ meshes, TDR efficiency curves -- none of which exist in the
container); they are stated in DESIGN.md section 5 and follow BASELINE.json
``configs`` / SURVEY.md section 8(d).
"""
from .rng import uniform01  # noqa: F401
from .scenes import Scene, toy_rich_scene, lhcb_like_scene, flat_tables, c2_tables  # noqa: F401
from .photons import cone_point_source, track_photons, CHERENKOV_N  # noqa: F401
from .configs import make_config, CONFIG_NAMES  # noqa: F401
