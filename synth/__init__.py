"""Seeded synthetic inputs for the M3D-C1-K particle-push hot path.

This package only *generates inputs* (analytic tokamak fields, triangle meshes,
per-element least-squares polynomial tables, marker loads).  It contains none of
the method's arithmetic (no pusher, no finite-element evaluation, no weight
equation, no element search, no sort) and is the only code shared by the CPU
oracle (``oracle/``) and the CUDA path (``paper_2107_13663_b200/``).

Recipes follow SURVEY.md section 8(d) D1 and the readings G14, G17-G20; they are
restated in DESIGN.md section 4.
"""
from .tokamak import CircularTokamak, Perturbation, Harmonic  # noqa: F401
from .mesh import rect_tri_mesh, lattice_points, fit_tables, monomial_exponents  # noqa: F401
from .markers import load_markers, slow_manifold_velocity  # noqa: F401
from .configs import make_config, CONFIGS, Workload, F0Params  # noqa: F401
