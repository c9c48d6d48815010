"""Seeded synthetic inputs shared by the oracle and the CUDA path (no method arithmetic)."""
from .mesh import Mesh, rect_mesh, make_mesh, build_edge_tables, vertex_to_modal_p1, signed_areas  # noqa: F401
from .configs import Workload, c1, c2, c3, c4, c5, FULL, cfl_dt, default_params, holland_default, perturbed, with_forcing  # noqa: F401
