"""Seeded synthetic inputs for the multi-walk force path: particle generators and the host-side
tree / group / interaction-list builder.  Holds none of the method's arithmetic."""
from .generators import CONFIGS, SPH_CONFIGS, Config, make_particles, make_sph_fields, planetary_ring  # noqa: F401
from .tree import Workload, build_tree_and_lists, make_workload, pack_data_lists  # noqa: F401
