"""ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle/mwf_oracle.c and DESIGN.md "Oracle").

Python front end of the fp64 CPU oracle plus `bhtree_ref`, a plain Python restatement of the
tree / group / list construction used to pin the fast host builder.  Nothing under
paper_1907_02290_b200/ imports this package; only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs do.  Parity status: every function here is pinned by
tests/test_oracle_pins.py (closed forms, brute force, invariants); nothing is "parity unpinned".
"""
from .oracle import (build, direct, forces, kick, kick_drift, monopoles, num_threads, quadrupoles, set_num_threads,  # noqa: F401
                     sph_density, sph_density_direct, sph_dwdr, sph_hydro, sph_hydro_direct, sph_w)
