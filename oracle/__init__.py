"""CPU oracle of the two-fluid assembly (TEST INFRASTRUCTURE ONLY).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product package
``paper_1809_02532_b200`` never does.  See ``oracle/tfo.h`` for the rules and the pins.
"""
from .binding import (OracleMesh, Numerics, PhysicsC, build, lib, default_numerics, physics_c,  # noqa: F401
                      assemble, gradients, residual_frozen, flux_maxwell, flux_ausm, flux_face, phys_flux,
                      source, cons, dcons_dprim, num_threads, set_num_threads, ausm_split, wall_ghost, MESH_ITEMS,
                      BC_TRANSMISSIVE, BC_GHOST, BC_WALL)
