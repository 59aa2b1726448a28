"""CPU oracle for the polarizable-colloid electrostatics hot path (arxiv 2401.04865).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  Nothing under
paper_2401_04865_b200/ imports this package and this package imports nothing
from there.
"""
from .oracle import (  # noqa: F401
    build, M_free, R, R0, dR, ewald_eval, pair_matrix, body_centres, rel_positions,
    solve_induced, forces_torques, default_xi, num_threads, sigma_prime, capacitance, effective_permittivity,
)
from . import dynamics  # noqa: F401,E402  (Brownian-dynamics step and double-layer observables)
