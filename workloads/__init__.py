"""Seeded synthetic workloads (input generators only; none of the method's arithmetic)."""
from .configs import Workload, config1, config2, config3, config4, config5, config5_replica, tiny_random, fiber_in_field, fcc_array, ALL  # noqa: F401
from . import geometry  # noqa: F401
