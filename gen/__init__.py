"""Seeded synthetic workload generator (inputs only; no method arithmetic)."""
from .tpcgen import (Config, as_numpy_digits, clusters_per_row, config, fnv1a64,  # noqa: F401
                     generate_fragment, geometry_npads)
