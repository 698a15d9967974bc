"""Seeded synthetic input generators (no method arithmetic). See configs.py."""
from .bundle import GRID_DEFAULTS, bsr_pad_mask, bsr_to_dense, build_bsr, dense_to_bsr, make_config, make_q_values, make_xi  # noqa: F401
from .configs import (BASE_SEED, SPECIES, Bundle, bisect_batches, build_splines, cutoff_fn,  # noqa: F401
                      fibonacci_sphere, partition_weights, radial_analytic, radial_grid, smooth_fields)
from .periodic import make_periodic, make_periodic_si  # noqa: F401,E402
