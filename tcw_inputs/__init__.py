"""Seeded synthetic inputs for the tCW track-sum path (BASELINE.json:configs).

This package serves both the oracle and the CUDA path.  It holds input *synthesis*
only (noise, timestamps, detector velocities, grid axes, sky grids, injections) and
none of the search arithmetic; neither `oracle/` nor `paper_2507_07816_b200/` imports
it for anything but arrays.
"""
from .configs import (  # noqa: F401
    C_LIGHT,
    CONFIG_NAMES,
    Workload,
    detector_velocity,
    fibonacci_cap,
    fibonacci_sphere,
    make_workload,
    pack_bits,
    random_bank,
    sky_vector,
    synthetic_strain,
    synthetic_weights,
)
