"""Seeded synthetic inputs for libwtide: geometry descriptors of the five BASELINE.json
configs and track / carrier / trajectory generators.

This package serves BOTH the oracle-side tests and the CUDA-side tests / bench.  It holds
none of the method's arithmetic (no PDE solve, no Eq. 1.1): it only builds descriptors and
draws inputs.  The recipe is stated in DESIGN.md ("Synthetic inputs").
"""
from .configs import CONFIG_NAMES, geometry_desc, reduced_desc, sweep_descs  # noqa: F401
from .rng import uniform  # noqa: F401
from .tracks import (make_tracks, carriers_on_tracks, straight_drift_cfg0,  # noqa: F401
                     field_drift, concat_csr)
