"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This package holds NO arithmetic of the tracing method (no Philox stream, no sampling,
no packing, no majorant): it only produces the optical-property fields, surface albedo
and run parameters that stand in for the paper's LES cumulus fields (PAPER.md P:40-44,
P:60), which are not available.  Recipe: DESIGN.md §4; configurations: BASELINE.json.
"""
from .fields import (CONFIGS, Config, make_optics, make_optics_torch, factored_point, spectral_points, split_photons,  # noqa: F401
                     plane_parallel)
