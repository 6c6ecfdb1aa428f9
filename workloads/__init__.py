"""Seeded synthetic OSOG scenes (BASELINE.json `configs`; recipe in DESIGN.md §4).

This module only DRAWS inputs.  It contains none of the method's arithmetic (no rotation
matrices, no thickness, no binning, no optics) and imports neither `oracle/` nor the CUDA
package; both sides are fed the same float32 arrays it returns.
"""
from .configs import Scene, make_config, make_scene, CONFIG_NAMES, subset  # noqa: F401
