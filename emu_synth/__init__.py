"""Seeded synthetic emulsion views (inputs only).

This package serves both the CPU oracle (``oracle/``) and the CUDA library
(``paper_1311_5334_b200/``).  It holds NONE of the track-finding arithmetic:
it only draws grain clouds with the shapes, densities and structure of
BASELINE.json's five configs (recipe: DESIGN.md "Input recipe", after
SURVEY.md 8(d)).  It imports neither the oracle nor the CUDA package.
"""
from .views import (CONFIGS, Q_PER_UM, ViewBatch, default_params, make_batch,
                    make_config, make_view, noiseless_track_view)

__all__ = ["CONFIGS", "Q_PER_UM", "ViewBatch", "default_params", "make_batch",
           "make_config", "make_view", "noiseless_track_view"]
