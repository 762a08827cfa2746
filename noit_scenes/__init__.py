"""Seeded synthetic inputs for the neural-OIT resolve (input generation only; see raster.py)."""
from .raster import FragBuf, Primitives, rasterize, count_fragments, inject_front_ties  # noqa: F401
from .configs import (Scene, Sequence, cfg1, cfg2, cfg3, cfg4, cfg5, mlp_weights,  # noqa: F401
                      MLP_PARAMS, perspective, view_matrix)
