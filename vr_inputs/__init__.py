"""Seeded synthetic inputs (cubes, transfer-function tables, cameras, pixel
subsets) that serve BOTH the CPU oracle and the CUDA path.

This package holds none of the rendering method's arithmetic: it only makes
input bytes.  Recipes follow BASELINE.json `configs` and SURVEY.md Sec. 8(d).1-2
and are restated in DESIGN.md Sec. 4; they stand in for ASKAP spectral cubes
(PAPER.md:17-19), which are not available offline.
"""
from .cubes import (CONFIGS, CubeSpec, make_cube, make_box, noise_box, brick_boxes,  # noqa: F401
                    sources_in_box, source_params, ooc_spec)
from .luts import lut_a, lut_s, lut_5sigma  # noqa: F401
from .cameras import (config0_views, orbit_camera, orbit_views, ortho_axis_camera,  # noqa: F401
                      rotate_about_y)
from .pixels import tile_subset  # noqa: F401
