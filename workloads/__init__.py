"""Seeded synthetic inputs (AMR layouts, surface densities, target samples).

This package holds NONE of the method's arithmetic: it only produces the inputs
that both the CPU oracle (``oracle/``) and the CUDA library
(``paper_2001_02765_b200/``) consume.  Neither of those imports the other; both
may import this.
"""
from .configs import (Layout, CONFIG_NAMES, make_config, cell_rects, expected_counts,
                      sample_targets, paper_ilr_layout, paper_vlr_layout, d2_sigma,
                      d2_slopes, d22_sigma, d22_slopes, nested_layout, kuzmin_sigma, random_refined_layout,
                      make_config4_variant)
