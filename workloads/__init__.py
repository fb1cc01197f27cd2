"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NONE of the method's update arithmetic (no closure, no flux, no
chemistry): it only builds input arrays and the plain numbers that cross the C-ABI
(`emma_rt_config`).  Both `oracle/` and `paper_1508_07888_b200/` are fed the same
bytes from here; neither of them imports this package (the callers do).

Recipes follow SURVEY.md section 8(d); DESIGN.md "Input recipe" restates them.
"""
from .constants import CGS                                    # noqa: F401
from .groups import blackbody_groups, sigma_HI                # noqa: F401
from .fields import gaussian_random_field, lognormal_density  # noqa: F401
from .configs import make_config, make_hii_region_corner, make_shadow_clump, Workload, refine_by_density  # noqa: F401
