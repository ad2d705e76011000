"""Seeded synthetic planetesimal-disk inputs for the GENGA kick + encounter pre-check path.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2201_10058_b200/``) and therefore holds none of the method's arithmetic
(no changeover function, no force, no encounter test).  It only produces the *inputs*
of the path: heliocentric positions/velocities, masses and the per-body critical-radius
rows (eq. 5; PAPER.md:638 for the per-level rows).

Recipes follow BASELINE.json ``configs`` / SURVEY.md section 8(d); see DESIGN.md "Input recipe".
"""
from .splitmix import splitmix64, uniforms
from .disks import (
    K_GAUSS, G_AU_DAY_MSUN, M_EARTH, M_JUPITER, DT_DAYS, N1_HILL, N2_VEL,
    KickInputs, elements_to_cartesian, semi_major_axis, rcrit_rows,
    make_disk, make_config, make_ring, CONFIG_NAMES,
)

__all__ = [
    "splitmix64", "uniforms", "K_GAUSS", "G_AU_DAY_MSUN", "M_EARTH", "M_JUPITER", "DT_DAYS",
    "N1_HILL", "N2_VEL", "KickInputs", "elements_to_cartesian", "semi_major_axis", "rcrit_rows",
    "make_disk", "make_config", "make_ring", "CONFIG_NAMES",
]
