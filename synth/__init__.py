"""Seeded synthetic input generators (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic (no Dirac operator, no clover
term, no boundary logic): it only draws the random SU(3) links, U(1) fields and
Gaussian spinors described in DESIGN.md "Input recipe" (SURVEY.md §8(d),
BASELINE.json configs).  Values are a pure function of
(seed, field id, lexicographic site, direction, component) through a
counter-based generator, so they do not depend on traversal order, chunking,
thread count or language.
"""
from .fields import (  # noqa: F401
    splitmix64,
    uniform01,
    normal,
    su3_links,
    su3_links_smooth,
    u1_field,
    gaussian_spinor,
    random_su3,
    CONFIGS,
    config,
)
