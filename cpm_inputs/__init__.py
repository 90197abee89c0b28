"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs C1..C5; C6, C7: the SURVEY 8(f) motility workloads).

This module serves BOTH the oracle tests and the CUDA path (tests, bench.py).  It holds none of
the method's arithmetic: it only paints initial lattices, frozen masks, type tables and draws
parameter tables from a seed.  Recipes and what they stand in for are stated in DESIGN.md
("Input recipe").  numpy only.
"""
from .generators import (  # noqa: F401
    make_config, config_names, ball_moore_perimeter, jittered_cubes, obstacle_network,
    crop_config, circular_field,
)
