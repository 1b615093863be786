"""Seeded synthetic input generators for the MEB workloads.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2605_31425_b200/``).  It holds none of the method's arithmetic: it only
draws balls (centres, radii).  Neither the oracle nor the CUDA path is imported here.

Recipes (stated in DESIGN.md, "Input recipe"):

* ``config(k, ...)`` : the five synthetic configurations of BASELINE.json.
* ``paper_instance(m, d)`` : the deterministic LCG instances of the paper
  ("Test instances").
"""
from .generators import (  # noqa: F401
    BLOCK_ROWS,
    CONFIG_SHAPES,
    config,
    config_blocks,
    config_into,
    paper_instance,
)
