"""Seeded synthetic input generators (atom systems + weight blobs).

This package serves BOTH the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2506_04055_b200/``).  It holds none of the method's arithmetic: it only
draws random numbers and lays them out.  Recipes follow SURVEY.md §8(d) /
BASELINE.json ``configs`` and are restated in DESIGN.md §4.
"""
from .weights import make_weights, blob_layout, parse_blob, BLOB_MAGIC, HEADER_BYTES  # noqa: F401
from .systems import (  # noqa: F401
    CONFIGS, make_config, water_box, diamond, slab_with_ghosts, peptide_water,
    periodic_ghosts, replicate, extract_cluster, random_gas,
)
