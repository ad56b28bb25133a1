"""Seeded synthetic inputs shaped like the paper's workloads.

This package is the ONLY code shared by the CUDA path (``paper_2504_08081_b200``)
and the test oracle (``oracle``).  It holds none of the method's arithmetic: no
interpolation, no colour law, no band integral, no chi^2.  It only draws random
numbers and tabulates closed-form synthetic surfaces / filters (recipe: DESIGN.md
"Input recipe", following SURVEY.md section 8(d) and BASELINE.json `configs`).
"""
from .generators import (  # noqa: F401
    CONFIG_IDS,
    Workload,
    attach_data,
    jitter_band_grids,
    make_bands,
    make_colour_law,
    make_model,
    make_workload,
    shard_bounds,
    subset,
)
