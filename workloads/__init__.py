"""Seeded synthetic inputs for the SeKV decode hot path.

This package is the ONLY code shared by the oracle (``oracle/``) and the CUDA path
(``paper_2606_31145_b200/``).  It holds input synthesis only -- span-length draws, surprisal
values, random orthonormal factors, anchors, routing projections and queries -- and none of the
method's arithmetic (no segmentation rule, no summaries, no routing score, no attention).
The recipe is stated in DESIGN.md section 4 and follows BASELINE.json ``configs`` / SURVEY.md 8(d).
"""
from .configs import WorkloadSpec, CONFIGS, get_spec, seed_for  # noqa: F401
from .generators import (  # noqa: F401
    SequenceLayout,
    LayerInputs,
    make_layouts,
    make_layer_inputs,
    make_queries,
    make_routing_weights,
    next_queries_ar1,
    storage_torch_dtype,
)
