"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no RBF, no message passing, no
neighbour predicate used by either implementation): it only draws atomic numbers,
positions, cells, head indices and weight blobs from counter-based random streams,
in the shapes of BASELINE.json's five configs (recipe: DESIGN.md "Input recipe").
"""
from .synth import (  # noqa: F401
    BASE_SEED,
    Batch,
    ModelCfg,
    CONFIGS,
    model_cfg,
    weights_count,
    weights_layout,
    make_weights,
    make_head_weights,
    BRANCH_MLP_WIDTHS,
    branch_mlp_count,
    make_branch_mlp,
    make_batch,
    make_molecules,
    make_crystals,
    concat_batches,
)
