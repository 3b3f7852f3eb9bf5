"""Seeded synthetic inputs shared by the oracle tests and the CUDA-path tests.

This package is the ONLY code both sides use.  It builds block-sparse *inputs*
(labels, extents, placement, values) shaped like the paper's DMRG scratch data
(Fig 4(a) L75; recipe in DESIGN.md "Input recipe") and holds
none of the serializer's arithmetic: no 16-byte rounding, no stream offsets, no
header fields.  It imports neither ``oracle`` nor ``paper_2412_04676_b200``.
"""
from .blocksparse import (  # noqa: F401
    BASE_SEED,
    CONFIGS,
    LAYER_REC_DTYPE,
    STRUCT_REC_DTYPE,
    TENSOR_REC_DTYPE,
    BlockSparseSet,
    label_grid,
    layered_view,
    make_config,
    make_set,
    make_tree_set,
    selection_rules,
)
from .values import block_values, fill_pool_host, splitmix64_at  # noqa: F401
