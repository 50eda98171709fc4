"""Seeded synthetic inputs (events, MLP weights) and workload constants shared by tests, bench and smoke.

Holds no arithmetic of the reconstruction method; neither the CUDA package nor oracle/ is imported here.
"""
from . import constants  # noqa: F401
from .events import generate, generate_block, take_events, concat, with_clone_seeds, with_hit_jitter  # noqa: F401
from .mlp import mlp_weights, line_weights, embed_single_hidden, mlp_single_weights  # noqa: F401
