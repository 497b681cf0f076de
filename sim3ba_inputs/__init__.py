"""Seeded synthetic Sim(3) pose-graph inputs (shared by the oracle tests and the CUDA tests).

This package only *draws inputs*: scenes, keyframe poses, pointmaps, confidences, edge lists and
pixel-match maps shaped like the five workloads of BASELINE.json.  It
contains none of the method's arithmetic (no residual, Jacobian, normal equations, Sim(3) Exp/Log,
solve) and imports neither ``oracle/`` nor the CUDA package.
"""
from .graphs import (CONFIG_PARAMS, CONFIGS, DepthInputs, Graph, GraphSpec, PRESETS, clean_variant, config_params,  # noqa: F401
                     make_config, make_depth_inputs, make_graph)
