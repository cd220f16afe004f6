"""Seeded synthetic scenario generators (inputs only).

This package serves BOTH the CUDA path and the CPU oracle, so it holds none of the method's
arithmetic: no dynamics step (Eq. 1/2), no metric, no observation transform.  It only lays
out roadgraph polylines and draws agents, logged trajectories and actions with the shapes,
sizes and value ranges BASELINE.json's five configs name (stand-ins for WOMD, PAPER.md L78,
L176).  Logged trajectories are exact constant-acceleration / constant-curvature arcs in
closed form (a data recipe, deliberately *not* the paper's discrete bicycle update).

Randomness is counter-based: every draw is hash(seed, config, scenario b, stream, i), so
scenario ``b`` is identical whatever batch it is generated in (rank shards, parity samples).
"""
from .rng import uniform, randint, MASTER_SEED
from .configs import (
    make_config,
    make_paths,
    make_street_scenarios,
    make_config1,
    make_config4,
    CONFIG_SHAPES,
    TYPE_LANE,
    TYPE_ROAD_EDGE,
)

__all__ = [
    "uniform", "randint", "MASTER_SEED", "make_config", "make_paths", "make_street_scenarios",
    "make_config1", "make_config4", "CONFIG_SHAPES", "TYPE_LANE", "TYPE_ROAD_EDGE",
]
