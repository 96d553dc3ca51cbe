"""Seeded synthetic inputs for the TPMC hot path (meshes + gas/run parameters).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_1312_3691_b200/``).  It holds none of the method's arithmetic: no
Philox, no flux integral, no sampling, no ray tracing -- only geometry
generators and plain parameter records for the five BASELINE.json configs
(recipe in DESIGN.md, section "Input recipe").
"""
from .meshes import (  # noqa: F401
    Mesh,
    plate,
    geodesic_sphere,
    cylinder,
    satellite,
    large_body,
    hemisphere_shell,
    box,
    random_blob,
    lobster_pot,
    stacked_duplicates,
    deep_chain,
)
from .configs import (  # noqa: F401
    AMU,
    K_B,
    RunConfig,
    config,
    config_names,
    fibonacci_directions,
)
