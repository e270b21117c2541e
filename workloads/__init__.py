"""Seeded synthetic workloads shaped like the paper's (BASELINE.json:configs).

This package holds ONLY input generation: shapes, topologies and random draws.
It contains none of the method's arithmetic (no Hadamard transform, no cos, no
Gram product), and it imports neither `oracle/` nor the CUDA package, so both
sides can be fed the same arrays without sharing code.
"""
from .configs import (  # noqa: F401
    ELEMENTS,
    DescriptorGradient,
    SorfModel,
    Workload,
    make_model,
    make_workload,
    tiny_workload,
    CONFIG_NAMES,
    ProjectionInputs,
    projection_inputs,
)
from .geometry import FchlParams, FCHL_E, Geometry, molecules_geometry, cell_geometry  # noqa: F401
