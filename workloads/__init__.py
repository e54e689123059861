"""Seeded synthetic inputs for the VRC ray-cast hot path.

This package holds ONLY input generation (meshes, material maps, cross-section
tables, ray batches).  It contains none of the method's arithmetic (no
interpolation, no traversal, no scoring) and is the one module both the CUDA
path's tests/bench and the CPU oracle's tests are allowed to share.
"""
from .configs import (  # noqa: F401
    CONFIG_NAMES,
    FULL_RAYS,
    Problem,
    add_nuclides,
    make_problem,
    make_rays,
    make_rz_problem,
    make_rz_rays,
    rng_for,
)
