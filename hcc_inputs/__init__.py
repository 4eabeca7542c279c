"""Seeded synthetic inputs (scenes, host BVH, ray batches) shared by the oracle's tests
and the CUDA path's tests.  Holds none of the method's arithmetic (SURVEY.md §8(c)-B0,
§8(d)); neither `oracle/` nor `paper_2305_16652_b200/` is imported from here."""
from . import rng, scenes, bvh, rays, configs  # noqa: F401
from .bvh import BVH, NODE_DTYPE, build_bvh, make_bvh  # noqa: F401
from .configs import CONFIGS, Workload, make_scene  # noqa: F401
