import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def oracle_trace_closest(bvh, rays):
    """Closest-hit tracer handed to the input generator in tests: the oracle's."""
    import oracle
    t, p, _, _ = oracle.closest_bvh(rays, bvh.nodes, bvh.prim_idx, bvh.tris)
    return t, p


class Case:
    """One seeded workload with its first-bounce batches, traced by the oracle."""

    def __init__(self, name, **kw):
        import hcc_inputs
        self.w = hcc_inputs.Workload(name, **kw)
        self.bvh = self.w.bvh
        self.diffuse, self.shadow = self.w.first_bounce(oracle_trace_closest)


@pytest.fixture(scope="session")
def tiny():
    """Config 1 in full: 1,024 triangles, 4,096 diffuse + 8,192 shadow rays."""
    return Case("tiny")


@pytest.fixture(scope="session")
def room_small():
    """Config 2's scene in full (64,012 triangles) at 1/8 resolution, 1 spp: 4,096 + 8,192 rays."""
    return Case("room", res_scale=0.125, spp=1)


@pytest.fixture(scope="session")
def room_mid():
    """Config 2's scene at 1/4 resolution, 4 spp: 65,536 diffuse + 131,072 shadow rays."""
    return Case("room", res_scale=0.25)


def ancestors_of(nodes):
    """parent[] of a canonical BVH."""
    parent = np.full(nodes.shape[0], -1, dtype=np.int64)
    internal = np.nonzero(nodes["count"] == 0)[0]
    left = nodes["left_or_first"][internal].astype(np.int64)
    parent[left] = internal
    parent[left + 1] = internal
    return parent
