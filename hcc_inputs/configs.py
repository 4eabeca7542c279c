"""BASELINE.json's configs as seeded recipes; DESIGN.md restates them.

`make_scene(name)` -> float32 triangles; `Workload(name)` adds the BVH, the camera and
the per-bounce ray batches.  Tracing the primaries / previous bounce needs a closest-hit
tracer; it is passed in (`trace_closest(bvh, rays) -> (t, prim)`), so this module has no
intersection code.  `scale` < 1 shrinks object counts and resolution for fast CPU tests.
"""
import numpy as np

from . import bvh as _bvh
from . import rays as _rays
from . import scenes as _sc

SEED_BASE = 0x230516652000

CONFIGS = {
    # name: dict(...)
    "tiny": dict(idx=1, K=64, key_bits=32, width=64, height=64, spp=1, bounces=1,
                 n_diffuse=4096, eye=(0.5, 0.5, -1.2), look=(0, 0, 1), vfov=45.0,
                 light_center=(0.5, 1.2, 0.5), light_size=0.2),
    "room": dict(idx=2, K=1024, key_bits=32, width=512, height=512, spp=4, bounces=1,
                 eye=(0.5, 0.5, 0.02), look=(0, 0, 1), vfov=60.0,
                 light_center=(0.5, 0.999, 0.5), light_size=0.2),
    "fig1": dict(idx=3, K=4096, key_bits=64, width=1920, height=1080, spp=8, bounces=3,
                 eye=(0.5, 0.5, 0.02), look=(0, 0, 1), vfov=60.0,
                 light_center=(0.5, 0.999, 0.5), light_size=0.2),
    "large": dict(idx=5, K=16384, key_bits=64, width=1920, height=1080, spp=16, bounces=4,
                  eye=(0.5, 0.5, 0.02), look=(0, 0, 1), vfov=60.0,
                  light_center=(0.5, 0.999, 0.5), light_size=0.2),
}


def seed_of(name):
    return SEED_BASE + CONFIGS[name]["idx"]


def make_scene(name, scale=1.0):
    """Triangles [N,3,3] float32 of config `name`.  scale multiplies object counts."""
    seed = seed_of(name)
    s = float(scale)

    def cnt(x):
        return max(1, int(round(x * s)))
    if name == "tiny":
        tris = _sc.random_triangles(seed, cnt(1024), 0.01, 0.05)
    elif name == "room":
        # 12 + 200*320 = 64,012 triangles
        tris = np.concatenate([
            _sc.room_box(),
            _sc.clustered_spheres(seed, cnt(200), 2, 4, 0.2, 0.8, 0.08, -3.5, 0.5)], 0)
    elif name == "fig1":
        # 12 + 180*5120 + 6500*12 = 999,612 triangles
        tris = np.concatenate([
            _sc.room_box(),
            _sc.clustered_spheres(seed, cnt(180), 4, 6, 0.15, 0.85, 0.06, -3.2, 0.4),
            _sc.thin_slabs(seed, cnt(6500), 0.002, 0.01, 0.03, 0.25)], 0)
    elif name == "large":
        # 12 + 30000*320 + 100000*12 = 10,800,012 triangles (level-2 spheres: SURVEY §8(d))
        tris = np.concatenate([
            _sc.room_box(),
            _sc.clustered_spheres(seed, cnt(30000), 2, 24, 0.1, 0.9, 0.07, -4.8, 0.4),
            _sc.thin_slabs(seed, cnt(100000), 0.001, 0.004, 0.01, 0.06)], 0)
    else:
        raise KeyError(name)
    return _sc.to_f32(tris)


class Workload:
    """Scene + BVH + ray batches of one config.

    res_scale shrinks the image (fewer rays), scene_scale the object counts."""

    def __init__(self, name, scene_scale=1.0, res_scale=1.0, spp=None, rank=0):
        self.name = name
        self.cfg = dict(CONFIGS[name])
        self.seed = seed_of(name) + 0x10000 * int(rank)   # rank-specific samples, same scene
        self.tris = make_scene(name, scene_scale)
        self.bvh = _bvh.build_bvh(self.tris, max_leaf=4, n_bins=16)
        self.width = max(8, int(round(self.cfg["width"] * res_scale)))
        self.height = max(8, int(round(self.cfg["height"] * res_scale)))
        self.spp = int(spp if spp is not None else self.cfg["spp"])
        self.K = self.cfg["K"]
        self.key_bits = self.cfg["key_bits"]

    def primaries(self, sample_offset=0, spp=None):
        c = self.cfg
        return _rays.primary_rays(self.seed, c["eye"], c["look"], (0, 1, 0), c["vfov"],
                                  self.width, self.height, self.spp if spp is None else spp,
                                  sample_offset)

    def bounce(self, bounce, rays_in, hit_t, hit_prim):
        c = self.cfg
        return _rays.secondary_rays(self.seed, bounce, rays_in, hit_t, hit_prim, self.tris,
                                    c["light_center"], c["light_size"])

    def first_bounce(self, trace_closest):
        """(diffuse, shadow) batches of bounce 1.  For "tiny", passes of one sample per
        pixel are cast until n_diffuse hits are collected."""
        want = self.cfg.get("n_diffuse")
        if want is None:
            prim = self.primaries()
            t, p = trace_closest(self.bvh, prim)
            d, s, _ = self.bounce(1, prim, t, p)
            return d, s
        want = max(1, int(round(want * (self.width * self.height) / (self.cfg["width"] * self.cfg["height"]))))
        ds, ss, got, k = [], [], 0, 0
        while got < want and k < 64:
            prim = self.primaries(sample_offset=k, spp=1)
            t, p = trace_closest(self.bvh, prim)
            # sample number k enters the per-hit random dimensions through `bounce`
            d, s, _ = _rays.secondary_rays(self.seed + 0x100 * k, 1, prim, t, p, self.tris,
                                           self.cfg["light_center"], self.cfg["light_size"])
            ds.append(d); ss.append(s); got += d.shape[0]; k += 1
        d = np.concatenate(ds, 0)[:want]
        s = np.concatenate(ss, 0)[:2 * want]
        return np.ascontiguousarray(d), np.ascontiguousarray(s)
