"""Seeded ray batches: pinhole primaries and, from a set of
hit records, the diffuse (closest-hit) and shadow (any-hit) batches of one bounce.

A ray is 8 float32: (ox, oy, oz, tmin, dx, dy, dz, tmax), 32 bytes, AoS.
Directions are unit length (computed in float64, rounded once).

The hit records (t, prim) are an INPUT here: whoever calls decides which tracer
produced them (the oracle in the tests).  No intersection code lives in this
module.  Rays come out in primary-sample order, which is the NoSort order
(Table 2 "NoSort").
"""
import numpy as np

from . import rng

_S_CAM, _S_DIFF, _S_LIGHT = 11, 12, 13
MISS_PRIM = 0xFFFFFFFF


def _normalize(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def pack_rays(o, tmin, d, tmax):
    n = o.shape[0]
    r = np.empty((n, 8), dtype=np.float32)
    r[:, 0:3] = o
    r[:, 3] = tmin
    r[:, 4:7] = d
    r[:, 7] = tmax
    return r


def primary_rays(seed, eye, look, up, vfov_deg, width, height, spp, sample_offset=0):
    """width*height*spp rays, index = (py*width + px)*spp + s; sample number
    sample_offset + s selects the sub-pixel jitter."""
    eye = np.asarray(eye, dtype=np.float64)
    fwd = _normalize(np.asarray(look, dtype=np.float64))
    right = _normalize(np.cross(np.asarray(up, dtype=np.float64), fwd))
    upv = np.cross(fwd, right)
    n = width * height * spp
    i = np.arange(n, dtype=np.int64)
    pix, s = i // spp, i % spp + sample_offset
    px, py = pix % width, pix // width
    jx = rng.u01(seed, _S_CAM, pix, 2 * s)
    jy = rng.u01(seed, _S_CAM, pix, 2 * s + 1)
    th = np.tan(np.radians(vfov_deg) * 0.5)
    sx = (2.0 * (px + jx) / width - 1.0) * th * (width / height)
    sy = (1.0 - 2.0 * (py + jy) / height) * th
    d = _normalize(fwd[None, :] + sx[:, None] * right[None, :] + sy[:, None] * upv[None, :])
    o = np.broadcast_to(eye, (n, 3))
    return pack_rays(o, 0.0, d, np.inf)


def _onb(n):
    """Branch-light orthonormal basis around unit vectors n [m,3] (float64)."""
    sign = np.where(n[:, 2] >= 0.0, 1.0, -1.0)
    a = -1.0 / (sign + n[:, 2])
    b = n[:, 0] * n[:, 1] * a
    t = np.stack([1.0 + sign * n[:, 0] * n[:, 0] * a, sign * b, -sign * n[:, 0]], 1)
    bt = np.stack([b, sign + n[:, 1] * n[:, 1] * a, -n[:, 1]], 1)
    return t, bt


def secondary_rays(seed, bounce, rays_in, hit_t, hit_prim, tris, light_center, light_size,
                   shadow_per_hit=2, eps=1e-4):
    """From the hits of `rays_in`: one cosine-weighted diffuse ray and
    `shadow_per_hit` shadow rays per hit, in the order of the incoming rays.

    Returns (diffuse [h,8], shadow [h*shadow_per_hit,8], src [h]) where src[k] is the
    index in rays_in of the k-th hit.  Origin = hit point + eps * n with n the geometric
    normal on the side the ray came from.  Diffuse: tmin 0, tmax +inf.  Shadow: unit
    direction to a uniform sample of the light quad (in the plane y = light_center[1]),
    tmin 0, tmax = distance * (1 - eps)."""
    hit_prim = np.asarray(hit_prim)
    hit = hit_prim != MISS_PRIM
    src = np.nonzero(hit)[0]
    r = rays_in[src].astype(np.float64)
    t = np.asarray(hit_t)[src].astype(np.float64)
    tri = np.asarray(tris, dtype=np.float32).reshape(-1, 3, 3)[hit_prim[src].astype(np.int64)].astype(np.float64)
    o_in, d_in = r[:, 0:3], r[:, 4:7]
    p = o_in + t[:, None] * d_in
    ng = _normalize(np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0]))
    flip = np.einsum("ij,ij->i", ng, d_in) > 0.0
    ng[flip] = -ng[flip]
    org = p + eps * ng

    # diffuse: r = sqrt(u1), phi = 2 pi u2 about n
    u1 = rng.u01(seed, _S_DIFF, src, 2 * bounce)
    u2 = rng.u01(seed, _S_DIFF, src, 2 * bounce + 1)
    rad, phi = np.sqrt(u1), 2.0 * np.pi * u2
    tx, ty = _onb(ng)
    dl = np.stack([rad * np.cos(phi), rad * np.sin(phi), np.sqrt(np.maximum(0.0, 1.0 - u1))], 1)
    dd = _normalize(dl[:, 0:1] * tx + dl[:, 1:2] * ty + dl[:, 2:3] * ng)
    diffuse = pack_rays(org, 0.0, dd, np.inf)

    # shadow rays
    lc = np.asarray(light_center, dtype=np.float64)
    h = src.shape[0]
    so = np.repeat(org, shadow_per_hit, axis=0)
    k = np.repeat(src, shadow_per_hit)
    s = np.tile(np.arange(shadow_per_hit), h)
    dim = (bounce * shadow_per_hit + s) * 2
    lx = lc[0] + (rng.u01(seed, _S_LIGHT, k, dim) - 0.5) * light_size
    lz = lc[2] + (rng.u01(seed, _S_LIGHT, k, dim + 1) - 0.5) * light_size
    L = np.stack([lx, np.full_like(lx, lc[1]), lz], 1)
    v = L - so
    dist = np.linalg.norm(v, axis=1)
    sd = v / dist[:, None]
    shadow = pack_rays(so, 0.0, sd, dist * (1.0 - eps))
    return diffuse, shadow, src
