"""Seeded synthetic scenes shaped like the paper's workloads.

The paper's scenes are not available; these stand in
for them: "complex small objects inside a large room" at
the triangle counts BASELINE.json's configs state.  All coordinates are
computed in float64 and rounded once to float32, so the arrays are the same on
every machine.  No ray tracing or BVH arithmetic lives here.
"""
import numpy as np

from . import rng

# stream ids for the counter-based RNG
_S_TRI, _S_MEAN, _S_SPHERE, _S_SLAB = 1, 2, 3, 4


# ----------------------------------------------------------------------------
# primitives
# ----------------------------------------------------------------------------
def room_box(lo=0.0, hi=1.0):
    """12 inward-facing triangles of the axis-aligned box [lo,hi]^3."""
    l, h = float(lo), float(hi)
    c = np.array([[l, l, l], [h, l, l], [h, h, l], [l, h, l],
                  [l, l, h], [h, l, h], [h, h, h], [l, h, h]], dtype=np.float64)
    # quads listed so that the normal (v1-v0)x(v2-v0) points into the room
    quads = [(0, 1, 2, 3),   # z = lo, normal +z
             (5, 4, 7, 6),   # z = hi, normal -z
             (4, 0, 3, 7),   # x = lo, normal +x
             (1, 5, 6, 2),   # x = hi, normal -x
             (4, 5, 1, 0),   # y = lo, normal +y
             (3, 2, 6, 7)]   # y = hi, normal -y
    tris = []
    for a, b, cc, d in quads:
        tris.append([c[a], c[b], c[cc]])
        tris.append([c[a], c[cc], c[d]])
    return np.asarray(tris, dtype=np.float64)


def icosphere(level):
    """Unit icosphere as a triangle soup, 20 * 4**level triangles, float64.

    Midpoints are (a + b) normalised; a + b is commutative in IEEE arithmetic,
    so a vertex shared by two faces is bit-identical in both (no cracks).
    """
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
                  [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
                  [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]])
    tris = v[f]                                   # [20,3,3]
    for _ in range(level):
        a, b, c = tris[:, 0], tris[:, 1], tris[:, 2]

        def mid(p, q):
            m = p + q
            return m / np.linalg.norm(m, axis=1, keepdims=True)
        ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
        tris = np.concatenate([np.stack([a, ab, ca], 1), np.stack([b, bc, ab], 1),
                               np.stack([c, ca, bc], 1), np.stack([ab, bc, ca], 1)], 0)
    return tris


def _instances(template, centres, radii):
    """template [T,3,3] scaled by radii [M] and moved to centres [M,3] -> [M*T,3,3]."""
    out = template[None, :, :, :] * radii[:, None, None, None] + centres[:, None, None, :]
    return out.reshape(-1, 3, 3)


def clustered_spheres(seed, count, level, n_clusters, mean_lo, mean_hi, sigma, mu_r, sigma_r):
    """`count` icospheres; centres from an equal-weight isotropic Gaussian mixture whose
    means are U[mean_lo, mean_hi]^3; radius = exp(N(mu_r, sigma_r^2)); centres clamped
    to [r, 1-r] so every sphere stays inside the unit room."""
    k = np.arange(n_clusters)
    means = mean_lo + (mean_hi - mean_lo) * np.stack(
        [rng.u01(seed, _S_MEAN, k, d) for d in range(3)], 1)
    i = np.arange(count)
    comp = np.minimum((rng.u01(seed, _S_SPHERE, i, 0) * n_clusters).astype(np.int64), n_clusters - 1)
    centres = means[comp] + sigma * np.stack(
        [rng.normal01(seed, _S_SPHERE, i, 1 + d) for d in range(3)], 1)
    radii = np.exp(mu_r + sigma_r * rng.normal01(seed, _S_SPHERE, i, 4))
    radii = np.minimum(radii, 0.2)
    centres = np.clip(centres, radii[:, None] + 1e-3, 1.0 - radii[:, None] - 1e-3)
    return _instances(icosphere(level), centres, radii)


_BOX_CORNERS = np.array([[-1, -1, -1], [1, -1, -1], [1, 1, -1], [-1, 1, -1],
                         [-1, -1, 1], [1, -1, 1], [1, 1, 1], [-1, 1, 1]], dtype=np.float64)
_BOX_QUADS = [(0, 3, 2, 1), (4, 5, 6, 7), (0, 4, 7, 3), (1, 2, 6, 5), (0, 1, 5, 4), (3, 7, 6, 2)]


def thin_slabs(seed, count, thin_lo, thin_hi, wide_lo, wide_hi):
    """`count` boxes ("furniture"): one extent U(thin_lo, thin_hi), the other two
    U(wide_lo, wide_hi), thin axis drawn uniformly, then a random yaw about y;
    12 outward-facing triangles each, centres uniform so the box stays in the room."""
    i = np.arange(count)
    ext = wide_lo + (wide_hi - wide_lo) * np.stack(
        [rng.u01(seed, _S_SLAB, i, d) for d in range(3)], 1)
    thin = thin_lo + (thin_hi - thin_lo) * rng.u01(seed, _S_SLAB, i, 3)
    axis = np.minimum((rng.u01(seed, _S_SLAB, i, 4) * 3).astype(np.int64), 2)
    ext[i, axis] = thin
    half = 0.5 * ext
    yaw = 2.0 * np.pi * rng.u01(seed, _S_SLAB, i, 5)
    reach_xz = np.sqrt(half[:, 0] ** 2 + half[:, 2] ** 2) + 1e-3
    reach = np.stack([reach_xz, half[:, 1] + 1e-3, reach_xz], 1)
    centres = reach + (1.0 - 2.0 * reach) * np.stack(
        [rng.u01(seed, _S_SLAB, i, 6 + d) for d in range(3)], 1)
    corners = _BOX_CORNERS[None, :, :] * half[:, None, :]            # [M,8,3]
    c, s = np.cos(yaw)[:, None], np.sin(yaw)[:, None]
    x, z = corners[:, :, 0].copy(), corners[:, :, 2].copy()
    corners[:, :, 0] = c * x + s * z
    corners[:, :, 2] = -s * x + c * z
    corners += centres[:, None, :]
    tris = []
    for a, b, cc, d in _BOX_QUADS:
        tris.append(np.stack([corners[:, a], corners[:, b], corners[:, cc]], 1))
        tris.append(np.stack([corners[:, a], corners[:, cc], corners[:, d]], 1))
    return np.stack(tris, 1).reshape(-1, 3, 3)                       # [M*12,3,3]


def random_triangles(seed, count, edge_lo, edge_hi):
    """Config 1: centroid U[0,1]^3, uniformly random orientation, equilateral with
    edge length U(edge_lo, edge_hi)."""
    i = np.arange(count)
    cen = np.stack([rng.u01(seed, _S_TRI, i, d) for d in range(3)], 1)
    edge = edge_lo + (edge_hi - edge_lo) * rng.u01(seed, _S_TRI, i, 3)
    q = np.stack([rng.normal01(seed, _S_TRI, i, 2 + d) for d in range(4)], 1)  # uniform quaternion
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], 1),
                  np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], 1),
                  np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], 1)], 1)
    rad = edge / np.sqrt(3.0)                                         # circumradius
    ang = np.array([0.0, 2.0 * np.pi / 3.0, 4.0 * np.pi / 3.0])
    local = np.stack([np.cos(ang), np.sin(ang), np.zeros(3)], 1)       # [3 verts, 3]
    verts = np.einsum("mij,vj->mvi", R, local) * rad[:, None, None] + cen[:, None, :]
    return verts


def to_f32(tris):
    """[N,3,3] float64 -> C-contiguous float32 (one rounding)."""
    return np.ascontiguousarray(tris, dtype=np.float32)
