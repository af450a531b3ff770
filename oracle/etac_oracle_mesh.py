"""CPU oracle for the signed distance to a closed TRIANGLE MESH  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:L77: "contact events are first detected using SDFs between nodes and object meshes".  The product takes
object SDFs as sampled grids (ETAC_IND_GRID, R21); ``etac_mesh_to_sdf_grid`` (include/etac.h) samples the SDF of
a watertight triangle mesh onto such a grid.  This file states what that SDF is, in plain float64 numpy, one
triangle at a time, no acceleration structure:

    dist(x)  = min over the triangles of || x - closest point of the triangle ||      (the plain definition)
    inside   = | winding number w(x) | >= 1/2,   w(x) = (1 / 4 pi) * sum over the triangles of the signed solid angle
               the triangle subtends at x  (for a closed surface w is 0 outside and +-1 inside, whatever the
               orientation of the triangles, as long as it is consistent)
    phi(x)   = -dist(x) inside, +dist(x) outside

The closest point of a triangle is found by the barycentric region tests of the standard construction (vertex,
edge or face region of the point's projection); the solid angle of a triangle (a, b, c) seen from the origin is
    Omega = 2 atan2( a . (b x c),  |a||b||c| + (a . b)|c| + (b . c)|a| + (c . a)|b| )
(Van Oosterom & Strackee 1983).  Same rules as etac_oracle.py: only tests / smoke / bench baselines import it; no code
shared with the CUDA path.  Pins: tests/test_oracle_pins.py (closed-form box and sphere, face-plane distances inside a
tetrahedron, brute-force ray parity for the sign, invariance under triangle order and orientation).
"""
from __future__ import annotations

import numpy as np


def closest_point_on_triangle(p, a, b, c):
    """p [n, 3]; a, b, c [3] -> closest points [n, 3] of the (closed) triangle abc to every p."""
    p = np.asarray(p, dtype=np.float64)
    a, b, c = (np.asarray(v, dtype=np.float64) for v in (a, b, c))
    ab, ac, ap = b - a, c - a, p - a
    d1, d2 = ap @ ab, ap @ ac
    bp = p - b
    d3, d4 = bp @ ab, bp @ ac
    cp = p - c
    d5, d6 = cp @ ab, cp @ ac
    vc = d1 * d4 - d3 * d2
    vb = d5 * d2 - d1 * d6
    va = d3 * d6 - d5 * d4
    out = np.empty_like(p)
    done = np.zeros(p.shape[0], dtype=bool)

    def put(mask, pts):
        m = mask & ~done
        out[m] = pts[m] if pts.ndim == 2 else pts
        done[m] = True

    put((d1 <= 0) & (d2 <= 0), a)                                              # vertex region a
    put((d3 >= 0) & (d4 <= d3), b)                                             # vertex region b
    with np.errstate(divide="ignore", invalid="ignore"):
        t = d1 / (d1 - d3)
        put((vc <= 0) & (d1 >= 0) & (d3 <= 0), a + t[:, None] * ab)            # edge ab
        put((d6 >= 0) & (d5 <= d6), c)                                         # vertex region c
        t = d2 / (d2 - d6)
        put((vb <= 0) & (d2 >= 0) & (d6 <= 0), a + t[:, None] * ac)            # edge ac
        t = (d4 - d3) / ((d4 - d3) + (d5 - d6))
        put((va <= 0) & ((d4 - d3) >= 0) & ((d5 - d6) >= 0), b + t[:, None] * (c - b))   # edge bc
        den = 1.0 / (va + vb + vc)
        v, w = vb * den, vc * den
        put(np.ones_like(done), a + v[:, None] * ab + w[:, None] * ac)          # face region
    return out


def solid_angle(p, a, b, c):
    """Signed solid angle [n] that the triangle abc subtends at every p [n, 3]."""
    p = np.asarray(p, dtype=np.float64)
    ra, rb, rc = a - p, b - p, c - p
    la, lb, lc = (np.linalg.norm(r, axis=1) for r in (ra, rb, rc))
    det = np.einsum("ij,ij->i", ra, np.cross(rb, rc))
    den = la * lb * lc + np.einsum("ij,ij->i", ra, rb) * lc + np.einsum("ij,ij->i", rb, rc) * la + np.einsum("ij,ij->i", rc, ra) * lb
    return 2.0 * np.arctan2(det, den)


def mesh_signed_distance(vertices, triangles, points):
    """phi [n] of the closed triangle mesh (vertices [nv, 3], triangles [nt, 3] vertex indices) at points [n, 3]."""
    V = np.asarray(vertices, dtype=np.float64)
    T = np.asarray(triangles, dtype=np.int64)
    P = np.asarray(points, dtype=np.float64).reshape(-1, 3)
    best = np.full(P.shape[0], np.inf)
    omega = np.zeros(P.shape[0])
    for i0, i1, i2 in T:
        a, b, c = V[i0], V[i1], V[i2]
        q = closest_point_on_triangle(P, a, b, c)
        best = np.minimum(best, np.linalg.norm(P - q, axis=1))
        omega += solid_angle(P, a, b, c)
    inside = np.abs(omega) >= 2.0 * np.pi                                      # |w| >= 1/2
    return np.where(inside, -best, best)


def mesh_sdf_grid(vertices, triangles, shape, origin, spacing):
    """values[iz, iy, ix] = phi(origin + spacing * (ix, iy, iz)) for shape = (nx, ny, nz): the layout of
    etac_set_sdf_grid / etac_oracle.sdf_grid."""
    nx, ny, nz = shape
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    pts = np.asarray(origin, dtype=np.float64) + float(spacing) * np.stack([ix, iy, iz], axis=-1).reshape(-1, 3)
    return mesh_signed_distance(vertices, triangles, pts).reshape(nz, ny, nx)
