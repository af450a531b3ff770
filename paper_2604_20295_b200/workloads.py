"""Seeded synthetic workloads for the ETac tactile hot path.

This module only *places* geometry: sensor meshes, indenter shapes/poses, patch poses and
random MLP weights.  It holds none of the method's arithmetic (no SDF evaluation, no decay
kernel, no MLP) so that the CPU oracle (``oracle/``) and the CUDA path can both consume its
outputs without sharing any of the code under test.  Everything is rounded to fp32 before it
is handed out ("the oracle consumes the same fp32-rounded input arrays").

The paper's own workloads (ShadowHand in Isaac Gym, FEM elastomer datasets; PAPER.md:L114,
L145) are not available; these inputs take their shapes and statistics (node counts, 0-4 mm
indentation depths, flat and curved elastomers, one grasped object touching several links)
and stand in for them.

RNG: ``numpy.random.default_rng(SeedSequence([20295, cfg, stream, seed]))`` with
stream 0 = weights, 2 = indenters/poses.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

IND_NONE, IND_SPHERE, IND_BOX, IND_CAPSULE = 0, 1, 2, 3

#: mirrors ``etac_indenter`` in include/etac.h (48 bytes)
INDENTER_DTYPE = np.dtype(
    [("type", "<i4"), ("param", "<f4", (3,)), ("pose", "<f4", (7,)), ("skip_patch1", "<i4")]
)
assert INDENTER_DTYPE.itemsize == 48

FAR_AWAY = 1.0e4  # mm; where non-contacting patches / unused objects are parked


def _rng(cfg: int, stream: int, seed: int = 0) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([20295, cfg, stream, seed]))


# --------------------------------------------------------------------------------------
# small geometry helpers (placement only)
# --------------------------------------------------------------------------------------
def _unit(v):
    v = np.asarray(v, dtype=np.float64)
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def random_unit_vectors(rng, n):
    return _unit(rng.normal(size=(n, 3)))


def frame_from_z(z, roll):
    """Right-handed orthonormal frames [..., 3, 3] (columns x, y, z) whose z column is ``z``,
    rotated about z by ``roll``."""
    z = _unit(z)
    helper = np.where(np.abs(z[..., 2:3]) < 0.9, np.array([0.0, 0.0, 1.0]), np.array([1.0, 0.0, 0.0]))
    x0 = _unit(np.cross(helper, z))
    y0 = np.cross(z, x0)
    c, s = np.cos(roll)[..., None], np.sin(roll)[..., None]
    x = c * x0 + s * y0
    y = -s * x0 + c * y0
    return np.stack([x, y, z], axis=-1)


def quat_from_matrix(R):
    """Rotation matrices [..., 3, 3] -> unit quaternions [..., 4] in (x, y, z, w) order
    (Isaac-Gym order, include/etac.h).  Branch on the largest diagonal term for stability."""
    R = np.asarray(R, dtype=np.float64)
    m00, m11, m22 = R[..., 0, 0], R[..., 1, 1], R[..., 2, 2]
    tr = m00 + m11 + m22
    q = np.empty(R.shape[:-2] + (4,), dtype=np.float64)
    c0 = tr > 0
    c1 = (~c0) & (m00 >= m11) & (m00 >= m22)
    c2 = (~c0) & (~c1) & (m11 >= m22)
    c3 = ~(c0 | c1 | c2)
    with np.errstate(invalid="ignore"):
        s = np.sqrt(np.maximum(tr + 1.0, 1e-300)) * 2
        q0 = np.stack([(R[..., 2, 1] - R[..., 1, 2]) / s, (R[..., 0, 2] - R[..., 2, 0]) / s,
                       (R[..., 1, 0] - R[..., 0, 1]) / s, 0.25 * s], -1)
        s = np.sqrt(np.maximum(1.0 + m00 - m11 - m22, 1e-300)) * 2
        q1 = np.stack([0.25 * s, (R[..., 0, 1] + R[..., 1, 0]) / s, (R[..., 0, 2] + R[..., 2, 0]) / s,
                       (R[..., 2, 1] - R[..., 1, 2]) / s], -1)
        s = np.sqrt(np.maximum(1.0 + m11 - m00 - m22, 1e-300)) * 2
        q2 = np.stack([(R[..., 0, 1] + R[..., 1, 0]) / s, 0.25 * s, (R[..., 1, 2] + R[..., 2, 1]) / s,
                       (R[..., 0, 2] - R[..., 2, 0]) / s], -1)
        s = np.sqrt(np.maximum(1.0 + m22 - m00 - m11, 1e-300)) * 2
        q3 = np.stack([(R[..., 0, 2] + R[..., 2, 0]) / s, (R[..., 1, 2] + R[..., 2, 1]) / s, 0.25 * s,
                       (R[..., 1, 0] - R[..., 0, 1]) / s], -1)
    q[c0], q[c1], q[c2], q[c3] = q0[c0], q1[c1], q2[c2], q3[c3]
    return q / np.linalg.norm(q, axis=-1, keepdims=True)


def random_rotations(rng, n):
    z = random_unit_vectors(rng, n)
    return frame_from_z(z, rng.uniform(0, 2 * np.pi, n))


# --------------------------------------------------------------------------------------
# sensor meshes (node order == API order)
# --------------------------------------------------------------------------------------
@dataclass
class Mesh:
    pos: np.ndarray            # [N,3] fp32, undeformed, patch-local frame
    normal: np.ndarray         # [N,3] fp32, unit outward
    patch_offset: np.ndarray   # [P+1] int32
    adj_rowptr: np.ndarray | None = None   # CSR adjacency (optional)
    adj_col: np.ndarray | None = None

    @property
    def n_nodes(self):
        return int(self.pos.shape[0])

    @property
    def n_patches(self):
        return int(self.patch_offset.shape[0] - 1)


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def _grid_adjacency(g1, g2):
    idx = np.arange(g1 * g2).reshape(g1, g2)
    pairs = [np.stack([idx[:-1, :].ravel(), idx[1:, :].ravel()], 1),
             np.stack([idx[:, :-1].ravel(), idx[:, 1:].ravel()], 1)]
    e = np.concatenate(pairs, 0)
    return np.concatenate([e, e[:, ::-1]], 0)


def _csr_from_edges(n, edges):
    edges = np.unique(edges, axis=0)
    order = np.lexsort((edges[:, 1], edges[:, 0]))
    edges = edges[order]
    rowptr = np.zeros(n + 1, dtype=np.int32)
    np.add.at(rowptr, edges[:, 0] + 1, 1)
    rowptr = np.cumsum(rowptr).astype(np.int32)
    return rowptr, edges[:, 1].astype(np.int32)


def _knn_edges(pos, k):
    from scipy.spatial import cKDTree
    _, nb = cKDTree(pos).query(pos, k=k + 1)
    src = np.repeat(np.arange(pos.shape[0]), k)
    e = np.stack([src, nb[:, 1:].ravel()], 1)
    return np.concatenate([e, e[:, ::-1]], 0)


def flat_pad(g1, g2, spacing=1.0):
    """Flat pad, p=(ix*s, iy*s, 0), id = ix*g2+iy, n=+z, 4-neighbour adjacency."""
    ix, iy = np.meshgrid(np.arange(g1), np.arange(g2), indexing="ij")
    pos = np.stack([ix.ravel() * spacing, iy.ravel() * spacing, np.zeros(g1 * g2)], 1)
    nrm = np.tile([0.0, 0.0, 1.0], (g1 * g2, 1))
    return pos, nrm, _grid_adjacency(g1, g2)


def fib_cap(R, n):
    """Hemispherical cap: Fibonacci lattice z_k = 1-(k+1/2)/n, theta_k = k*pi*(3-sqrt 5)."""
    k = np.arange(n)
    z = 1.0 - (k + 0.5) / n
    th = k * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(1.0 - z * z)
    nrm = np.stack([s * np.cos(th), s * np.sin(th), z], 1)
    return R * nrm, nrm, _knn_edges(R * nrm, 6)


def half_cylinder(r, length, n_arc, n_ax):
    """Half cylinder, axis along local y; theta=(k+1/2)pi/n_arc - pi/2; radial normals."""
    th = (np.arange(n_arc) + 0.5) * math.pi / n_arc - math.pi / 2
    ax = (np.arange(n_ax) + 0.5) * length / n_ax
    T, A = np.meshgrid(th, ax, indexing="ij")
    nrm = np.stack([np.sin(T).ravel(), np.zeros(T.size), np.cos(T).ravel()], 1)
    pos = r * nrm + np.stack([np.zeros(T.size), A.ravel(), np.zeros(T.size)], 1)
    return pos, nrm, _grid_adjacency(n_arc, n_ax)


def cyl_sheet(r, arc_rad, n_arc, n_ax, ax_spacing=1.0):
    """Cylindrical section: n_arc samples over arc_rad (centred), n_ax axial samples."""
    th = (np.arange(n_arc) + 0.5) * arc_rad / n_arc - arc_rad / 2
    ax = (np.arange(n_ax) + 0.5) * ax_spacing
    T, A = np.meshgrid(th, ax, indexing="ij")
    nrm = np.stack([np.sin(T).ravel(), np.zeros(T.size), np.cos(T).ravel()], 1)
    pos = r * nrm + np.stack([np.zeros(T.size), A.ravel(), np.zeros(T.size)], 1)
    return pos, nrm, _grid_adjacency(n_arc, n_ax)


def assemble(patches) -> Mesh:
    """Concatenate per-patch (pos, normal, edges) into one Mesh with contiguous patches."""
    off = [0]
    P, Nn, E = [], [], []
    for pos, nrm, edges in patches:
        P.append(pos)
        Nn.append(nrm)
        E.append(edges + off[-1])
        off.append(off[-1] + pos.shape[0])
    n = off[-1]
    rowptr, col = _csr_from_edges(n, np.concatenate(E, 0))
    return Mesh(_f32(np.concatenate(P, 0)), _f32(np.concatenate(Nn, 0)),
                np.asarray(off, dtype=np.int32), rowptr, col)


def hand_mesh() -> Mesh:
    """Config 3 sensor set: 5 fingertip caps (R=9, 512 nodes) + 10 phalanx half-cylinders
    (r=8, len 25, 16x16) + palm 24x24 at 2 mm.  N = 5696, 16 patches, each in its own frame."""
    patches = [fib_cap(9.0, 512) for _ in range(5)]
    patches += [half_cylinder(8.0, 25.0, 16, 16) for _ in range(10)]
    patches += [flat_pad(24, 24, 2.0)]
    return assemble(patches)


# --------------------------------------------------------------------------------------
# residual MLP weights
# --------------------------------------------------------------------------------------
def make_weights(cfg: int, seed: int = 0, hidden: int = 64, std: float = 0.02):
    """W1[h,9] b1[h] W2[h,h] b2[h] W3[3,h] b3[3], i.i.d. N(0,std^2) drawn in fp64 -> fp32."""
    rng = _rng(cfg, 0, seed)
    shp = {"W1": (hidden, 9), "b1": (hidden,), "W2": (hidden, hidden), "b2": (hidden,),
           "W3": (3, hidden), "b3": (3,)}
    return {k: _f32(rng.normal(0.0, std, size=s)) for k, s in shp.items()}


def make_pointnet_weights(cfg: int, seed: int = 0, std: float = 0.1):
    """Weights of the paper's PointNet form of Phi with this repo's reading of
    the widths: E1[64,9] e1 E2[64,64] e2 | G1[64,64] g1 | D1[64,128] d1 D2[3,64] d2; N(0,std^2)."""
    rng = _rng(cfg, 3, seed)
    shp = {"E1": (64, 9), "e1": (64,), "E2": (64, 64), "e2": (64,), "G1": (64, 64), "g1": (64,),
           "D1": (64, 128), "d1": (64,), "D2": (3, 64), "d2": (3,)}
    return {k: _f32(rng.normal(0.0, std, size=s)) for k, s in shp.items()}


# --------------------------------------------------------------------------------------
# closed triangle meshes of objects (inputs of etac_mesh_to_sdf_grid; geometry only)
# --------------------------------------------------------------------------------------
def box_mesh(hx, hy, hz):
    """Axis-aligned box with half extents (hx, hy, hz): 8 vertices, 12 outward-oriented triangles."""
    v = np.array([[sx * hx, sy * hy, sz * hz] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)], np.float64)
    quads = [(0, 1, 3, 2), (4, 6, 7, 5), (0, 4, 5, 1), (2, 3, 7, 6), (0, 2, 6, 4), (1, 5, 7, 3)]
    t = [tri for a, b, c, d in quads for tri in ((a, b, c), (a, c, d))]
    return v, np.asarray(t, np.int32)


def tetra_mesh(scale=1.0):
    """Regular tetrahedron centred at the origin, outward-oriented."""
    v = scale * np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], np.float64)
    t = np.array([[0, 1, 2], [0, 3, 1], [0, 2, 3], [1, 3, 2]], np.int32)
    return v, t


def icosphere(radius, subdivisions):
    """Icosahedron subdivided `subdivisions` times, vertices on the sphere of `radius` (20 * 4^s triangles)."""
    g = (1.0 + math.sqrt(5.0)) / 2.0
    v = [(-1, g, 0), (1, g, 0), (-1, -g, 0), (1, -g, 0), (0, -1, g), (0, 1, g), (0, -1, -g), (0, 1, -g),
         (g, 0, -1), (g, 0, 1), (-g, 0, -1), (-g, 0, 1)]
    v = [np.asarray(x, np.float64) / np.linalg.norm(x) for x in v]
    t = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2), (10, 7, 6),
         (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7),
         (9, 8, 1)]
    for _ in range(subdivisions):
        mid, t2 = {}, []

        def m(i, j):
            key = (min(i, j), max(i, j))
            if key not in mid:
                x = v[i] + v[j]
                v.append(x / np.linalg.norm(x))
                mid[key] = len(v) - 1
            return mid[key]
        for a, b, c in t:
            ab, bc, ca = m(a, b), m(b, c), m(c, a)
            t2 += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        t = t2
    return radius * np.asarray(v), np.asarray(t, np.int32)


# --------------------------------------------------------------------------------------
# workload container
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    mesh: Mesh
    alpha: np.ndarray                 # [1] or [P] fp32, 1/mm
    weights: dict
    n_envs: int
    max_indenters: int
    indenters: np.ndarray             # [E, M] INDENTER_DTYPE
    patch_pose: np.ndarray | None     # [E, P, 7] fp32 or None (= identity)
    precision: str                    # "fp32" | "bf16"
    meta: dict = field(default_factory=dict)


def _blank_indenters(E, M):
    ind = np.zeros((E, M), dtype=INDENTER_DTYPE)
    ind["pose"][..., 6] = 1.0
    ind["pose"][..., 0:3] = FAR_AWAY
    return ind


def _press_on_node(mesh_pos, mesh_nrm, c, shape, size, depth, roll):
    """Pose (centre, quaternion) of an indenter pressed ``depth`` into node ``c`` along the
    node normal: its lowest surface point sits at p_c - depth*n_c, local z parallel to n_c.
    ``size`` = distance from the indenter centre to that surface point (sphere/capsule
    radius, box half-height)."""
    p, n = mesh_pos[c].astype(np.float64), mesh_nrm[c].astype(np.float64)
    centre = p + n * (size - depth)[:, None]
    q = quat_from_matrix(frame_from_z(n, roll))
    return centre, q


def config1(seed: int = 0, n_envs: int = 1) -> Workload:
    """1 env, flat 16x16 pad (1 mm), one sphere r=3 at seeded xy, penetration U(0,1) mm; fp32."""
    pos, nrm, edges = flat_pad(16, 16, 1.0)
    mesh = assemble([(pos, nrm, edges)])
    rng = _rng(1, 2, seed)
    ind = _blank_indenters(n_envs, 1)
    xy = rng.uniform(3.0, 12.0, size=(n_envs, 2))
    d = rng.uniform(0.0, 1.0, size=n_envs)
    ind["type"][:, 0] = IND_SPHERE
    ind["param"][:, 0, 0] = 3.0
    ind["pose"][:, 0, 0:2] = xy
    ind["pose"][:, 0, 2] = 3.0 - d
    ind["pose"][:, 0, 3:7] = [0, 0, 0, 1]
    return Workload("cfg1_flat_pad_16x16", mesh, _f32([0.5]), make_weights(1, seed), n_envs, 1,
                    ind, None, "fp32", {"depth": d})


def config2(seed: int = 0, n_envs: int = 64) -> Workload:
    """64 envs, hemispherical cap R=10, N=1024; 1-3 indenters (sphere r 2-6 / box side 4-10),
    depth U(0,1.5); fp32."""
    mesh = assemble([fib_cap(10.0, 1024)])
    rng = _rng(2, 2, seed)
    E, M = n_envs, 3
    ind = _blank_indenters(E, M)
    cand = np.nonzero(mesh.normal[:, 2] > 0.15)[0]
    m_cnt = rng.integers(1, 4, size=E)
    for k in range(M):
        use = m_cnt > k
        c = rng.choice(cand, size=E)
        is_box = rng.random(E) < 0.5
        r = rng.uniform(2.0, 6.0, E)
        h = rng.uniform(4.0, 10.0, E) / 2
        d = rng.uniform(0.0, 1.5, E)
        roll = rng.uniform(0, 2 * np.pi, E)
        size = np.where(is_box, h, r)
        centre, q = _press_on_node(mesh.pos, mesh.normal, c, None, size, d, roll)
        ind["type"][:, k] = np.where(use, np.where(is_box, IND_BOX, IND_SPHERE), IND_NONE)
        ind["param"][:, k, :] = np.where(is_box[:, None], h[:, None] * np.ones(3), np.stack([r, 0 * r, 0 * r], 1))
        ind["pose"][use, k, 0:3] = centre[use]
        ind["pose"][use, k, 3:7] = q[use]
    return Workload("cfg2_fingertip_cap_1024", mesh, _f32([0.5]), make_weights(2, seed), E, M,
                    ind, None, "fp32", {"n_indenters": m_cnt})


def _object_surface_points(rng, otype, param, n):
    """Random surface point s and outward unit normal m (object frame) for each of n objects.
    otype: IND_*; param [n,3] as in etac_indenter."""
    s = np.zeros((n, 3))
    m = np.zeros((n, 3))
    u = random_unit_vectors(rng, n)
    # sphere
    sp = otype == IND_SPHERE
    s[sp] = u[sp] * param[sp, 0:1]
    m[sp] = u[sp]
    # box: face chosen with probability proportional to its area, uniform point kept away
    # from the rim by 10 % so the contact is a face contact
    bx = np.nonzero(otype == IND_BOX)[0]
    if bx.size:
        h = param[bx]
        area = np.stack([h[:, 1] * h[:, 2], h[:, 0] * h[:, 2], h[:, 0] * h[:, 1]], 1)
        cdf = np.cumsum(area / area.sum(1, keepdims=True), 1)
        ax = (rng.random(bx.size)[:, None] > cdf).sum(1).clip(0, 2)
        sign = rng.choice([-1.0, 1.0], size=bx.size)
        pt = rng.uniform(-0.9, 0.9, size=(bx.size, 3)) * h
        pt[np.arange(bx.size), ax] = sign * h[np.arange(bx.size), ax]
        nm = np.zeros((bx.size, 3))
        nm[np.arange(bx.size), ax] = sign
        s[bx], m[bx] = pt, nm
    # capsule (axis = local z, radius param0, half length param1): side or caps by area
    cp = np.nonzero(otype == IND_CAPSULE)[0]
    if cp.size:
        r, L = param[cp, 0], param[cp, 1]
        side = rng.random(cp.size) < (2 * L) / (2 * L + 2 * r)
        uu = u[cp].copy()
        uside = uu.copy()
        uside[:, 2] = 0
        uside = _unit(uside + 1e-12)
        t = rng.uniform(-1, 1, cp.size) * L
        pt_side = np.stack([r * uside[:, 0], r * uside[:, 1], t], 1)
        cz = np.where(uu[:, 2] >= 0, L, -L)
        pt_cap = uu * r[:, None] + np.stack([0 * cz, 0 * cz, cz], 1)
        s[cp] = np.where(side[:, None], pt_side, pt_cap)
        m[cp] = np.where(side[:, None], uside, uu)
    return s, m


def config3(seed: int = 0, n_envs: int = 4096) -> Workload:
    """Dexterous-hand sensor set (N=5696, 16 patches, block-diagonal K); per env ONE object
    (sphere / box / capsule, 20-60 mm) at the world origin with a random rotation, touched by
    2-8 patches posed onto its surface (``patch_pose`` [E,16,7]); bf16 GEMM, fp32 accumulate."""
    mesh = hand_mesh()
    rng = _rng(3, 2, seed)
    E, P = n_envs, mesh.n_patches
    off = mesh.patch_offset
    ind = _blank_indenters(E, 1)
    otype = rng.integers(1, 4, size=E)
    param = np.zeros((E, 3))
    param[:, 0] = rng.uniform(20, 60, E) / 2                      # sphere radius
    box = otype == IND_BOX
    param[box] = rng.uniform(20, 60, size=(int(box.sum()), 3)) / 2
    cap = otype == IND_CAPSULE
    rc = rng.uniform(20, 40, int(cap.sum())) / 2
    tot = rng.uniform(2 * rc, 60.0)                               # total length <= 60
    param[cap, 0], param[cap, 1], param[cap, 2] = rc, (tot - 2 * rc) / 2, 0.0
    Robj = random_rotations(rng, E)
    ind["type"][:, 0] = otype
    ind["param"][:, 0, :] = param
    ind["pose"][:, 0, 0:3] = 0.0
    ind["pose"][:, 0, 3:7] = quat_from_matrix(Robj)

    n_c = rng.integers(2, 9, size=E)
    # choose n_c distinct patches per env: rank of a random key
    key = rng.random((E, P))
    chosen = key.argsort(1).argsort(1) < n_c[:, None]
    pose = np.zeros((E, P, 7))
    pose[..., 6] = 1.0
    # parked far away, each patch at a different spot
    pose[..., 0] = FAR_AWAY + 100.0 * np.arange(P)[None, :]
    pose[..., 1] = FAR_AWAY
    depth_all = np.zeros((E, P))
    for p in range(P):
        sel = np.nonzero(chosen[:, p])[0]
        if sel.size == 0:
            continue
        c = rng.integers(off[p], off[p + 1], size=sel.size)
        s_o, m_o = _object_surface_points(rng, otype[sel], param[sel], sel.size)
        s = np.einsum("nij,nj->ni", Robj[sel], s_o)
        m = np.einsum("nij,nj->ni", Robj[sel], m_o)
        d = rng.uniform(0.0, 1.5, sel.size)
        roll = rng.uniform(0, 2 * np.pi, sel.size)
        A = frame_from_z(mesh.normal[c].astype(np.float64), np.zeros(sel.size))   # local frame, z = n_c
        B = frame_from_z(-m, roll)                                                # world frame, z = -m
        Rp = np.einsum("nij,nkj->nik", B, A)                                      # B A^T
        t = (s - d[:, None] * m) - np.einsum("nij,nj->ni", Rp, mesh.pos[c].astype(np.float64))
        pose[sel, p, 0:3] = t
        pose[sel, p, 3:7] = quat_from_matrix(Rp)
        depth_all[sel, p] = d
    return Workload("cfg3_dexterous_hand_5696", mesh, _f32([0.5]), make_weights(3, seed), E, 1,
                    ind, _f32(pose), "bf16", {"chosen": chosen, "n_c": n_c, "depth": depth_all})


def _sheet_indenters(rng, mesh, E, M_max, frac_lo, frac_hi, sheet_R, node_area, shapes):
    """Press up to M_max indenters per env so the summed contact area is roughly
    f*N*node_area with f~U(frac_lo, frac_hi) (closed-form second-order contact-patch area on
    a surface of curvature 1/sheet_R along the arc; flat if sheet_R is inf).  Depth capped at
    4 mm; if the cap binds the indenter is enlarged instead."""
    N = mesh.n_nodes
    ind = _blank_indenters(E, M_max)
    m_cnt = rng.integers(1, M_max + 1, size=E)
    f = rng.uniform(frac_lo, frac_hi, size=E)
    area = f * N * node_area / m_cnt
    kappa = 0.0 if not np.isfinite(sheet_R) else 1.0 / sheet_R
    for k in range(M_max):
        use = m_cnt > k
        c = rng.integers(0, N, size=E)
        shape = rng.choice(shapes, size=E)
        roll = rng.uniform(0, 2 * np.pi, E)
        r = rng.uniform(20.0, 120.0, E)
        # sphere / capsule end-on: ellipse area = 2*pi*d / sqrt((kappa+1/r)/r)
        d = area * np.sqrt((kappa + 1.0 / r) / r) / (2 * np.pi)
        bind = d > 4.0
        # enlarge r so that d == 4 gives the area: (kappa + 1/r)/r = (8 pi / area)^2 =: g,
        # a quadratic in x = 1/r : x^2 + kappa x - g = 0
        g = (8 * np.pi / area) ** 2
        x = (-kappa + np.sqrt(kappa * kappa + 4 * g)) / 2
        r = np.where(bind, 1.0 / x, r)
        d = np.where(bind, 4.0, d)
        is_box = shape == IND_BOX
        h = rng.uniform(20.0, 60.0, E) / 2
        if kappa > 0:
            # flat face on a convex arc: strip of width min(2h, 2 sqrt(2 R d)) times 2h
            w = np.minimum(area / (2 * h), 2 * h)
            d_box = np.minimum((w / 2) ** 2 * kappa / 2, 4.0)
        else:
            d_box = rng.uniform(0.05, 1.0, E)
            h = np.sqrt(area) / 2
        is_cap = shape == IND_CAPSULE
        cap_L = np.where(is_cap, rng.uniform(0.0, 10.0, E), 0.0)       # end-on capsule: tip at r + L
        size = np.where(is_box, h, r + cap_L)
        depth = np.where(is_box, d_box, d)
        centre, q = _press_on_node(mesh.pos, mesh.normal, c, None, size, depth, roll)
        ind["type"][:, k] = np.where(use, shape, IND_NONE)
        prm = np.stack([r, np.zeros(E), np.zeros(E)], 1)
        prm = np.where(is_cap[:, None], np.stack([r, cap_L, np.zeros(E)], 1), prm)
        prm = np.where(is_box[:, None], h[:, None] * np.ones(3), prm)
        ind["param"][:, k, :] = prm
        ind["pose"][use, k, 0:3] = centre[use]
        ind["pose"][use, k, 3:7] = q[use]
    return ind, {"n_indenters": m_cnt, "target_frac": f}


def config4(seed: int = 0, n_envs: int = 4096) -> Workload:
    """Large curved sheet N=8192 (cylindrical section r=40, 90 deg: 64 arc x 128 axial), one
    dense K[8192x8192]; 1-5 indenters per env aimed at 5-20 % of nodes in contact; bf16."""
    mesh = assemble([cyl_sheet(40.0, math.pi / 2, 64, 128, 1.0)])
    rng = _rng(4, 2, seed)
    node_area = (40.0 * (math.pi / 2) / 64) * 1.0
    ind, meta = _sheet_indenters(rng, mesh, n_envs, 5, 0.05, 0.20, 40.0, node_area,
                                 [IND_SPHERE, IND_BOX, IND_CAPSULE])
    return Workload("cfg4_curved_sheet_8192", mesh, _f32([0.5]), make_weights(4, seed), n_envs, 5,
                    ind, None, "bf16", meta)


CFG5_GRIDS = {256: (16, 16), 1024: (32, 32), 4096: (64, 64), 8192: (64, 128)}


def config5(n_envs: int, n_nodes: int, curved: bool, frac: float, precision: str, seed: int = 0) -> Workload:
    """Sweep point: flat G1xG2 pad at 1 mm or the cfg-4 style cylinder on the same grid; one
    sphere per env sized for a contact fraction ``frac``."""
    g1, g2 = CFG5_GRIDS[n_nodes]
    if curved:
        R = 40.0
        arc = g1 * 1.0 / R
        mesh = assemble([cyl_sheet(R, arc, g1, g2, 1.0)])
    else:
        R = math.inf
        mesh = assemble([flat_pad(g1, g2, 1.0)])
    rng = _rng(5, 2, seed + 7919 * (n_nodes + (1 if curved else 0)) + int(frac * 1000))
    ind, meta = _sheet_indenters(rng, mesh, n_envs, 1, frac, frac, R, 1.0, [IND_SPHERE])
    meta["curved"] = curved
    return Workload(f"cfg5_N{n_nodes}_{'curved' if curved else 'flat'}_f{frac}", mesh, _f32([0.5]),
                    make_weights(5, seed), n_envs, 1, ind, None, precision, meta)


def get_config(cfg: int, seed: int = 0, n_envs: int | None = None) -> Workload:
    if cfg == 1:
        return config1(seed, n_envs or 1)
    if cfg == 2:
        return config2(seed, n_envs or 64)
    if cfg == 3:
        return config3(seed, n_envs or 4096)
    if cfg == 4:
        return config4(seed, n_envs or 4096)
    raise ValueError(f"unknown config {cfg}")


def shard_envs(n_envs: int, world_size: int, rank: int):
    """Contiguous env range [lo, hi) owned by ``rank`` (environments are the
    independent units; no collective on the data path)."""
    base, rem = divmod(n_envs, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
