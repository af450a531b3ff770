"""CPU oracle for the ETac tactile hot path  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It shares no code with the CUDA path
under ``paper_2604_20295_b200/csrc`` and never imports the package's binding.

What it computes (plain numpy, float64, in the paper's order and notation):

  O0  K_p[i,j] = exp(-alpha_p * ||p_j - p_i||_2)  for i,j in the same patch p, 0 across
      patches                                       PAPER.md:L83-L87, Eq. (1), Omega
  O1  contact detection: phi = min_k sdf_k(x_i), active <=> phi < 0, penalty displacement
      u_hat_i = -delta_i n_i with delta_i = max(0,-phi)   PAPER.md:L77 (+ DESIGN.md R5)
  O3  decay-based linear propagation  u_lin = Omega U_a
  O4  residual correction Phi and mask M_p, U_p = Omega U_a + Phi_p   PAPER.md:L91-L102, Eq. (2)

Readings of silent points (alpha, penalty formula, zero-contact gating, per-node MLP form
of Phi, ...) are listed in DESIGN.md §3 (R1..R20); each function cites the one it uses.

Pins (tests/test_oracle_pins.py, ``-m "not gpu"``): closed-form single-point-contact decay,
lattice row sums, brute-force triple loops, scipy cdist / torch float64 library
cross-checks, linearity, rigid invariance, SDF spot values, hand-derived worked examples
under tests/golden/; the sampled-grid SDF against scipy's RegularGridInterpolator, exactness
on affine fields and the h^2 interpolation bound on a sphere.  Unpinned: numerical agreement with the paper's *trained* Phi and its
Table II (no weights / FEM data exist here)  -> "parity unpinned" for that item only; and
the PointNet form of Phi is pinned only by its structural invariants (hidden widths are not
given in the paper: Fig. 3 is an image).  The backward pass (calibration gradients of Eq. 3)
is in etac_oracle_grad.py, pinned by finite differences of this module.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

IND_NONE, IND_SPHERE, IND_BOX, IND_CAPSULE, IND_GRID = 0, 1, 2, 3, 4


@dataclass
class OracleModel:
    pos: np.ndarray               # [N,3] fp32-rounded inputs, promoted on use (P)
    normal: np.ndarray            # [N,3]  (N in the paper)
    patch_offset: np.ndarray      # [P+1]
    alpha: np.ndarray             # [1] or [P]  (Eq. 1, learnable alpha; value = reading R1)
    weights: dict | None = None   # per-node MLP: W1 b1 W2 b2 W3 b3 (reading R10); None = no residual
    resid_arch: str = "pernode"   # "none" | "pernode" | "pointnet"
    active_mode: str = "passthrough"   # "passthrough" (mask M_p) | "propagate"
    ablation: str = "full"        # Table II rows: "full" | "residual_only" | "linear_only";
                                  # "no_propagation": U = U_hat, penalty displacement of the contact nodes only
    grids: dict = field(default_factory=dict)   # id -> (values [nz,ny,nx] fp32, origin [3], spacing): sampled SDFs
    _K: dict = field(default_factory=dict)

    @property
    def n_nodes(self):
        return int(self.pos.shape[0])

    @property
    def n_patches(self):
        return int(len(self.patch_offset) - 1)

    def alpha_of(self, p):
        a = np.asarray(self.alpha, dtype=np.float64).ravel()
        return float(a[p] if a.size > 1 else a[0])


# ------------------------------------------------------------------ O0: Eq. (1)
def kernel_block(model: OracleModel, p: int) -> np.ndarray:
    """Omega restricted to patch p: K_p[i,j] = exp(-alpha ||p_j - p_i||_2).
    Euclidean chord distance on UNDEFORMED positions (reading R2)."""
    if p not in model._K:
        lo, hi = int(model.patch_offset[p]), int(model.patch_offset[p + 1])
        P = model.pos[lo:hi].astype(np.float64)
        d2 = np.zeros((hi - lo, hi - lo))
        for c in range(3):
            diff = P[:, None, c] - P[None, :, c]
            d2 += diff * diff
        dist = np.sqrt(d2)
        model._K[p] = np.exp(-model.alpha_of(p) * dist)
    return model._K[p]


# ------------------------------------------------------------------ O1: contact detection
def quat_to_rot(q, dt=np.float64):
    """Unit quaternion (x,y,z,w) -> 3x3 rotation, textbook formula.  The evaluation order is
    the one DESIGN.md §5 fixes for the fp32 decision twin: products first, then
    R00 = 1 - 2*(yy+zz), R01 = 2*(xy - wz), ... every operation individually rounded."""
    x, y, z, w = (dt(q[0]), dt(q[1]), dt(q[2]), dt(q[3]))
    one, two = dt(1.0), dt(2.0)
    xx, yy, zz = x * x, y * y, z * z
    xy, xz, yz = x * y, x * z, y * z
    wx, wy, wz = w * x, w * y, w * z
    return np.array([
        [one - two * (yy + zz), two * (xy - wz), two * (xz + wy)],
        [two * (xy + wz), one - two * (xx + zz), two * (yz - wx)],
        [two * (xz - wy), two * (yz + wx), one - two * (xx + yy)],
    ], dtype=dt)


def sdf_local(itype, param, y0, y1, y2, dt=np.float64):
    """Exact signed distance of the three analytic indenters in the indenter's local frame
    (DESIGN.md §3 R6; textbook closed forms).  y* are arrays; param = etac_indenter.param."""
    if itype == IND_SPHERE:
        return np.sqrt((y0 * y0 + y1 * y1) + y2 * y2) - dt(param[0])
    if itype == IND_BOX:
        zero = dt(0.0)
        q0 = np.abs(y0) - dt(param[0])
        q1 = np.abs(y1) - dt(param[1])
        q2 = np.abs(y2) - dt(param[2])
        o0, o1, o2 = np.maximum(q0, zero), np.maximum(q1, zero), np.maximum(q2, zero)
        outside = np.sqrt((o0 * o0 + o1 * o1) + o2 * o2)
        inside = np.minimum(np.maximum(np.maximum(q0, q1), q2), zero)
        return outside + inside
    if itype == IND_CAPSULE:
        L = dt(param[1])
        cz = np.minimum(np.maximum(y2, -L), L)
        dz = y2 - cz
        return np.sqrt((y0 * y0 + y1 * y1) + dz * dz) - dt(param[0])
    raise ValueError(f"bad indenter type {itype}")


def sdf_grid(values, origin, spacing, y0, y1, y2, dt=np.float64):
    """Signed distance of a SAMPLED object (PAPER.md:L77 detects contact with SDFs against
    object meshes; a sampled grid is how such an SDF is handed over; R21).
    values[iz, iy, ix] = SDF sample at origin + spacing*(ix, iy, iz).  Definition: clamp the
    query point to the grid's box, interpolate the samples TRILINEARLY there (x, then y, then
    z; lerp written a + f*(b - a)), and add the Euclidean distance from the point to the box.
    Every operation is rounded to ``dt`` (fp32 twin: no fused multiply-add)."""
    v = np.asarray(values)
    nz, ny, nx = v.shape
    h, inv_h = dt(spacing), dt(1.0) / dt(spacing)
    y = [np.asarray(y0, dtype=dt), np.asarray(y1, dtype=dt), np.asarray(y2, dtype=dt)]
    n = [nx, ny, nz]
    yc, idx, fr = [], [], []
    for a in range(3):
        lo = dt(origin[a])
        hi = lo + h * dt(n[a] - 1)
        c = np.minimum(np.maximum(y[a], lo), hi)
        t = (c - lo) * inv_h
        i = np.minimum(np.floor(t), dt(n[a] - 2)).astype(np.int64)
        yc.append(c), idx.append(i), fr.append(t - i.astype(dt))
    ix, iy, iz = idx
    fx, fy, fz = fr
    V = lambda dz, dy, dx: v[iz + dz, iy + dy, ix + dx].astype(dt)
    lerp = lambda a, b, f: a + f * (b - a)
    c00, c10 = lerp(V(0, 0, 0), V(0, 0, 1), fx), lerp(V(0, 1, 0), V(0, 1, 1), fx)
    c01, c11 = lerp(V(1, 0, 0), V(1, 0, 1), fx), lerp(V(1, 1, 0), V(1, 1, 1), fx)
    c = lerp(lerp(c00, c10, fy), lerp(c01, c11, fy), fz)
    d0, d1, d2 = y[0] - yc[0], y[1] - yc[1], y[2] - yc[2]
    return c + np.sqrt((d0 * d0 + d1 * d1) + d2 * d2)


def signed_distance(model: OracleModel, indenters_e, patch_pose_e=None, dt=np.float64):
    """phi[i] = min over the env's indenters (type != NONE) of sdf_k(R_k^T (x_i - t_k)),
    x_i = R(q_{e,p}) p_i + t_{e,p} (identity if no patch poses); +inf if no indenter.
    Self-contact: an indenter with skip_patch1 = p + 1 is the collision shape of the link
    patch p is mounted on and is left out of that patch's union (the other patches see it).
    PAPER.md:L77 'contact events are first detected using SDFs between nodes and objects';
    union of several indenters = min (reading R6).  ``dt=np.float32`` gives the fp32
    decision twin: same formulas, same order, every op rounded to fp32."""
    N = model.n_nodes
    pos = model.pos.astype(dt)
    X = np.empty((N, 3), dtype=dt)
    if patch_pose_e is None:
        X[:] = pos
    else:
        for p in range(model.n_patches):
            lo, hi = int(model.patch_offset[p]), int(model.patch_offset[p + 1])
            R = quat_to_rot(patch_pose_e[p, 3:7], dt)
            t = patch_pose_e[p, 0:3].astype(dt)
            pp = pos[lo:hi]
            for a in range(3):
                X[lo:hi, a] = ((R[a, 0] * pp[:, 0] + R[a, 1] * pp[:, 1]) + R[a, 2] * pp[:, 2]) + t[a]
    phi = np.full(N, np.inf, dtype=dt)
    for ind in indenters_e:
        itype = int(ind["type"])
        if itype == IND_NONE:
            continue
        R = quat_to_rot(ind["pose"][3:7], dt)
        t = ind["pose"][0:3].astype(dt)
        d0, d1, d2 = X[:, 0] - t[0], X[:, 1] - t[1], X[:, 2] - t[2]
        # y = R^T d
        y0 = (R[0, 0] * d0 + R[1, 0] * d1) + R[2, 0] * d2
        y1 = (R[0, 1] * d0 + R[1, 1] * d1) + R[2, 1] * d2
        y2 = (R[0, 2] * d0 + R[1, 2] * d1) + R[2, 2] * d2
        if itype == IND_GRID:
            values, origin, spacing = model.grids[int(ind["param"][0])]
            phi_k = sdf_grid(values, origin, spacing, y0, y1, y2, dt)
        else:
            phi_k = sdf_local(itype, ind["param"], y0, y1, y2, dt)
        skip = int(ind["skip_patch1"]) - 1 if "skip_patch1" in ind.dtype.names else -1
        if 0 <= skip < model.n_patches:
            lo, hi = int(model.patch_offset[skip]), int(model.patch_offset[skip + 1])
            phi_k = phi_k.copy()
            phi_k[lo:hi] = np.inf
        phi = np.minimum(phi, phi_k)
    return phi


# ------------------------------------------------------------------ O4: residual networks
def silu(x):
    return x / (1.0 + np.exp(-x))


def residual_pernode(w, ulin, pos, nrm):
    """BASELINE.json per-node form of Phi (reading R10/R11): input [u_lin(3), p(3), n(3)],
    9 -> 64 -> 64 -> 3 with SiLU; weights are Linear-layer style [out, in]."""
    x9 = np.concatenate([ulin, pos, nrm], axis=1)
    h1 = silu(x9 @ w["W1"].astype(np.float64).T + w["b1"].astype(np.float64))
    h2 = silu(h1 @ w["W2"].astype(np.float64).T + w["b2"].astype(np.float64))
    return h2 @ w["W3"].astype(np.float64).T + w["b3"].astype(np.float64)


def residual_pointnet(w, uhat, pos, nrm):
    """Paper form of Phi: n x 9 input [P, N, U_hat] -> shared MLP ->
    max-pool -> 64-d global feature -> MLP -> broadcast + concat (n x 128) -> shared-MLP
    decoder -> n x 3.  Hidden widths/activation are NOT given (Fig. 3 is an image): the
    widths 9->64->64 | 64->64 | 128->64->3 and SiLU are reading R10 ("parity unpinned")."""
    f64 = lambda k: w[k].astype(np.float64)
    x9 = np.concatenate([pos, nrm, uhat], axis=1)
    f = silu(x9 @ f64("E1").T + f64("e1"))
    f = silu(f @ f64("E2").T + f64("e2"))              # n x 64 point-wise features
    g = f.max(axis=0)                                   # 64-d global feature (max-pool)
    g = silu(g @ f64("G1").T + f64("g1"))               # "further encoded by another MLP"
    cat = np.concatenate([f, np.broadcast_to(g, f.shape)], axis=1)   # n x 128
    h = silu(cat @ f64("D1").T + f64("d1"))
    return h @ f64("D2").T + f64("d2")


# ------------------------------------------------------------------ the step
def step(model: OracleModel, indenters=None, patch_pose=None, penetration=None, envs=None):
    """One tactile update for the listed envs (default all).  Returns float64 arrays
    U [E',N,3], analytic [E',N,3] (unmasked K.U_hat on all rows), delta [E',N], and the
    decisions mask [E',N] (bool), contact [E',P] (bool), plus phi/delta of the fp32 twin.

    Mask decision precision: the active test phi < 0 is taken on the fp32 twin (the
    kernel's precision); delta's value is the float64 one."""
    if (indenters is None) == (penetration is None):
        raise ValueError("give exactly one of indenters / penetration")
    E_all = (indenters if indenters is not None else penetration).shape[0]
    envs = list(range(E_all)) if envs is None else list(envs)
    N, Pn = model.n_nodes, model.n_patches
    nrm = model.normal.astype(np.float64)
    pos = model.pos.astype(np.float64)
    out = {k: np.zeros((len(envs), N, 3)) for k in ("U", "analytic")}
    out["delta"] = np.zeros((len(envs), N))
    out["delta32"] = np.zeros((len(envs), N), dtype=np.float32)
    out["mask"] = np.zeros((len(envs), N), dtype=bool)
    out["contact"] = np.zeros((len(envs), Pn), dtype=bool)
    out["patch_offset"] = np.asarray(model.patch_offset)
    for oi, e in enumerate(envs):
        # ---- O1
        if indenters is not None:
            pp = None if patch_pose is None else patch_pose[e]
            phi64 = signed_distance(model, indenters[e], pp, np.float64)
            phi32 = signed_distance(model, indenters[e], pp, np.float32)
            active = phi32 < np.float32(0.0)                     # strict: phi == 0 is passive (R7)
            delta = np.where(active, np.maximum(0.0, -phi64), 0.0)
            out["delta32"][oi] = np.where(active, -phi32, np.float32(0.0))
        else:
            d_in = penetration[e]
            delta32 = np.maximum(np.float32(0.0), d_in.astype(np.float32))   # negatives clamp (R19)
            active = delta32 > 0
            delta = delta32.astype(np.float64)
            out["delta32"][oi] = delta32
        uhat = -delta[:, None] * nrm                              # penalty model, reading R5
        out["delta"][oi], out["mask"][oi] = delta, active
        for p in range(Pn):
            lo, hi = int(model.patch_offset[p]), int(model.patch_offset[p + 1])
            act = active[lo:hi]
            if not act.any():                                     # O2 + reading R8: gate per (env, patch)
                continue
            out["contact"][oi, p] = True
            K = kernel_block(model, p)
            # ---- O3: sum over ACTIVE j only (Omega U_a); includes j = i
            ulin = K[:, act] @ uhat[lo:hi][act]
            out["analytic"][oi, lo:hi] = ulin
            # ---- O4 (Eq. 2)
            if model.ablation == "no_propagation":                # nothing but the contact nodes moves
                out["U"][oi, lo:hi] = uhat[lo:hi]
                continue
            if model.resid_arch == "none" or model.ablation == "linear_only":   # "Linear Decay Only"
                r = 0.0
            elif model.resid_arch == "pernode":
                r = residual_pernode(model.weights, ulin, pos[lo:hi], nrm[lo:hi])
            elif model.resid_arch == "pointnet":
                r = residual_pointnet(model.weights, uhat[lo:hi], pos[lo:hi], nrm[lo:hi])
            else:
                raise ValueError(model.resid_arch)
            if model.ablation not in ("full", "residual_only", "linear_only"):
                raise ValueError(model.ablation)
            U = r + 0.0 * ulin if model.ablation == "residual_only" else ulin + r   # "Residual Network Only": U_p = Phi_p
            if model.active_mode == "passthrough":                # mask M_p, reading R4
                U = np.where(act[:, None], uhat[lo:hi], U)
            out["U"][oi, lo:hi] = U
    return out


def model_from_workload(wl, resid_arch="pernode", active_mode="passthrough") -> OracleModel:
    return OracleModel(wl.mesh.pos, wl.mesh.normal, wl.mesh.patch_offset, wl.alpha,
                       wl.weights, resid_arch, active_mode, grids=dict(wl.meta.get("grids", {})))
