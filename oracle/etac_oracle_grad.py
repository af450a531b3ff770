"""CPU oracle for the backward pass of the ETac tactile update  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Same rules as ``etac_oracle.py`` (only tests / smoke / bench baselines may import it; no code shared
with the CUDA path).  It differentiates exactly what ``etac_oracle.step`` computes:

  L(alpha, Phi) is any scalar function of U with G = dL/dU given (calibration, PAPER.md:L104-L108,
  Eq. (3): L = || U_p - U_p* ||_2 fitted by gradient descent; Table I lists differentiability).

  For a row i of a contacting (env, patch) that the mask of Eq. (2) does not overwrite with u^
      U_i = u_i + Phi(u_i, p_i, n_i),  u_i = sum_{j active} K_ij u^_j,  K_ij = exp(-alpha d_ij)   (Eq. 1-2)
      dK_ij / dalpha = -d_ij K_ij                       (d_ij = ||p_j - p_i||_2 from the positions)
      dL/dalpha = sum_i (G_i + J^T G_i) . sum_j dK_ij/dalpha u^_j ,   J = dPhi/du at row i
      dL/dW     = the chain rule through the per-node MLP 9 -> 64 -> 64 -> 3 (SiLU), written out
  Rows overwritten with u^ = -delta n (active rows, "passthrough") and rows of contact-free pairs do not
  depend on alpha or Phi.  dL/ddelta_j of the nodes in contact follows from u^_j = -delta_j n_j (PAPER.md:L77 +
  DESIGN.md R5): dL/ddelta_j = -n_j . (sum_i K_ij dL/du_i + G_j if row j is u^_j itself); 0 for the other nodes.
  The contact set is held fixed (it does not depend on alpha or Phi).

  PointNet form of Phi (the network Eq. (3) calibrates): its input is [P, N, U^], so Phi does
  not depend on alpha (dL/dalpha comes from u_i alone) and dL/ddelta_j gains -n_j . dL/du^_j through the encoder
  input of the nodes in contact.  The chain rule runs backwards through the decoder, the broadcast of the global
  feature (sum of the decoder-input gradients over the rows), the global MLP, the max-pool (the gradient of
  column k goes to the row that attains the maximum) and the shared encoder.

float64 numpy, one (env, patch) at a time, no fusion.  Pins (tests/test_oracle_pins.py): central
finite differences of ``etac_oracle.step`` (itself pinned) with respect to alpha, to sampled weights
of every layer and (penetration input mode) to the penetration of sampled contact nodes; ``pose_gradients``
(dL/ddelta chained to indenter and patch poses) by central differences of ``etac_oracle.step`` under translations
and small left rotations of the poses, for every indenter type.
"""
from __future__ import annotations

import numpy as np

from . import etac_oracle as O


def silu_prime(z):
    s = 1.0 / (1.0 + np.exp(-z))
    return s * (1.0 + z * (1.0 - s))


def backward(model: O.OracleModel, G, indenters=None, patch_pose=None, penetration=None, envs=None):
    """G: dL/dU [E', N, 3] for the listed envs (default all).  Returns float64 gradients
    {"alpha": [n_alpha], "delta": [E', N]} and, per residual form, "W1": [64, 9], "b1", "W2", "b2", "W3", "b3"
    (per-node) or "E1", "e1", "E2", "e2", "G1", "g1", "D1", "d1", "D2", "d2" (PointNet)."""
    if model.resid_arch not in ("none", "pernode", "pointnet") or model.ablation != "full":
        raise ValueError("backward oracle: full pipeline only")
    G = np.asarray(G, dtype=np.float64)
    fwd = O.step(model, indenters=indenters, patch_pose=patch_pose, penetration=penetration, envs=envs)
    alpha = np.atleast_1d(np.asarray(model.alpha, dtype=np.float64))
    grads = {"alpha": np.zeros(alpha.shape[0]), "delta": np.zeros((G.shape[0], model.n_nodes))}
    mlp = model.resid_arch == "pernode"
    pnet = model.resid_arch == "pointnet"
    if mlp or pnet:
        w = {k: np.asarray(v, dtype=np.float64) for k, v in model.weights.items()}
        names = ("W1", "b1", "W2", "b2", "W3", "b3") if mlp else ("E1", "e1", "E2", "e2", "G1", "g1", "D1", "d1", "D2", "d2")
        for k in names:
            grads[k] = np.zeros_like(w[k])
    pos = model.pos.astype(np.float64)
    nrm = model.normal.astype(np.float64)
    for oi in range(G.shape[0]):
        delta, active = fwd["delta"][oi], fwd["mask"][oi]
        uhat = -delta[:, None] * nrm
        for p in range(model.n_patches):
            lo, hi = int(model.patch_offset[p]), int(model.patch_offset[p + 1])
            act = active[lo:hi]
            if not act.any():
                continue
            K = O.kernel_block(model, p)
            P = pos[lo:hi]
            dist = np.sqrt(((P[:, None, :] - P[None, :, :]) ** 2).sum(-1))
            dK = -dist * K                                        # dK/dalpha, Eq. (1)
            ua = uhat[lo:hi][act]
            ulin = K[:, act] @ ua
            v = dK[:, act] @ ua
            rows = ~act if model.active_mode == "passthrough" else np.ones_like(act)
            g = np.where(rows[:, None], G[oi, lo:hi], 0.0)
            glin = g.copy()
            if mlp:
                x9 = np.concatenate([ulin, P, nrm[lo:hi]], axis=1)
                z1 = x9 @ w["W1"].T + w["b1"]
                h1 = O.silu(z1)
                z2 = h1 @ w["W2"].T + w["b2"]
                h2 = O.silu(z2)
                grads["W3"] += g.T @ h2
                grads["b3"] += g.sum(0)
                gz2 = (g @ w["W3"]) * silu_prime(z2)
                grads["W2"] += gz2.T @ h1
                grads["b2"] += gz2.sum(0)
                gz1 = (gz2 @ w["W2"]) * silu_prime(z1)
                grads["W1"] += gz1.T @ x9
                grads["b1"] += gz1.sum(0)
                glin += (gz1 @ w["W1"])[:, 0:3]
            guhat = 0.0                                           # dL/du^ through the input of Phi (PointNet only)
            if pnet:
                x9 = np.concatenate([P, nrm[lo:hi], uhat[lo:hi]], axis=1)     # [P, N, U^]
                z1 = x9 @ w["E1"].T + w["e1"]
                f1 = O.silu(z1)
                z2 = f1 @ w["E2"].T + w["e2"]
                f = O.silu(z2)                                    # n x 64 point-wise features
                arg = f.argmax(axis=0)                            # max-pool: the row that gives column k
                gmax = f[arg, np.arange(f.shape[1])]
                zg = gmax @ w["G1"].T + w["g1"]
                gp = O.silu(zg)                                   # global feature after its MLP
                cat = np.concatenate([f, np.broadcast_to(gp, f.shape)], axis=1)
                zc = cat @ w["D1"].T + w["d1"]
                h = O.silu(zc)
                grads["D2"] += g.T @ h
                grads["d2"] += g.sum(0)
                gzc = (g @ w["D2"]) * silu_prime(zc)
                grads["D1"] += gzc.T @ cat
                grads["d1"] += gzc.sum(0)
                gcat = gzc @ w["D1"]
                gf = gcat[:, :64].copy()
                ggp = gcat[:, 64:].sum(0)                         # the broadcast global feature collects every row
                gzg = ggp * silu_prime(zg)
                grads["G1"] += np.outer(gzg, gmax)
                grads["g1"] += gzg
                np.add.at(gf, (arg, np.arange(64)), gzg @ w["G1"])            # max-pool routes to the arg-max rows
                gz2 = gf * silu_prime(z2)
                grads["E2"] += gz2.T @ f1
                grads["e2"] += gz2.sum(0)
                gz1 = (gz2 @ w["E2"]) * silu_prime(z1)
                grads["E1"] += gz1.T @ x9
                grads["e1"] += gz1.sum(0)
                guhat = (gz1 @ w["E1"])[:, 6:9][act]
            grads["alpha"][p if alpha.shape[0] > 1 else 0] += float((glin * v).sum())
            # u^_j = -delta_j n_j: dL/ddelta_j = -n_j . (sum_i K_ij dL/du_i + G_j if row j is u^_j itself
            #                                            + dL/du^_j through the input of Phi)
            back = K[:, act].T @ glin + guhat
            if model.active_mode == "passthrough":
                back = back + G[oi, lo:hi][act]
            grads["delta"][oi, lo:hi][act] = -(nrm[lo:hi][act] * back).sum(1)
    return grads


# ------------------------------------------------------------------ dL/d(poses) from dL/ddelta
def sdf_local_gradient(itype, param, y):
    """Gradient [n, 3] of ``etac_oracle.sdf_local`` with respect to the local point y [n, 3] (closed forms):
    sphere y/|y|; box outside sign(y) max(q, 0)/|max(q, 0)|, q = |y| - b, inside the unit vector of the axis with the
    largest q, signed like y; capsule (y0, y1, y2 - clamp(y2, -L, L)) / |.|."""
    y = np.asarray(y, dtype=np.float64)
    if itype == O.IND_SPHERE:
        return y / np.linalg.norm(y, axis=1, keepdims=True)
    if itype == O.IND_BOX:
        b = np.asarray(param[:3], dtype=np.float64)
        q = np.abs(y) - b
        o = np.maximum(q, 0.0)
        no = np.linalg.norm(o, axis=1, keepdims=True)
        sgn = np.where(y < 0, -1.0, 1.0)
        with np.errstate(invalid="ignore", divide="ignore"):
            g_out = sgn * o / no
        g_in = np.zeros_like(y)
        a = q.argmax(axis=1)
        g_in[np.arange(y.shape[0]), a] = sgn[np.arange(y.shape[0]), a]
        return np.where(no > 0, g_out, g_in)
    if itype == O.IND_CAPSULE:
        L = float(param[1])
        v = y.copy()
        v[:, 2] = y[:, 2] - np.clip(y[:, 2], -L, L)
        return v / np.linalg.norm(v, axis=1, keepdims=True)
    raise ValueError(f"bad indenter type {itype}")


def sdf_grid_gradient(values, origin, spacing, y):
    """Gradient [n, 3] of ``etac_oracle.sdf_grid`` with respect to y [n, 3]: along an axis on which y lies inside the
    grid's box the derivative of the trilinear interpolant (difference of the two faces of the cell along that
    axis, interpolated bilinearly on the other two, over the spacing); along an axis on which y was clamped the
    interpolant is constant and the distance term gives (y - clamp(y)) / |y - clamp(y)|."""
    v = np.asarray(values, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    nz, ny, nx = v.shape
    n = np.array([nx, ny, nz])
    h = float(spacing)
    lo = np.asarray(origin, dtype=np.float64)
    hi = lo + h * (n - 1)
    yc = np.clip(y, lo, hi)
    t = (yc - lo) / h
    i = np.minimum(np.floor(t), n - 2).astype(np.int64)
    f = t - i
    g = np.zeros_like(y)
    for r in range(y.shape[0]):
        c = v[i[r, 2]:i[r, 2] + 2, i[r, 1]:i[r, 1] + 2, i[r, 0]:i[r, 0] + 2]      # [z, y, x] corner samples of the cell
        wx = np.array([1 - f[r, 0], f[r, 0]])
        wy = np.array([1 - f[r, 1], f[r, 1]])
        wz = np.array([1 - f[r, 2], f[r, 2]])
        dx = np.einsum("zy,z,y->", c[:, :, 1] - c[:, :, 0], wz, wy) / h
        dy = np.einsum("zx,z,x->", c[:, 1, :] - c[:, 0, :], wz, wx) / h
        dz = np.einsum("yx,y,x->", c[1, :, :] - c[0, :, :], wy, wx) / h
        inside = y[r] == yc[r]
        g[r] = np.where(inside, [dx, dy, dz], 0.0)
        off = y[r] - yc[r]
        dist = np.linalg.norm(off)
        if dist > 0:
            g[r] += off / dist
    return g


def pose_gradients(model: O.OracleModel, g_delta, indenters, patch_pose=None, envs=None):
    """Chains dL/ddelta [E', N] (``backward(...)["delta"]``) to the poses the penetration came from
    (delta from SDFs between nodes and objects; Table I: differentiability).

    For a node in contact  delta_i = -phi_k*(y),  y = R_k^T (x_i - t_k),  x_i = R_p p_i + t_p,  k* the indenter that
    attains the min of the union (the contact set and k* are held fixed).  With n_w = R_k grad phi_k(y) (the SDF's
    gradient in the world frame), d = x_i - t_k, r = x_i - t_p, and rotations perturbed on the LEFT in the world
    frame, R <- exp([theta]x) R:
        d delta/d t_k = +n_w          d delta/d theta_k = -(n_w x d)
        d delta/d t_p = -n_w          d delta/d theta_p = -(r x n_w)
    Returns float64 {"indenter": [E', max_ind, 6], "patch": [E', P, 6]}, each row (dL/dt, dL/dtheta); the patch part
    is zero if there are no patch poses."""
    g_delta = np.asarray(g_delta, dtype=np.float64)
    E_all = indenters.shape[0]
    envs = list(range(E_all)) if envs is None else list(envs)
    pos = model.pos.astype(np.float64)
    out = {"indenter": np.zeros((len(envs), indenters.shape[1], 6)), "patch": np.zeros((len(envs), model.n_patches, 6))}
    for oi, e in enumerate(envs):
        X = pos.copy()
        tp = np.zeros((model.n_patches, 3))
        if patch_pose is not None:
            for p in range(model.n_patches):
                lo, hi = int(model.patch_offset[p]), int(model.patch_offset[p + 1])
                tp[p] = np.asarray(patch_pose[e][p, 0:3], dtype=np.float64)
                X[lo:hi] = pos[lo:hi] @ O.quat_to_rot(patch_pose[e][p, 3:7]).T + tp[p]
        phi = np.full((indenters.shape[1], model.n_nodes), np.inf)
        grad_w = np.zeros((indenters.shape[1], model.n_nodes, 3))
        for k, ind in enumerate(indenters[e]):
            itype = int(ind["type"])
            if itype == O.IND_NONE:
                continue
            R = O.quat_to_rot(ind["pose"][3:7])
            y = (X - np.asarray(ind["pose"][0:3], dtype=np.float64)) @ R          # rows R^T d
            if itype == O.IND_GRID:
                values, origin, spacing = model.grids[int(ind["param"][0])]
                phi[k] = O.sdf_grid(values, origin, spacing, y[:, 0], y[:, 1], y[:, 2])
                gl = sdf_grid_gradient(values, origin, spacing, y)
            else:
                phi[k] = O.sdf_local(itype, ind["param"], y[:, 0], y[:, 1], y[:, 2])
                gl = sdf_local_gradient(itype, ind["param"], y)
            grad_w[k] = gl @ R.T
            skip = int(ind["skip_patch1"]) - 1 if "skip_patch1" in ind.dtype.names else -1
            if 0 <= skip < model.n_patches:
                phi[k, int(model.patch_offset[skip]):int(model.patch_offset[skip + 1])] = np.inf
        kstar = phi.argmin(axis=0)
        for p in range(model.n_patches):
            lo, hi = int(model.patch_offset[p]), int(model.patch_offset[p + 1])
            for i in range(lo, hi):
                g = g_delta[oi, i]
                if g == 0.0:
                    continue
                k = int(kstar[i])
                nw = grad_w[k, i]
                d = X[i] - np.asarray(indenters[e][k]["pose"][0:3], dtype=np.float64)
                r = X[i] - tp[p]
                out["indenter"][oi, k, 0:3] += g * nw
                out["indenter"][oi, k, 3:6] += -g * np.cross(nw, d)
                if patch_pose is not None:
                    out["patch"][oi, p, 0:3] += -g * nw
                    out["patch"][oi, p, 3:6] += -g * np.cross(r, nw)
    return out
