"""Shared helpers of the GPU parity tests: run a workload through the C ABI (via the thin
binding) and through the CPU oracle on the same seeded inputs, and compare element by element.

Tolerances (BASELINE.json north_star, written out in tests/test_parity_gpu.py):
  masks bit-exact; fp32 path max|u_gpu-u_ref| <= 1e-4*max|u_ref|; bf16 path <= 2e-2*max|u_ref|."""
import numpy as np

from oracle import etac_oracle as O
from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W

TOL = {"fp32": 1e-4, "bf16": 2e-2}


def run_gpu(wl, *, precision=None, path=T.ETAC_PATH_AUTO, resid=True, active_mode=T.ETAC_ACTIVE_PASSTHROUGH,
            penetration=None, max_envs=None, n_envs=None, steps=1, group_bytes=None):
    import torch
    n_envs = wl.n_envs if n_envs is None else n_envs
    eng = T.Etac(wl, precision=precision, resid=resid, active_mode=active_mode, debug_outputs=True,
                 max_envs=max_envs or max(n_envs, 1))
    try:
        T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, path)
        if group_bytes is not None:
            T.etac_set_option(eng.ctx, T.ETAC_OPT_L2_GROUP_BYTES, group_bytes)
        if penetration is not None:
            dev = eng.upload(penetration=penetration)
        else:
            dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        # poison the outputs: every element must be overwritten by the step
        eng.out.fill_(float("nan")), eng.analytic.fill_(float("nan")), eng.pen_out.fill_(float("nan"))
        eng.contact.fill_(77), eng.active_count.fill_(-5)
        for _ in range(steps):
            eng.step(n_envs, dev)
        torch.cuda.synchronize()
        res = {"U": eng.out[:n_envs].cpu().numpy(), "analytic": eng.analytic[:n_envs].cpu().numpy(),
               "delta": eng.pen_out[:n_envs].cpu().numpy(), "mask": eng.mask_bool(n_envs),
               "contact": eng.contact[:n_envs].cpu().numpy(), "active_count": eng.active_count[:n_envs].cpu().numpy(),
               "pairs": T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_CONTACT_PAIRS),
               "path": T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_PATH),
               "launches": T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_LAUNCHES)}
    finally:
        eng.close()
    return res


def run_oracle(wl, *, resid=True, active_mode="passthrough", penetration=None, envs=None):
    arch = "none" if not resid else ("pointnet" if "E1" in wl.weights else "pernode")
    m = O.model_from_workload(wl, resid_arch=arch, active_mode=active_mode)
    if penetration is not None:
        return O.step(m, penetration=penetration, envs=envs)
    return O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose, envs=envs)


def compare(gpu, ref, tol, envs=None, resid_tol=None, label="", delta_tol=1e-5):
    """gpu: dict from run_gpu (all envs); ref: oracle dict for `envs` (default all).
    delta_tol: fp32-vs-fp64 bound on delta relative to max(1, max delta); the fp32 evaluation of
    |y| - r loses ~ulp(r), so workloads with very large indenters pass a looser bound."""
    sel = slice(None) if envs is None else np.asarray(list(envs))
    U, A, D, M = gpu["U"][sel], gpu["analytic"][sel], gpu["delta"][sel], gpu["mask"][sel]
    assert np.isfinite(U).all() and np.isfinite(A).all() and np.isfinite(D).all(), f"{label}: unwritten output"
    # decisions: bit-exact (taken in fp32 on both sides)
    assert np.array_equal(M, ref["mask"]), f"{label}: mask differs at {np.argwhere(M != ref['mask'])[:5]}"
    assert np.array_equal(D, ref["delta32"]), f"{label}: delta not bit-exact vs the fp32 twin"
    # link-contact vector and active-node count: integer work, bit-exact
    assert np.array_equal(gpu["contact"][sel].astype(bool), ref["contact"]), f"{label}: contact vector differs"
    assert np.array_equal(gpu["active_count"][sel], ref["mask"].sum(1)), f"{label}: active-node count differs"
    scale_d = max(1.0, float(np.abs(ref["delta"]).max()))
    assert np.abs(D - ref["delta"]).max() <= delta_tol * scale_d
    umax = float(np.abs(ref["U"]).max())
    amax = float(np.abs(ref["analytic"]).max())
    err_u = float(np.abs(U - ref["U"]).max())
    err_a = float(np.abs(A - ref["analytic"]).max())
    stats = {"umax": umax, "err_u": err_u, "err_a": err_a, "rel_u": err_u / max(umax, 1e-30),
             "rel_a": err_a / max(amax, 1e-30)}
    assert err_u <= tol * umax, f"{label}: U err {err_u:.3e} > {tol}*{umax:.3e}"
    assert err_a <= tol * amax, f"{label}: analytic err {err_a:.3e} > {tol}*{amax:.3e}"
    # non-contacting (env, patch) pairs are exactly zero
    zero_rows = ~np.repeat(ref["contact"], np.diff(ref["patch_offset"]), axis=1) if "patch_offset" in ref else None
    if zero_rows is not None:
        assert np.all(U[zero_rows] == 0.0) and np.all(A[zero_rows] == 0.0)
    if resid_tol is not None:
        # the residual alone: r = U - u_lin on passive nodes of contacting patches
        passive = ~ref["mask"] & (np.abs(ref["U"]).sum(-1) > 0)
        r_ref = (ref["U"] - ref["analytic"])[passive]
        r_gpu = (U - A)[passive]
        rmax = float(np.abs(r_ref).max())
        err_r = float(np.abs(r_gpu - r_ref).max())
        stats["rel_r"] = err_r / max(rmax, 1e-30)
        assert err_r <= resid_tol * rmax, f"{label}: residual err {err_r:.3e} > {resid_tol}*{rmax:.3e}"
    return stats


def self_contact_workload(mesh, caps, seed, n_envs, n_ind, precision="bf16", weights=None, alpha=0.5):
    """Self-contact: the patches listed in ``caps`` = {patch: cap radius} sit on links whose
    collision shape is a sphere a little larger than the cap (it would press on every node of its own
    patch).  Per env one such link A is pressed onto a node of another patch B; slot 0 of the indenters is
    A's shape at A's pose with skip_patch1 = A + 1, the other slots are free objects pressed on other
    patches.  Every patch has its own rigid pose; patches not involved are parked apart."""
    rng = np.random.default_rng(4000 + seed)
    P, N = mesh.n_patches, mesh.n_nodes
    off = np.asarray(mesh.patch_offset)
    pos, nrm = mesh.pos.astype(np.float64), mesh.normal.astype(np.float64)
    ind = W._blank_indenters(n_envs, n_ind)
    pose = np.zeros((n_envs, P, 7), np.float32)
    meta = {"A": [], "B": []}
    for e in range(n_envs):
        Rm = W.random_rotations(rng, P)
        t = np.stack([60.0 * (np.arange(P) - P // 2), np.zeros(P), np.zeros(P)], 1) + rng.uniform(-5, 5, (P, 3))
        A = int(rng.choice(list(caps)))
        B = int(rng.choice([p for p in range(P) if p != A]))
        r_link = caps[A] + 0.25
        c = int(rng.integers(off[B], off[B + 1]))
        depth = rng.uniform(0.2, 1.0)
        centre_local = pos[c] + nrm[c] * (r_link - depth)            # A's sphere centre in B's frame
        t[B] = t[A] - Rm[B] @ centre_local                            # ... lands on A's world centre t[A]
        pose[e, :, 0:3] = t
        pose[e, :, 3:7] = W.quat_from_matrix(Rm)
        ind["type"][e, 0], ind["param"][e, 0, 0] = W.IND_SPHERE, r_link
        ind["pose"][e, 0, 0:3], ind["pose"][e, 0, 3:7] = t[A], [0, 0, 0, 1]
        ind["skip_patch1"][e, 0] = A + 1
        others = [p for p in range(P) if p not in (A, B)]
        for k in range(1, n_ind):                                     # free objects on other patches
            if not others or rng.random() < 0.3:
                continue
            C = int(rng.choice(others))
            cc = np.array([rng.integers(off[C], off[C + 1])])
            size = rng.uniform(2.0, 4.0, 1)
            cl, q = W._press_on_node(mesh.pos, mesh.normal, cc, None, size, rng.uniform(0.2, 0.9, 1), rng.uniform(0, 6.28, 1))
            from scipy.spatial.transform import Rotation as Rot
            ind["type"][e, k], ind["param"][e, k] = W.IND_CAPSULE, [size[0], rng.uniform(0, 3), 0]
            ind["pose"][e, k, 0:3] = Rm[C] @ cl[0] + t[C]
            ind["pose"][e, k, 3:7] = (Rot.from_matrix(Rm[C]) * Rot.from_quat(q[0])).as_quat()
        meta["A"].append(A), meta["B"].append(B)
    wl = W.Workload("self_contact", mesh, np.asarray([alpha], np.float32), weights or W.make_weights(3, seed), n_envs,
                    n_ind, ind, pose, precision, meta)
    return wl


def random_case(seed):
    """Seeded random workload for the randomised sweeps: 1-6 patches (caps and pads of 9-1400 nodes, sometimes a
    2048-3300-node cap: the cluster-pair path), 1-260 envs, 1-3 indenter slots (sphere / box / capsule, a quarter
    empty) each pressed 0.05-1.2 mm into a random node and shifted sideways off the shape's axis, with or without
    per-patch rigid poses; random residual form, alpha per patch or shared, precision, path and active-row mode.
    Returns (workload, resid_arch, precision, path, active_mode)."""
    rng = np.random.default_rng(seed)
    P = int(rng.integers(1, 7))
    parts = []
    for p in range(P):
        kind = rng.integers(0, 3)
        if kind == 0:
            parts.append(W.fib_cap(float(rng.uniform(5, 12)), int(rng.integers(9, 700))))
        elif kind == 1:
            g1, g2 = int(rng.integers(3, 26)), int(rng.integers(3, 26))
            parts.append(W.flat_pad(g1, g2, float(rng.uniform(0.6, 1.5))))
        else:
            big = rng.random() < 0.35
            parts.append(W.fib_cap(float(rng.uniform(8, 14)), int(rng.integers(2048, 3300)) if big else int(rng.integers(128, 1400))))
    mesh = W.assemble(parts)
    E = int(rng.integers(1, 72)) if rng.random() < 0.7 else int(rng.integers(72, 260))
    M = int(rng.integers(1, 4))
    ind = W._blank_indenters(E, M)
    off = np.asarray(mesh.patch_offset)
    posed = bool(rng.integers(0, 2))
    pose = None
    if posed:
        pose = np.zeros((E, P, 7), np.float32)
        for e in range(E):
            Rm = W.random_rotations(rng, P)
            pose[e, :, 0:3] = np.stack([70.0 * np.arange(P), np.zeros(P), np.zeros(P)], 1) + rng.uniform(-5, 5, (P, 3))
            pose[e, :, 3:7] = W.quat_from_matrix(Rm)
    for e in range(E):
        for k in range(M):
            if rng.random() < 0.25:
                continue
            p = int(rng.integers(0, P))
            c = np.asarray([int(rng.integers(off[p], off[p + 1]))])
            itype = int(rng.integers(1, 4))
            size = rng.uniform(1.5, 5.0, 1)
            centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, rng.uniform(0.05, 1.2, 1), rng.uniform(0, 6.28, 1))
            prm = [size[0], 0, 0]
            if itype == W.IND_BOX: prm = [rng.uniform(1.5, 5), rng.uniform(1.5, 5), size[0]]
            if itype == W.IND_CAPSULE: prm = [size[0] * 0.6, size[0] * 0.4, 0]
            cen, qq = centre[0], np.asarray(q[0], np.float64)
            cen = cen + O.quat_to_rot(qq) @ np.asarray([rng.uniform(0.05, 0.3), rng.uniform(0.05, 0.3), 0.0])   # no node on the shape's axis
            if posed:
                Rp = O.quat_to_rot(pose[e, p, 3:7].astype(np.float64))
                Rk = O.quat_to_rot(qq)
                cen = Rp @ cen + pose[e, p, 0:3]
                qq = W.quat_from_matrix(Rp @ Rk)
            ind["type"][e, k], ind["param"][e, k] = itype, prm
            ind["pose"][e, k, 0:3], ind["pose"][e, k, 3:7] = cen, qq
    arch = ["pernode", "pointnet", "none"][int(rng.integers(0, 3))]
    weights = W.make_pointnet_weights(9, seed, std=0.15) if arch == "pointnet" else W.make_weights(9, seed, std=0.2)
    alpha = np.asarray(rng.uniform(0.3, 0.9, P if rng.random() < 0.5 else 1), np.float32)
    prec = "bf16" if rng.random() < 0.6 else "fp32"
    wl = W.Workload(f"random{seed}", mesh, alpha, weights, E, M, ind, pose, prec)
    path = T.ETAC_PATH_AUTO if prec == "fp32" else [T.ETAC_PATH_DENSE, T.ETAC_PATH_SPARSE][int(rng.integers(0, 2))]
    mode = [T.ETAC_ACTIVE_PASSTHROUGH, T.ETAC_ACTIVE_PROPAGATE][int(rng.integers(0, 2))]
    return wl, arch, prec, path, mode
