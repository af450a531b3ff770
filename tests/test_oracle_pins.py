"""Pins of the CPU oracle against things other than itself.

Every check here compares oracle/etac_oracle.py with a closed form, a hand-derived value
(tests/golden/*.txt), a brute-force pure-Python loop, or a library routine (scipy cdist,
torch float64 linear/silu) -- never with the CUDA path."""
import math
import os

import numpy as np
import pytest

from oracle import etac_oracle as O
from paper_2604_20295_b200 import workloads as W
from conftest import read_golden


def pad_model(g1=16, g2=16, spacing=1.0, alpha=0.5, resid="none", weights=None, mode="passthrough"):
    pos, nrm, edges = W.flat_pad(g1, g2, spacing)
    mesh = W.assemble([(pos, nrm, edges)])
    return O.OracleModel(mesh.pos, mesh.normal, mesh.patch_offset, np.float32([alpha]), weights, resid, mode)


def one_sphere(centre, r):
    ind = np.zeros((1, 1), dtype=W.INDENTER_DTYPE)
    ind["type"] = W.IND_SPHERE
    ind["param"][0, 0, 0] = r
    ind["pose"][0, 0] = [*centre, 0, 0, 0, 1]
    return ind


# ---------------------------------------------------------------- P1
def test_zero_contact_gives_zero():
    wl = W.config2(seed=1, n_envs=3)
    m = O.model_from_workload(wl)
    ind = wl.indenters.copy()
    ind["pose"][..., 0:3] += 500.0          # far away
    r = O.step(m, indenters=ind)
    assert not r["mask"].any() and not r["contact"].any()
    assert np.all(r["U"] == 0.0) and np.all(r["analytic"] == 0.0)
    ind["type"][:] = W.IND_NONE             # no indenter at all
    r = O.step(m, indenters=ind)
    assert np.all(r["U"] == 0.0) and not r["mask"].any()


# ---------------------------------------------------------------- P2
def test_linear_term_is_linear_and_superposes():
    m = pad_model()
    rng = np.random.default_rng(0)
    d1 = np.zeros((1, 256), np.float32)
    d2 = np.zeros((1, 256), np.float32)
    d1[0, rng.choice(256, 9, replace=False)] = rng.uniform(0.1, 1, 9)
    d2[0, rng.choice(256, 5, replace=False)] = rng.uniform(0.1, 1, 5)
    a, b = 2.0, 0.5                          # exact in fp32
    r1 = O.step(m, penetration=d1)["analytic"]
    r2 = O.step(m, penetration=d2)["analytic"]
    r12 = O.step(m, penetration=(a * d1 + b * d2).astype(np.float32))["analytic"]
    np.testing.assert_allclose(r12, a * r1 + b * r2, rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P3
def test_single_point_contact_closed_form_decay():
    m = pad_model(21, 21)
    c = 10 * 21 + 10
    d = np.zeros((1, 441), np.float32)
    d[0, c] = 0.75
    r = O.step(m, penetration=d)
    uz = r["analytic"][0, :, 2].reshape(21, 21)
    assert np.all(r["analytic"][0, :, 0:2] == 0)
    # e^{-alpha r} with alpha = 0.5: mathematical constants
    expect = {(1, 0): 0.6065306597126334, (1, 1): 0.4930686913952398, (2, 0): 0.36787944117144233,
              (5, 0): 0.0820849986238988, (10, 0): 0.006737946999085467, (3, 4): 0.0820849986238988}
    for (dx, dy), k in expect.items():
        assert uz[10 + dx, 10 + dy] == pytest.approx(-0.75 * k, abs=1e-14)
    # radially symmetric and strictly decreasing with distance
    for dx, dy in [(1, 2), (3, 4), (0, 5)]:
        vals = {uz[10 + sx * a, 10 + sy * b] for a, b in [(dx, dy), (dy, dx)] for sx in (1, -1) for sy in (1, -1)}
        assert max(vals) - min(vals) < 1e-15
    rr = np.hypot(*(np.mgrid[0:21, 0:21] - 10)).ravel()
    order = np.argsort(rr)
    mag = -uz.ravel()[order]
    assert np.all(np.diff(mag)[np.diff(rr[order]) > 1e-9] < 0)
    # passthrough keeps u_hat on the active node
    assert r["U"][0, c, 2] == pytest.approx(-0.75, abs=0)


# ---------------------------------------------------------------- P4
def test_bruteforce_triple_loop_and_libraries():
    from scipy.spatial.distance import cdist
    import torch
    wl = W.config2(seed=3, n_envs=1)
    sub = np.arange(0, 1024, 37)[:28]
    mesh = wl.mesh
    m = O.OracleModel(mesh.pos[sub], mesh.normal[sub], np.int32([0, 12, 28]), np.float32([0.5, 0.3]), None, "none")
    rng = np.random.default_rng(5)
    d = np.where(rng.random((1, 28)) < 0.3, rng.uniform(0.1, 1.0, (1, 28)), 0).astype(np.float32)
    d[0, 0] = 0.5
    d[0, 20] = 0.25
    r = O.step(m, penetration=d)
    P = m.pos.astype(np.float64)
    Nn = m.normal.astype(np.float64)
    ref = np.zeros((28, 3))
    for lo, hi, al in [(0, 12, float(np.float32(0.5))), (12, 28, float(np.float32(0.3)))]:
        for i in range(lo, hi):
            for j in range(lo, hi):
                if d[0, j] > 0:
                    dist = math.sqrt(sum((P[i, c] - P[j, c]) ** 2 for c in range(3)))
                    for c in range(3):
                        ref[i, c] += math.exp(-al * dist) * (-float(d[0, j]) * Nn[j, c])
    np.testing.assert_allclose(r["analytic"][0], ref, rtol=0, atol=1e-14)
    # library: scipy cdist + torch float64 matmul on the dense zero-padded form K @ U_hat (R3)
    K0 = np.exp(-float(np.float32(0.5)) * cdist(P[:12], P[:12]))
    np.testing.assert_allclose(O.kernel_block(m, 0), K0, rtol=1e-14)
    Uhat = -d[0, :12, None].astype(np.float64) * Nn[:12]
    dense = (torch.from_numpy(K0) @ torch.from_numpy(Uhat)).numpy()
    np.testing.assert_allclose(r["analytic"][0, :12], dense, rtol=0, atol=1e-14)
    # block-diagonal: patch 1's contact does not leak into patch 0 (R9)
    d2 = d.copy()
    d2[0, 12:] = 0
    np.testing.assert_array_equal(O.step(m, penetration=d2)["analytic"][0, :12], r["analytic"][0, :12])


# ---------------------------------------------------------------- P5 / P6
def test_kernel_structure_and_lattice_sums(golden_dir):
    g = read_golden(os.path.join(golden_dir, "lattice_rowsums.txt"))
    m = pad_model()
    K = O.kernel_block(m, 0)
    assert np.array_equal(K, K.T) and np.all(np.diag(K) == 1.0) and K.min() > 0 and K.max() <= 1.0
    np.linalg.cholesky(K)                      # exponential kernel is positive definite
    ev = np.linalg.eigvalsh(K)
    assert ev[0] == pytest.approx(g["eig_min"][0], abs=5e-5) and ev[-1] == pytest.approx(g["eig_max"][0], abs=5e-4)
    assert K[0].sum() == pytest.approx(g["corner_0_0"][0], abs=g["tol"][0])
    assert K[7 * 16 + 7].sum() == pytest.approx(g["node_7_7"][0], abs=g["tol"][0])
    # pure-Python restatement of the corner sum
    s = sum(math.exp(-0.5 * math.hypot(a, b)) for a in range(16) for b in range(16))
    assert K[0].sum() == pytest.approx(s, abs=1e-12)
    assert K[7 * 16 + 7].sum() < 25.2465451858737 < 2 * math.pi / 0.25 + 0.2


# ---------------------------------------------------------------- W1 / W2 / P7
def test_worked_example_w1(golden_dir):
    g = read_golden(os.path.join(golden_dir, "w1_collinear.txt"))
    pos = np.float32([[0, 0, 0], [1, 0, 0], [2, 0, 0], [3, 0, 0]])
    nrm = np.float32([[0, 0, 1]] * 4)
    m = O.OracleModel(pos, nrm, np.int32([0, 4]), np.float32([0.5]), None, "none")
    r = O.step(m, penetration=np.float32([[0.4, 0, 0, 0.2]]))
    # fp32 inputs 0.4, 0.2 are not exact: tolerance covers their rounding (6e-9)
    np.testing.assert_allclose(r["analytic"][0, :, 2], g["analytic_z"], rtol=0, atol=2e-8)
    np.testing.assert_allclose(r["U"][0, :, 2], g["U_z"], rtol=0, atol=2e-8)
    assert list(r["mask"][0]) == [True, False, False, True]


def test_worked_example_w2_and_mask_semantics(golden_dir):
    g = read_golden(os.path.join(golden_dir, "w2_pad_sphere.txt"))
    m = pad_model()
    r = O.step(m, indenters=one_sphere((7.3, 8.6, 2.2), 3.0))
    ids = np.nonzero(r["mask"][0])[0]
    assert list(ids) == [int(x) for x in g["active_ids"]]
    tol = 5e-7        # centre coordinates 7.3/8.6/2.2 are fp32-rounded inputs
    for n in (120, 121, 137):
        assert r["delta"][0, n] == pytest.approx(g[f"delta_{n}"][0], abs=tol)
    assert r["delta"][0].sum() == pytest.approx(g["delta_sum"][0], abs=13 * tol)
    for n in (0, 89, 169, 255, 121):
        assert r["analytic"][0, n, 2] == pytest.approx(g[f"analytic_z_{n}"][0], abs=20 * tol)
    # P7: active rows keep u_hat, analytic on an active row double-counts
    K = O.kernel_block(m, 0)
    i = 121
    others = [j for j in ids if j != i]
    dbl = -r["delta"][0, i] - sum(K[i, j] * r["delta"][0, j] for j in others)
    assert r["analytic"][0, i, 2] == pytest.approx(dbl, abs=1e-13)
    assert r["U"][0, i, 2] == -r["delta"][0, i]
    # contact radius sqrt(2 r d - d^2) for a sphere on a flat pad (P9)
    d = 0.8
    rc = math.sqrt(2 * 3.0 * d - d * d)
    xy = m.pos[:, :2].astype(np.float64) - np.array([np.float32(7.3), np.float32(8.6)], dtype=np.float64)
    assert np.array_equal(np.hypot(xy[:, 0], xy[:, 1]) < rc - 1e-6, r["mask"][0])


# ---------------------------------------------------------------- P8
def test_rigid_invariance_via_patch_pose():
    wl = W.config2(seed=2, n_envs=2)
    m = O.model_from_workload(wl, resid_arch="none")
    base = O.step(m, indenters=wl.indenters)
    rng = np.random.default_rng(11)
    R = W.random_rotations(rng, 1)[0]
    t = np.array([12.0, -7.0, 3.5])
    ind = wl.indenters.copy()
    pose = np.zeros((2, 1, 7), np.float32)
    pose[..., 0:3] = t
    pose[..., 3:7] = W.quat_from_matrix(R)
    for e in range(2):
        for k in range(ind.shape[1]):
            c = ind["pose"][e, k, 0:3].astype(np.float64)
            Rk = O.quat_to_rot(ind["pose"][e, k, 3:7].astype(np.float64))
            ind["pose"][e, k, 0:3] = R @ c + t
            ind["pose"][e, k, 3:7] = W.quat_from_matrix(R @ Rk)
    moved = O.step(m, indenters=ind, patch_pose=pose)
    far = np.abs(base["delta"]) > 1e-4
    np.testing.assert_allclose(moved["delta"], base["delta"], rtol=0, atol=2e-5)
    assert np.array_equal(moved["mask"][far], base["mask"][far])
    np.testing.assert_allclose(moved["analytic"], base["analytic"], rtol=0, atol=2e-3)


# ---------------------------------------------------------------- P9
def test_sdf_spot_values_and_special_cases(golden_dir):
    kinds = {"sphere": O.IND_SPHERE, "box": O.IND_BOX, "capsule": O.IND_CAPSULE}
    n = 0
    with open(os.path.join(golden_dir, "sdf_spot_values.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].split()
            if not line:
                continue
            k, p, y, exp = kinds[line[0]], [float(x) for x in line[1:4]], [float(x) for x in line[4:7]], float(line[7])
            got = O.sdf_local(k, p, *[np.array([v]) for v in y])[0]
            assert got == pytest.approx(exp, abs=1e-14), line
            n += 1
    assert n == 12
    rng = np.random.default_rng(3)
    y = rng.normal(size=(3, 200)) * 4
    # capsule with zero half-length is a sphere
    np.testing.assert_allclose(O.sdf_local(O.IND_CAPSULE, [2.5, 0, 0], *y), O.sdf_local(O.IND_SPHERE, [2.5, 0, 0], *y), atol=1e-15)
    # box with two huge half extents is a slab: |y2| - h
    np.testing.assert_allclose(O.sdf_local(O.IND_BOX, [1e6, 1e6, 1.5], *y), np.abs(y[2]) - 1.5, atol=1e-9)
    # 1-Lipschitz (exact distance fields): |phi(a)-phi(b)| <= |a-b|
    a, b = rng.normal(size=(3, 500)) * 5, rng.normal(size=(3, 500)) * 5
    for k, p in [(O.IND_SPHERE, [3, 0, 0]), (O.IND_BOX, [2, 3, 4]), (O.IND_CAPSULE, [2, 5, 0])]:
        assert np.all(np.abs(O.sdf_local(k, p, *a) - O.sdf_local(k, p, *b)) <= np.linalg.norm(a - b, axis=0) + 1e-12)
    # flat pad under a slab: delta equals the plane depth everywhere
    m = pad_model()
    ind = np.zeros((1, 1), dtype=W.INDENTER_DTYPE)
    ind["type"], ind["param"][0, 0] = W.IND_BOX, [1e4, 1e4, 2.0]
    ind["pose"][0, 0] = [0, 0, 1.75, 0, 0, 0, 1]
    r = O.step(m, indenters=ind)
    np.testing.assert_allclose(r["delta"][0], 0.25, atol=1e-12)
    # quaternion -> rotation: 90 deg about z maps x to y; orthonormal; matches scipy
    from scipy.spatial.transform import Rotation
    q = np.array([0, 0, math.sin(math.pi / 4), math.cos(math.pi / 4)])
    np.testing.assert_allclose(O.quat_to_rot(q) @ [1, 0, 0], [0, 1, 0], atol=1e-15)
    qs = W.quat_from_matrix(W.random_rotations(rng, 20))
    for qq in qs:
        np.testing.assert_allclose(O.quat_to_rot(qq), Rotation.from_quat(qq).as_matrix(), atol=1e-14)


# ---------------------------------------------------------------- P10
def test_mlp_matches_torch_float64():
    import torch
    w = W.make_weights(9, seed=4, std=0.3)
    rng = np.random.default_rng(2)
    ul, p, n = rng.normal(size=(50, 3)), rng.normal(size=(50, 3)) * 5, rng.normal(size=(50, 3))
    got = O.residual_pernode(w, ul, p, n)
    t = {k: torch.from_numpy(v.astype(np.float64)) for k, v in w.items()}
    x = torch.from_numpy(np.concatenate([ul, p, n], 1))
    F = torch.nn.functional
    ref = F.linear(F.silu(F.linear(F.silu(F.linear(x, t["W1"], t["b1"])), t["W2"], t["b2"])), t["W3"], t["b3"])
    np.testing.assert_allclose(got, ref.numpy(), rtol=0, atol=1e-13)
    # zero weights -> r = b3 ; zero everything -> U_passive = u_lin
    z = {k: np.zeros_like(v) for k, v in w.items()}
    z["b3"] = np.float32([0.1, -0.2, 0.3])
    np.testing.assert_allclose(O.residual_pernode(z, ul, p, n), np.tile(z["b3"].astype(np.float64), (50, 1)))
    m0 = pad_model(resid="pernode", weights={k: np.zeros_like(v) for k, v in w.items()})
    r = O.step(m0, indenters=one_sphere((7.3, 8.6, 2.2), 3.0))
    passive = ~r["mask"][0]
    np.testing.assert_array_equal(r["U"][0][passive], r["analytic"][0][passive])
    # input order [u_lin, p, n]: only W1[:,0:3] sees u_lin
    w2 = {k: v.copy() for k, v in w.items()}
    w2["W1"][:, 3:] = 0
    a = O.residual_pernode(w2, ul, p, n)
    b = O.residual_pernode(w2, ul, p * 0 + 1, n * 0 - 2)
    np.testing.assert_allclose(a, b, atol=1e-15)


# ---------------------------------------------------------------- P11
def test_mode_reductions():
    wl = W.config2(seed=5, n_envs=3)
    full = O.step(O.model_from_workload(wl), indenters=wl.indenters)
    lin = O.step(O.model_from_workload(wl, resid_arch="none"), indenters=wl.indenters)
    passive = ~full["mask"]
    np.testing.assert_array_equal(lin["U"][passive], lin["analytic"][passive])
    np.testing.assert_array_equal(full["analytic"], lin["analytic"])
    assert np.abs(full["U"] - lin["U"])[passive & full["contact"][:, [0]]].max() > 1e-4   # residual is there
    # PENETRATION fed with the fp32 delta that INDENTERS emitted -> same masks, U within fp32 rounding
    pen = O.step(O.model_from_workload(wl), penetration=full["delta32"])
    assert np.array_equal(pen["mask"], full["mask"])
    np.testing.assert_allclose(pen["U"], full["U"], rtol=0, atol=1e-5)
    # propagate mode: no mask, active rows get u_lin + r too
    prop = O.step(O.model_from_workload(wl, active_mode="propagate"), indenters=wl.indenters)
    np.testing.assert_array_equal(prop["U"][passive], full["U"][passive])
    act = full["mask"]
    assert np.abs(prop["U"][act] - full["U"][act]).max() > 1e-3


def test_ablation_modes_reduce_to_their_definitions():
    """Table II rows as oracle modes: "linear_only" is the model without Phi,
    "residual_only" + "linear_only" add up to "full" on the passive rows, "no_propagation" is U^."""
    wl = W.config2(seed=5, n_envs=3)
    def run(abl, **kw):
        m = O.model_from_workload(wl, **kw)
        m.ablation = abl
        return O.step(m, indenters=wl.indenters)
    full, lin, res, nop = run("full"), run("linear_only"), run("residual_only"), run("no_propagation")
    none = run("full", resid_arch="none")
    np.testing.assert_array_equal(lin["U"], none["U"])
    passive = ~full["mask"]
    np.testing.assert_allclose((lin["U"] + res["U"])[passive], full["U"][passive], rtol=0, atol=1e-12)
    nrm = wl.mesh.normal.astype(np.float64)
    np.testing.assert_array_equal(nop["U"], -full["delta"][:, :, None] * nrm[None])
    assert np.all(nop["U"][passive] == 0) and np.abs(nop["U"][full["mask"]]).max() > 0.05


def test_self_contact_skip_is_per_patch():
    """Self-contact: a link's collision shape is an indenter for every patch but its own.
    Brute force per patch: with the skip, patch A sees only the other indenters; every other patch sees the
    plain union."""
    from parity_util import self_contact_workload
    mesh = W.assemble([W.fib_cap(6.0, 72), W.flat_pad(10, 12, 1.0), W.fib_cap(5.0, 60)])
    wl = self_contact_workload(mesh, {0: 6.0, 2: 5.0}, seed=3, n_envs=6, n_ind=2, precision="fp32")
    m = O.model_from_workload(wl)
    off = np.asarray(mesh.patch_offset)
    for e in range(wl.n_envs):
        A, B = wl.meta["A"][e], wl.meta["B"][e]
        phi = O.signed_distance(m, wl.indenters[e], wl.patch_pose[e])
        plain = wl.indenters[e].copy()
        plain["skip_patch1"] = 0
        phi_plain = O.signed_distance(m, plain, wl.patch_pose[e])
        without = plain.copy()
        without["type"][0] = W.IND_NONE
        phi_without = O.signed_distance(m, without, wl.patch_pose[e])
        sl = slice(off[A], off[A + 1])
        np.testing.assert_array_equal(phi[sl], phi_without[sl])
        rest = np.ones(mesh.n_nodes, bool)
        rest[sl] = False
        np.testing.assert_array_equal(phi[rest], phi_plain[rest])
        # the own shape alone would press on every node of A by 0.25; B is pressed by A's shape
        np.testing.assert_allclose(phi_plain[sl], -0.25, atol=5e-6)   # fp32 poses and positions
        assert (phi_plain[sl] < 0).all() and (phi[off[B]:off[B + 1]] < 0).any()


def _grad_case(n_alpha_per_patch, active_mode="passthrough", resid_arch="pernode"):
    import dataclasses
    mesh = W.assemble([W.fib_cap(6.0, 72), W.flat_pad(10, 12, 1.0)])
    rng = np.random.default_rng(77)
    E = 3
    ind = W._blank_indenters(E, 2)
    for k in range(2):
        c = rng.integers(0, mesh.n_nodes, size=E)
        size = rng.uniform(2.0, 4.0, E)
        centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, rng.uniform(0.2, 1.0, E), rng.uniform(0, 6.28, E))
        ind["type"][:, k], ind["param"][:, k, 0] = W.IND_SPHERE, size
        ind["pose"][:, k, 0:3], ind["pose"][:, k, 3:7] = centre, q
    alpha = np.asarray([0.45, 0.7] if n_alpha_per_patch else [0.5], np.float32)
    weights = W.make_weights(9, 1, std=0.3)
    if resid_arch == "pointnet":
        weights = {**weights, **W.make_pointnet_weights(9, 1, std=0.3)}
    wl = W.Workload("grad_case", mesh, alpha, weights, E, 2, ind, None, "fp32")
    target = rng.normal(0, 0.2, (E, mesh.n_nodes, 3))

    def loss(wl_):
        U = O.step(O.model_from_workload(wl_, resid_arch=resid_arch, active_mode=active_mode), indenters=wl_.indenters)["U"]
        return 0.5 * float(((U - target) ** 2).sum()), U
    return wl, target, loss, dataclasses


@pytest.mark.parametrize("per_patch,active_mode,resid_arch", [(True, "passthrough", "pernode"), (False, "propagate", "pernode"),
                                                               (True, "passthrough", "none"), (True, "passthrough", "pointnet"),
                                                               (False, "propagate", "pointnet")])
def test_backward_oracle_matches_finite_differences(per_patch, active_mode, resid_arch):
    """The gradient oracle against its definition: central differences of the (pinned) forward oracle's
    loss 0.5*||U - U*||^2 (Eq. 3) in alpha and in sampled weights of every layer."""
    from oracle import etac_oracle_grad as OG
    wl, target, loss, dataclasses = _grad_case(per_patch, active_mode, resid_arch)
    _, U = loss(wl)
    m = O.model_from_workload(wl, resid_arch=resid_arch, active_mode=active_mode)
    g = OG.backward(m, U - target, indenters=wl.indenters)
    eps = 1e-6
    for k in range(len(wl.alpha)):
        a = wl.alpha.astype(np.float64)
        ap, am = a.copy(), a.copy()
        ap[k] += eps
        am[k] -= eps
        fd = (loss(dataclasses.replace(wl, alpha=ap))[0] - loss(dataclasses.replace(wl, alpha=am))[0]) / (2 * eps)
        assert abs(fd - g["alpha"][k]) <= 1e-6 * max(1.0, abs(fd)), (k, fd, g["alpha"][k])
    assert np.abs(g["alpha"]).min() > 1e-3                        # the case exercises every alpha
    # dL/ddelta in penetration input mode (the contact set stays fixed under a small change of a positive delta)
    pen = O.step(m, indenters=wl.indenters)["delta"].astype(np.float32).astype(np.float64)   # the input is fp32
    eps_p = 2.0 ** -12                                            # d +- eps_p is exact in fp32

    def loss_pen(d):
        U_ = O.step(m, penetration=d)["U"]
        return 0.5 * float(((U_ - target) ** 2).sum()), U_
    _, U_pen = loss_pen(pen)
    gp = OG.backward(m, U_pen - target, penetration=pen)["delta"]
    act = np.argwhere(pen > 0.05)
    assert np.all(gp[pen == 0] == 0) and len(act) > 10
    for e_, j_ in act[:: max(1, len(act) // 6)]:
        dp, dm = pen.copy(), pen.copy()
        dp[e_, j_] += eps_p
        dm[e_, j_] -= eps_p
        fd = (loss_pen(dp)[0] - loss_pen(dm)[0]) / (2 * eps_p)
        assert abs(fd - gp[e_, j_]) <= 1e-5 * max(1.0, abs(fd)), (e_, j_, fd, gp[e_, j_])
    if resid_arch == "none":
        return
    rng = np.random.default_rng(5)
    names = ("W1", "b1", "W2", "b2", "W3", "b3") if resid_arch == "pernode" else ("E1", "e1", "E2", "e2", "G1", "g1", "D1", "d1", "D2", "d2")
    noise = 8 * np.finfo(np.float64).eps * abs(loss(wl)[0]) / eps       # rounding of the two losses in the difference quotient
    for name in names:
        base = wl.weights[name].astype(np.float64)
        tested = 0
        for _ in range(200):
            idx = tuple(rng.integers(0, s) for s in base.shape)
            if abs(g[name][idx]) < 100 * noise:                       # the quotient's rounding would hide a mistake
                continue
            tested += 1
            wp, wm = base.copy(), base.copy()
            wp[idx] += eps
            wm[idx] -= eps
            fd = (loss(dataclasses.replace(wl, weights={**wl.weights, name: wp}))[0]
                  - loss(dataclasses.replace(wl, weights={**wl.weights, name: wm}))[0]) / (2 * eps)
            assert abs(fd - g[name][idx]) <= 2e-6 * max(1.0, abs(fd)) + noise, (name, idx, fd, g[name][idx], noise)
            if tested == 3:
                break
        assert tested == 3 and np.abs(g[name]).max() > 1e-4


# ---------------------------------------------------------------- P12
def test_pointnet_branch_is_permutation_equivariant():
    rng = np.random.default_rng(8)
    shp = {"E1": (64, 9), "e1": (64,), "E2": (64, 64), "e2": (64,), "G1": (64, 64), "g1": (64,),
           "D1": (64, 128), "d1": (64,), "D2": (3, 64), "d2": (3,)}
    w = {k: rng.normal(0, 0.2, s).astype(np.float32) for k, s in shp.items()}
    n = 40
    uh, p, nr = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)), rng.normal(size=(n, 3))
    perm = rng.permutation(n)
    a = O.residual_pointnet(w, uh, p, nr)
    b = O.residual_pointnet(w, uh[perm], p[perm], nr[perm])
    np.testing.assert_allclose(a[perm], b, atol=1e-13)
    assert a.shape == (n, 3)
    # the global feature couples nodes: changing one node's input changes another node's output
    uh2 = uh.copy()
    uh2[0] += 5.0
    assert np.abs(O.residual_pointnet(w, uh2, p, nr)[1:] - a[1:]).max() > 1e-6


def _pointnet_weights(seed, std=0.2):
    rng = np.random.default_rng(seed)
    shp = {"E1": (64, 9), "e1": (64,), "E2": (64, 64), "e2": (64,), "G1": (64, 64), "g1": (64,),
           "D1": (64, 128), "d1": (64,), "D2": (3, 64), "d2": (3,)}
    return {k: rng.normal(0, std, s).astype(np.float32) for k, s in shp.items()}


def test_pointnet_branch_against_torch_float64_restatement():
    """PAPER.md:L93-L99 restated with library routines in the paper's order: n x 9 input [P, N, U^]
    -> shared MLP (point-wise features) -> Max-Pooling into a 64-d global feature -> another MLP ->
    broadcast + concatenate with the per-node features (n x 128) -> shared-MLP decoder -> n x 3.
    torch float64 F.linear / F.silu / torch.max / torch.cat; no code shared with the oracle."""
    import torch
    import torch.nn.functional as F
    w = _pointnet_weights(31)
    rng = np.random.default_rng(32)
    for n in (1, 7, 300):
        uh, p, nr = rng.normal(0, 0.7, (n, 3)), rng.normal(0, 3.0, (n, 3)), rng.normal(size=(n, 3))
        t = {k: torch.from_numpy(v.astype(np.float64)) for k, v in w.items()}
        x = torch.cat([torch.from_numpy(p), torch.from_numpy(nr), torch.from_numpy(uh)], dim=1)   # [P, N, U^]
        f = F.silu(F.linear(F.silu(F.linear(x, t["E1"], t["e1"])), t["E2"], t["e2"]))                # n x 64
        g = torch.max(f, dim=0).values                                                               # 64-d global feature
        g = F.silu(F.linear(g, t["G1"], t["g1"]))                                                    # "another MLP"
        cat = torch.cat([f, g.unsqueeze(0).expand(n, 64)], dim=1)                                    # n x 128, [f_i ; g']
        want = F.linear(F.silu(F.linear(cat, t["D1"], t["d1"])), t["D2"], t["d2"]).numpy()
        got = O.residual_pointnet(w, uh, p, nr)
        assert got.shape == (n, 3)
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-13 * max(1.0, np.abs(want).max()))


def test_pointnet_branch_structure():
    """What the permutation test cannot see: (a) the max-pool is the ONLY coupling between nodes: changing
    the input of a node that holds no column maximum leaves every other node's output unchanged; (b) the
    concatenation order is [f_i ; g']: with D1[:, :64] = 0 the output does not depend on f_i (all rows
    equal), with D1[:, 64:] = 0 it does not depend on the other nodes; (c) the global MLP sits between the
    pool and the concat (zero G1 and g1 => g' = 0, so the output equals the one with D1[:, 64:] = 0);
    (d) the pool is a max, not a mean or sum: duplicating a node changes nothing."""
    w = _pointnet_weights(33)
    rng = np.random.default_rng(34)
    n = 50
    uh, p, nr = rng.normal(0, 0.5, (n, 3)), rng.normal(size=(n, 3)), rng.normal(size=(n, 3))
    a = O.residual_pointnet(w, uh, p, nr)
    # (a) find a node that is arg-max of no encoder column, perturb it slightly (it must stay below the maxima)
    f64 = lambda k: w[k].astype(np.float64)
    x9 = np.concatenate([p, nr, uh], 1)
    f = O.silu(O.silu(x9 @ f64("E1").T + f64("e1")) @ f64("E2").T + f64("e2"))
    holders = set(np.argmax(f, axis=0).tolist())
    free = [i for i in range(n) if i not in holders]
    assert free
    i0 = free[0]
    uh2 = uh.copy()
    uh2[i0] += 1e-3
    x9b = np.concatenate([p, nr, uh2], 1)
    fb = O.silu(O.silu(x9b @ f64("E1").T + f64("e1")) @ f64("E2").T + f64("e2"))
    assert np.array_equal(fb.max(0), f.max(0))                    # still below every column maximum
    b = O.residual_pointnet(w, uh2, p, nr)
    others = np.arange(n) != i0
    assert np.array_equal(a[others], b[others]) and np.abs(a[i0] - b[i0]).max() > 0
    # (b) concat order
    wz = dict(w)
    wz["D1"] = w["D1"].copy()
    wz["D1"][:, :64] = 0
    c = O.residual_pointnet(wz, uh, p, nr)
    assert np.abs(c - c[0]).max() < 1e-14 and np.abs(a - a[0]).max() > 1e-3
    wy = dict(w)
    wy["D1"] = w["D1"].copy()
    wy["D1"][:, 64:] = 0
    d_all = O.residual_pointnet(wy, uh, p, nr)
    d_sub = O.residual_pointnet(wy, uh[:10], p[:10], nr[:10])
    np.testing.assert_allclose(d_all[:10], d_sub, atol=1e-14)     # per-node only once the global half is cut
    # (c) the global MLP: g' = silu(G1 g + g1); zero G1, g1 => g' = 0 => same as cutting D1[:, 64:]
    wg = dict(w)
    wg["G1"], wg["g1"] = np.zeros_like(w["G1"]), np.zeros_like(w["g1"])
    np.testing.assert_allclose(O.residual_pointnet(wg, uh, p, nr), d_all, atol=1e-14)
    # (d) max-pool: a duplicated node changes nothing for the original nodes
    dup = lambda v: np.concatenate([v, v[3:4]], 0)
    e = O.residual_pointnet(w, dup(uh), dup(p), dup(nr))
    np.testing.assert_allclose(e[:n], a, atol=1e-14)
    np.testing.assert_allclose(e[n], a[3], atol=1e-14)


# ---------------------------------------------------------------- fp32 decision twin
@pytest.mark.parametrize("cfg", ["cfg3", "cfg4"])
def test_full_size_twin_band_is_empty_or_harmless(cfg):
    """SURVEY.md Q7 / DESIGN.md §5 at BASELINE.json's full sizes: the contact decision is taken on the fp32
    twin; the two evaluations may only disagree for nodes within the band |phi64| < 1e-4 of the surface.
    Counts the nodes of the full-size bench workloads in that band and asserts that the twin's mask equals
    the float64 mask everywhere outside it (cfg 3: all 4096 envs; cfg 4: every 8th env)."""
    if cfg == "cfg3":
        wl, envs, band = W.config3(0, 4096), range(4096), 1e-4
    else:
        wl, envs, band = W.config4(0, 4096), range(0, 4096, 8), 1e-4
    m = O.model_from_workload(wl)
    in_band = disagree = evaluated = 0
    for e in envs:
        pp = None if wl.patch_pose is None else wl.patch_pose[e]
        p64 = O.signed_distance(m, wl.indenters[e], pp, np.float64)
        p32 = O.signed_distance(m, wl.indenters[e], pp, np.float32)
        near = np.abs(p64) < band
        in_band += int(near.sum())
        evaluated += int((p64 < 50.0).sum())
        diff = (p32 < 0) != (p64 < 0)
        disagree += int(diff.sum())
        assert not (diff & ~near).any(), (e, np.argwhere(diff & ~near)[:4])
    print(f"[twin band] {cfg}: {in_band} of {evaluated} nodes within 50 mm of an indenter have |phi64| < {band}; "
          f"{disagree} decisions differ (all inside the band)")
    assert in_band <= 1e-4 * evaluated + 5


def test_fp32_twin_agrees_with_fp64_away_from_the_surface():
    for wl in (W.config2(seed=7, n_envs=6), W.config3(seed=7, n_envs=4)):
        m = O.model_from_workload(wl)
        for e in range(wl.n_envs):
            pp = None if wl.patch_pose is None else wl.patch_pose[e]
            p64 = O.signed_distance(m, wl.indenters[e], pp, np.float64)
            p32 = O.signed_distance(m, wl.indenters[e], pp, np.float32)
            assert p32.dtype == np.float32
            near = p64 < 100.0
            assert np.abs(p32[near] - p64[near]).max() < 1e-4
            far = np.abs(p64) > 1e-4
            assert np.array_equal((p32 < 0)[far], (p64 < 0)[far])


# ---------------------------------------------------------------- sampled-grid SDF (R21)
def _grid_of(fn, n=(9, 11, 13), origin=(-2.0, -2.5, -3.0), h=0.5):
    nx, ny, nz = n
    x = origin[0] + h * np.arange(nx)
    y = origin[1] + h * np.arange(ny)
    z = origin[2] + h * np.arange(nz)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return fn(X, Y, Z).astype(np.float32), (x, y, z)


def test_grid_sdf_matches_library_trilinear_interpolation_inside():
    from scipy.interpolate import RegularGridInterpolator
    rng = np.random.default_rng(21)
    vals = rng.normal(size=(13, 11, 9)).astype(np.float32)          # arbitrary samples: pure interpolation
    origin, h = (-2.0, -2.5, -3.0), 0.5
    x, y, z = (origin[a] + h * np.arange(n) for a, n in zip(range(3), (9, 11, 13)))
    rgi = RegularGridInterpolator((z, y, x), vals.astype(np.float64), method="linear")
    q = np.stack([rng.uniform(x[0], x[-1], 500), rng.uniform(y[0], y[-1], 500), rng.uniform(z[0], z[-1], 500)], 1)
    got = O.sdf_grid(vals, origin, h, q[:, 0], q[:, 1], q[:, 2])
    np.testing.assert_allclose(got, rgi(q[:, ::-1]), atol=1e-12)
    # at a grid point the sample itself comes back
    assert O.sdf_grid(vals, origin, h, x[3], y[10], z[12]) == pytest.approx(float(vals[12, 10, 3]), abs=1e-12)


def test_grid_sdf_is_exact_for_a_plane_and_adds_the_distance_outside():
    vals, (x, y, z) = _grid_of(lambda X, Y, Z: Z - 0.25)            # half-space z < 0.25: affine => exact
    origin, h = (-2.0, -2.5, -3.0), 0.5
    rng = np.random.default_rng(22)
    q = np.stack([rng.uniform(x[0], x[-1], 200), rng.uniform(y[0], y[-1], 200), rng.uniform(-6.0, 6.0, 200)], 1)
    got = O.sdf_grid(vals, origin, h, q[:, 0], q[:, 1], q[:, 2])
    np.testing.assert_allclose(got, q[:, 2] - 0.25 + np.where(q[:, 2] < z[0], 2 * (z[0] - q[:, 2]), 0.0), atol=1e-6)
    # sideways outside the box: value at the clamped point plus the distance to the box
    far = O.sdf_grid(vals, origin, h, x[-1] + 3.0, 0.0, 1.0)
    assert far == pytest.approx((1.0 - 0.25) + 3.0, abs=1e-6)


def test_grid_sdf_of_a_sphere_obeys_the_interpolation_bound():
    R, h = 1.5, 0.25
    vals, (x, y, z) = _grid_of(lambda X, Y, Z: np.sqrt(X * X + Y * Y + Z * Z) - R, n=(25, 25, 25),
                               origin=(-3.0, -3.0, -3.0), h=h)
    rng = np.random.default_rng(23)
    q = rng.uniform(-2.9, 2.9, (2000, 3))
    rho = np.linalg.norm(q, axis=1)
    keep = rho > 1.0
    got = O.sdf_grid(vals, (-3.0, -3.0, -3.0), h, q[keep, 0], q[keep, 1], q[keep, 2])
    # trilinear error <= h^2/8 * sum |d2 phi / dx_a^2| <= h^2/8 * 2/rho (Laplacian of |x|), + fp32 samples
    assert np.all(np.abs(got - (rho[keep] - R)) <= h * h / 8 * 2 / (rho[keep] - h * np.sqrt(3)) + 1e-6)
    # fp32 twin: same formula, every op in float32, agrees to rounding
    got32 = O.sdf_grid(vals, (-3.0, -3.0, -3.0), h, q[keep, 0], q[keep, 1], q[keep, 2], np.float32)
    assert got32.dtype == np.float32 and np.abs(got32 - got).max() < 5e-6


# ---------------------------------------------------------------- P13: signed distance to a closed triangle mesh
def _ray_parity_inside(V, T, P, direction):
    """Brute force: a point is inside a closed surface iff a ray from it crosses the surface an odd number of times
    (Moeller-Trumbore ray/triangle test, written out here; random direction, so no edge is hit exactly)."""
    inside = np.zeros(len(P), dtype=bool)
    for a, b, c in V[T]:
        e1, e2 = b - a, c - a
        h = np.cross(direction, e2)
        det = e1 @ h
        s = P - a
        u = (s @ h) / det
        qv = np.cross(s, e1)
        v = (qv @ direction) / det
        t = (qv @ e2) / det
        inside ^= (u >= 0) & (v >= 0) & (u + v <= 1) & (t > 0)
    return inside


def test_mesh_sdf_oracle_against_closed_forms_and_ray_parity():
    """oracle/etac_oracle_mesh.py (the SDF of an object mesh) against what the mathematics fixes:
    a box mesh = the closed-form box SDF everywhere; inside a tetrahedron = minus the smallest face-plane distance;
    an icosphere within its sagitta of |x| - r with the right sign; the sign against brute-force ray parity; the
    result does not depend on the order or the (consistent) orientation of the triangles."""
    from oracle import etac_oracle_mesh as M
    rng = np.random.default_rng(11)
    # (1) box: exact closed form, inside and outside, faces / edges / corners regions
    V, T = W.box_mesh(1.0, 2.0, 0.5)
    P = rng.uniform(-3.0, 3.0, (3000, 3))
    phi = M.mesh_signed_distance(V, T, P)
    ref = O.sdf_local(O.IND_BOX, [1.0, 2.0, 0.5], P[:, 0], P[:, 1], P[:, 2])
    assert (ref < 0).sum() > 50 and np.abs(phi - ref).max() <= 1e-12
    # (2) convex polyhedron, interior points: phi = -min_f distance to the plane of face f
    V, T = W.tetra_mesh(1.5)
    Q = rng.uniform(-0.4, 0.4, (500, 3))
    n = np.cross(V[T[:, 1]] - V[T[:, 0]], V[T[:, 2]] - V[T[:, 0]])
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    plane = np.einsum("fj,nfj->nf", n, V[T[:, 0]][None] - Q[:, None])           # > 0 inside (outward normals)
    assert (plane > 0).all()
    assert np.abs(M.mesh_signed_distance(V, T, Q) + plane.min(1)).max() <= 1e-12
    # (3) icosphere: polyhedron inscribed in the sphere of radius r; its faces stay within the sagitta of the sphere
    r = 2.0
    V, T = W.icosphere(r, 2)
    inradius = np.abs(np.einsum("fj,fj->f", np.cross(V[T[:, 1]] - V[T[:, 0]], V[T[:, 2]] - V[T[:, 0]]) /
                                np.linalg.norm(np.cross(V[T[:, 1]] - V[T[:, 0]], V[T[:, 2]] - V[T[:, 0]]), axis=1, keepdims=True),
                                V[T[:, 0]])).min()
    sag = r - inradius
    assert 0 < sag < 0.05 * r
    P = rng.uniform(-3.0, 3.0, (2000, 3))
    phi = M.mesh_signed_distance(V, T, P)
    rad = np.linalg.norm(P, axis=1)
    assert (np.abs(phi - (rad - r)) <= sag + 1e-12).all()
    assert (phi[rad < inradius] < 0).all() and (phi[rad > r] > 0).all()
    # (4) sign = ray parity (brute force), on the icosphere and on the box
    d = rng.normal(size=3)
    d /= np.linalg.norm(d)
    assert np.array_equal(phi < 0, _ray_parity_inside(V, T, P, d))
    Vb, Tb = W.box_mesh(1.0, 2.0, 0.5)
    Pb = rng.uniform(-2.5, 2.5, (2000, 3))
    assert np.array_equal(M.mesh_signed_distance(Vb, Tb, Pb) < 0, _ray_parity_inside(Vb, Tb, Pb, d))
    # (5) triangle order and orientation do not matter
    perm = rng.permutation(len(T))
    assert np.abs(M.mesh_signed_distance(V, T[perm], P[:300]) - phi[:300]).max() <= 1e-12
    assert np.abs(M.mesh_signed_distance(V, T[:, ::-1], P[:300]) - phi[:300]).max() <= 1e-12
    # (6) the grid layout of etac_set_sdf_grid: values[iz, iy, ix] at origin + h (ix, iy, iz)
    g = M.mesh_sdf_grid(Vb, Tb, (4, 5, 3), (-1.5, -2.0, -1.0), 1.0)
    assert g.shape == (3, 5, 4)
    assert abs(g[2, 1, 3] - O.sdf_local(O.IND_BOX, [1.0, 2.0, 0.5], np.float64(1.5), np.float64(-1.0), np.float64(1.0))) <= 1e-12


# ---------------------------------------------------------------- pose gradients (dL/ddelta chained to the poses)
IND64 = np.dtype([("type", "<i4"), ("param", "<f8", (3,)), ("pose", "<f8", (7,)), ("skip_patch1", "<i4")])


def _quat_mul(a, b):
    """Hamilton product a (x) b of quaternions stored (x, y, z, w): the rotation b followed by the rotation a."""
    ax, ay, az, aw = a
    bx, by, bz, bw = b
    return np.array([aw * bx + ax * bw + ay * bz - az * by, aw * by - ax * bz + ay * bw + az * bx,
                     aw * bz + ax * by - ay * bx + az * bw, aw * bw - ax * bx - ay * by - az * bz])


def _perturb_pose(pose7, dof, eps):
    """pose (t, q) with t[dof] += eps (dof 0-2) or rotated on the left by eps about world axis dof - 3."""
    out = np.array(pose7, dtype=np.float64)
    if dof < 3:
        out[dof] += eps
    else:
        dq = np.zeros(4)
        dq[dof - 3], dq[3] = math.sin(eps / 2), math.cos(eps / 2)
        out[3:7] = _quat_mul(dq, out[3:7])
    return out


def pose_grad_case(seed=91, n_envs=2):
    """Two patches under their own rigid poses; four indenter slots per env -- sphere, box (tilted), capsule (pressed
    with its rounded end and its side), sampled grid (an ellipsoid-like field) -- each pressed into a node of one of
    the patches.  Poses are fp32-representable float64 (the fp32 decision twin sees the same numbers)."""
    mesh = W.assemble([W.fib_cap(6.0, 260), W.flat_pad(14, 16, 0.7)])
    rng = np.random.default_rng(seed)
    E, M = n_envs, 4
    off = mesh.patch_offset
    ppose = np.zeros((E, 2, 7))
    ind = np.zeros((E, M), dtype=IND64)
    Rp = W.random_rotations(rng, E * 2).reshape(E, 2, 3, 3)
    gvals, _ = _grid_of(lambda X, Y, Z: np.sqrt((X / 1.2) ** 2 + Y ** 2 + (Z / 1.5) ** 2) * 1.2 - 2.0, n=(17, 17, 21),
                        origin=(-4.13, -3.87, -5.06), h=0.5)   # no grid plane through the local z axis,
    # on which the pressed node lies: the interpolant has kinks on the planes and a central difference would straddle one
    for e in range(E):
        for p in range(2):
            ppose[e, p, 0:3] = rng.uniform(-20, 20, 3) + (40.0 * p, 0, 0)
            ppose[e, p, 3:7] = W.quat_from_matrix(Rp[e, p])
        for k, itype in enumerate((O.IND_SPHERE, O.IND_BOX, O.IND_CAPSULE, O.IND_GRID)):
            p = (k + e) % 2
            cand = np.arange(off[p], off[p + 1])
            cand = cand[mesh.normal[cand, 2] > 0.6]
            c = rng.choice(cand, size=1)
            size = rng.uniform(2.0, 3.0, 1)
            prm = [size[0], 0.0, 0.0]
            if itype == O.IND_BOX:
                prm = [rng.uniform(2, 4), rng.uniform(2, 4), size[0]]
            if itype == O.IND_CAPSULE:
                prm = [size[0] * 0.6, size[0] * 0.4, 0.0]           # r + L = size: pressed with its rounded end
            if itype == O.IND_GRID:
                prm, size = [0.0, 0.0, 0.0], np.asarray([2.0 * 1.5 / 1.2])   # zero level set on local z: 1.2 |z|/1.5 = 2
            centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, rng.uniform(0.6, 1.0, 1), rng.uniform(0, 6.28, 1))
            Rk = O.quat_to_rot(np.asarray(q[0], dtype=np.float64))
            if itype in (O.IND_BOX, O.IND_CAPSULE):                 # tilt by ~0.1 / 0.5 rad about a local x
                a = 0.1 if itype == O.IND_BOX else 0.5
                Rk = Rk @ np.array([[1, 0, 0], [0, math.cos(a), -math.sin(a)], [0, math.sin(a), math.cos(a)]])
            R = Rp[e, p] @ Rk                                       # carried along by the patch's pose
            t = Rp[e, p] @ centre[0] + ppose[e, p, 0:3]
            ind[e, k]["type"], ind[e, k]["param"] = itype, prm
            ind[e, k]["pose"][0:3], ind[e, k]["pose"][3:7] = t, W.quat_from_matrix(R)
    ind["pose"] = ind["pose"].astype(np.float32).astype(np.float64)
    ppose = ppose.astype(np.float32).astype(np.float64)
    wl = W.Workload("pose_grad_case", mesh, np.asarray([0.45, 0.7], np.float32), W.make_weights(9, 1, std=0.3), E, M, ind, ppose, "fp32",
                    {"grids": {0: (gvals, (-4.13, -3.87, -5.06), 0.5)}})
    return wl, rng.normal(0, 0.2, (E, mesh.n_nodes, 3))


def test_sdf_gradients_against_central_differences_of_the_sdfs():
    """grad phi of every indenter type (the building block of the pose gradients), inside, outside and -- capsule,
    grid -- beyond the ends / the box: central differences of the pinned SDFs; |grad| = 1 for the exact ones."""
    from oracle import etac_oracle_grad as OG
    rng = np.random.default_rng(3)
    y = rng.uniform(-5, 5, (400, 3))
    h = 1e-6
    cases = [(O.IND_SPHERE, [2.5, 0, 0]), (O.IND_BOX, [2.0, 3.0, 1.5]), (O.IND_CAPSULE, [1.5, 2.0, 0])]
    for itype, prm in cases:
        g = OG.sdf_local_gradient(itype, np.asarray(prm), y)
        for a in range(3):
            e = np.zeros(3)
            e[a] = h
            fd = (O.sdf_local(itype, prm, *(y + e).T) - O.sdf_local(itype, prm, *(y - e).T)) / (2 * h)
            assert np.abs(fd - g[:, a]).max() < 1e-8, (itype, a)
        np.testing.assert_allclose(np.linalg.norm(g, axis=1), 1.0, atol=1e-12)
        assert (O.sdf_local(itype, prm, *y.T) < 0).sum() > 10       # the sample has points inside (where contact is)
    vals, _ = _grid_of(lambda X, Y, Z: np.sqrt(X ** 2 + (Y / 1.5) ** 2 + Z ** 2) - 1.5)
    origin, sp = (-2.0, -2.5, -3.0), 0.5
    g = OG.sdf_grid_gradient(vals, origin, sp, y)                   # many of these points are outside the grid's box
    for a in range(3):
        e = np.zeros(3)
        e[a] = h
        fd = (O.sdf_grid(vals, origin, sp, *(y + e).T) - O.sdf_grid(vals, origin, sp, *(y - e).T)) / (2 * h)
        cell = ((y[:, a] - origin[a]) / sp) % 1.0                   # away from the interpolant's kinks along this axis
        hi = origin[a] + sp * (vals.shape[2 - a] - 1)
        ok = (np.minimum(cell, 1 - cell) > 1e-4) & (np.abs(y[:, a] - origin[a]) > 1e-4) & (np.abs(y[:, a] - hi) > 1e-4)
        assert ok.sum() > 350 and np.abs(fd - g[:, a])[ok].max() < 1e-7, a


def test_pose_gradient_oracle_matches_finite_differences():
    """pose_gradients against its definition: central differences of the (pinned) forward oracle's loss under a
    translation of / a small left rotation about each world axis of every indenter's and every patch's pose, with
    all four indenter types in contact (the contact set must not change under the perturbation: checked)."""
    import dataclasses
    from oracle import etac_oracle_grad as OG
    wl, target = pose_grad_case()
    m = O.model_from_workload(wl, resid_arch="pernode")

    def loss(ind, ppose):
        r = O.step(m, indenters=ind, patch_pose=ppose)
        return 0.5 * float(((r["U"] - target) ** 2).sum()), r
    l0, r0 = loss(wl.indenters, wl.patch_pose)
    g_delta = OG.backward(m, r0["U"] - target, indenters=wl.indenters, patch_pose=wl.patch_pose)["delta"]
    pg = OG.pose_gradients(m, g_delta, wl.indenters, wl.patch_pose)
    # every indenter type is in contact in every env, on its own nodes
    for e in range(wl.n_envs):
        for k in range(4):
            solo = wl.indenters[e:e + 1].copy()
            solo["type"][0, [j for j in range(4) if j != k]] = O.IND_NONE
            assert O.step(m, indenters=solo, patch_pose=wl.patch_pose[e:e + 1])["mask"].sum() >= 3, (e, k)
    eps = 1e-6
    noise = 8 * np.finfo(np.float64).eps * abs(l0) / eps
    worst = 0.0
    for e in range(wl.n_envs):
        for kind, count in (("indenter", 4), ("patch", 2)):
            for k in range(count):
                for dof in range(6):
                    vals = []
                    for s in (+1, -1):
                        ind, pp = wl.indenters.copy(), wl.patch_pose.copy()
                        if kind == "indenter":
                            ind[e, k]["pose"] = _perturb_pose(ind[e, k]["pose"], dof, s * eps)
                        else:
                            pp[e, k] = _perturb_pose(pp[e, k], dof, s * eps)
                        l, r = loss(ind, pp)
                        assert np.array_equal(r["mask"], r0["mask"])
                        vals.append(l)
                    fd = (vals[0] - vals[1]) / (2 * eps)
                    got = pg[kind][e, k, dof]
                    worst = max(worst, abs(fd - got) / max(1.0, abs(fd)))
                    assert abs(fd - got) <= 2e-6 * max(1.0, abs(fd)) + noise, (e, kind, k, dof, fd, got)
    assert np.abs(pg["indenter"]).min(axis=(0, 2)).max() > 0 and (np.abs(pg["indenter"]).max(axis=2) > 1e-2).all()
    assert (np.abs(pg["patch"]).max(axis=2) > 1e-2).all()
    # a rigid motion of the whole scene changes nothing: the gradients of an env sum to zero force, and to zero torque
    # about the world origin (torques are about each body's own origin: shift them by t x force)
    for e in range(wl.n_envs):
        f = pg["indenter"][e, :, 0:3].sum(0) + pg["patch"][e, :, 0:3].sum(0)
        tq = pg["indenter"][e, :, 3:6].sum(0) + pg["patch"][e, :, 3:6].sum(0)
        tq = tq + sum(np.cross(wl.indenters[e, k]["pose"][0:3], pg["indenter"][e, k, 0:3]) for k in range(4))
        tq = tq + sum(np.cross(wl.patch_pose[e, p, 0:3], pg["patch"][e, p, 0:3]) for p in range(2))
        scale = np.abs(pg["indenter"][e]).max()
        assert np.abs(f).max() < 1e-9 * scale and np.abs(tq).max() < 1e-7 * scale, (f, tq)
    print(f"[pose grad pin] worst relative FD mismatch {worst:.2e}")
