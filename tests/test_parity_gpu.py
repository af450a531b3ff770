"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerances are BASELINE.json's:
   masks / contact decisions : bit-exact
   fp32 path                 : max|u_gpu - u_ref| <= 1e-4 * max|u_ref|
   bf16 tensor-core path     : max|u_gpu - u_ref| <= 2e-2 * max|u_ref|   (fp32 accumulation)
The residual MLP is ~1 % of max|u| with the N(0, 0.02) weights of the configs, so it is also
checked on its own (r = U - u_lin on passive nodes) and with larger weights."""
import ctypes as C

import numpy as np
import pytest

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W
from parity_util import TOL, compare, random_case, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _report(name, st):
    print(f"[parity] {name}: " + " ".join(f"{k}={v:.3e}" for k, v in st.items()))


@pytest.mark.parametrize("seed,n_envs", [(0, 1), (1, 5)])
def test_config1_fp32(seed, n_envs):
    wl = W.config1(seed, n_envs)
    gpu, ref = run_gpu(wl), run_oracle(wl)
    assert gpu["path"] == T.ETAC_PATH_SPARSE and gpu["launches"] == 2
    _report("cfg1", compare(gpu, ref, TOL["fp32"], resid_tol=1e-4, label="cfg1"))


def test_config2_fp32():
    wl = W.config2(0, 64)
    gpu, ref = run_gpu(wl), run_oracle(wl)
    _report("cfg2", compare(gpu, ref, TOL["fp32"], resid_tol=1e-4, label="cfg2"))
    assert gpu["pairs"] == int(ref["contact"].sum())


@pytest.mark.parametrize("n_envs", [40, 97])
def test_config3_bf16_dense_small(n_envs):
    wl = W.config3(1, n_envs)      # 40: one ragged env tile per patch; 97: several tiles + tail
    gpu, ref = run_gpu(wl), run_oracle(wl)
    assert gpu["path"] == T.ETAC_PATH_DENSE
    _report(f"cfg3 E={n_envs}", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="cfg3"))
    assert gpu["pairs"] == int(ref["contact"].sum())


def test_config3_sparse_paths():
    """Omega U_a as a gather over the active nodes: the fp32 SIMT kernel of an fp32 context at the
    fp32 tolerance, and the bf16-K / tensor-core-MLP form of a bf16 context at the bf16 tolerance."""
    wl = W.config3(2, 24)
    ref = run_oracle(wl)
    gpu = run_gpu(wl, path=T.ETAC_PATH_SPARSE, precision="fp32")
    _report("cfg3 sparse fp32", compare(gpu, ref, TOL["fp32"], resid_tol=1e-4, label="cfg3-sparse"))
    wl = W.config3(2, 97)          # several env tiles per patch + a ragged one
    gpu = run_gpu(wl, path=T.ETAC_PATH_SPARSE)
    assert gpu["path"] == T.ETAC_PATH_SPARSE and gpu["launches"] == 3      # S1 (cull, evaluate), fused
    _report("cfg3 sparse bf16", compare(gpu, run_oracle(wl), TOL["bf16"], resid_tol=5e-2, label="cfg3-sparse16"))


def test_config4_bf16_dense_small():
    wl = W.config4(0, 12)          # N = 8192: 64 node blocks x 128 k-blocks per env tile
    gpu, ref = run_gpu(wl), run_oracle(wl)
    _report("cfg4", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="cfg4"))


def test_large_weights_bf16_mlp():
    """With N(0, 0.3) weights the residual is comparable to u_lin: a wrong MLP cannot hide."""
    wl = W.config3(3, 33)
    wl.weights = W.make_weights(3, seed=9, std=0.3)
    gpu, ref = run_gpu(wl), run_oracle(wl)
    st = compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="large-w")
    _report("large weights", st)
    r = np.abs(ref["U"] - ref["analytic"])[~ref["mask"]].max()
    assert r > 0.05 * st["umax"]


def test_large_weights_fp32_mlp():
    wl = W.config2(4, 16)
    wl.weights = W.make_weights(2, seed=9, std=0.3)
    _report("large weights fp32", compare(run_gpu(wl), run_oracle(wl), TOL["fp32"], resid_tol=1e-4, label="large-w32"))


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_penetration_input_mode(precision):
    wl = W.config2(5, 9)
    rng = np.random.default_rng(3)
    pen = np.where(rng.random((9, 1024)) < 0.03, rng.uniform(-0.5, 1.5, (9, 1024)), 0).astype(np.float32)
    pen[4] = 0.0                                   # one env without contact
    pen[5] = -1.0                                  # negatives clamp to zero (R19)
    gpu = run_gpu(wl, precision=precision, penetration=pen)
    ref = run_oracle(wl, penetration=pen)
    _report(f"penetration {precision}", compare(gpu, ref, TOL[precision], label="pen"))
    assert np.all(gpu["U"][4] == 0) and np.all(gpu["U"][5] == 0)


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_modes_no_residual_and_propagate(precision):
    wl = W.config3(6, 17)
    gpu = run_gpu(wl, precision=precision, resid=False)
    ref = run_oracle(wl, resid=False)
    compare(gpu, ref, TOL[precision], label="no-resid")
    passive = ~ref["mask"]
    assert np.array_equal(gpu["U"][passive], gpu["analytic"][passive])     # "linear decay only" (L137)
    gpu = run_gpu(wl, precision=precision, active_mode=T.ETAC_ACTIVE_PROPAGATE)
    compare(gpu, run_oracle(wl, active_mode="propagate"), TOL[precision], label="propagate")


def test_zero_contact_and_edge_sizes():
    wl = W.config2(7, 6)
    wl.indenters["pose"][..., 0:3] += 500.0
    for precision in ("fp32", "bf16"):
        gpu = run_gpu(wl, precision=precision)
        assert not gpu["mask"].any() and np.all(gpu["U"] == 0) and np.all(gpu["analytic"] == 0)
        assert gpu["pairs"] == 0
    wl = W.config2(7, 6)
    # n_envs < max_envs, and the step is stateless: running twice gives the same answer
    ref = run_oracle(wl, envs=range(3))
    for precision in ("fp32", "bf16"):
        gpu = run_gpu(wl, precision=precision, max_envs=64, n_envs=3, steps=2)
        compare(gpu, ref, TOL[precision], label="partial")


def test_ragged_patches_bf16_and_fp32():
    """Patch sizes that are not multiples of the 128-node tile or the 64-wide k-block, patch
    offsets not multiples of 32 (mask words shared by two patches), per-patch alpha."""
    parts = [W.flat_pad(10, 20, 1.0), W.fib_cap(6.0, 72), W.half_cylinder(5.0, 12.0, 9, 15)]   # 200, 72, 135
    mesh = W.assemble(parts)
    rng = np.random.default_rng(12)
    E = 37
    pen = np.where(rng.random((E, mesh.n_nodes)) < 0.05, rng.uniform(0.05, 1.0, (E, mesh.n_nodes)), 0).astype(np.float32)
    pen[3, :200] = 0
    pen[9] = 0
    wl = W.Workload("ragged", mesh, np.float32([0.5, 0.8, 0.3]), W.make_weights(7, 1, std=0.1), E, 0,
                    np.zeros((E, 0), dtype=W.INDENTER_DTYPE), None, "bf16")
    ref = run_oracle(wl, penetration=pen)
    _report("ragged bf16", compare(run_gpu(wl, penetration=pen), ref, TOL["bf16"], resid_tol=5e-2, label="ragged"))
    _report("ragged fp32", compare(run_gpu(wl, precision="fp32", penetration=pen), ref, TOL["fp32"], resid_tol=1e-4,
                                   label="ragged32"))


def test_patches_derived_from_adjacency_on_device():
    wl = W.config3(8, 4)
    import torch
    ctx = T.etac_create(wl.mesh.pos, wl.mesh.normal, wl.alpha, adj_rowptr=wl.mesh.adj_rowptr,
                        adj_col=wl.mesh.adj_col, weights=wl.weights, max_envs=4, precision=T.ETAC_PREC_BF16)
    assert T.etac_get_info(ctx, T.ETAC_INFO_N_PATCHES) == 16 and T.etac_get_info(ctx, T.ETAC_INFO_N_NODES) == 5696
    out = torch.empty((5, 5696, 3), device="cuda")
    with pytest.raises(T.EtacError) as ei:
        T.etac_step(ctx, None, T.make_step_args(5, out, indenters=out))
    assert ei.value.status == T.ETAC_ERR_CAPACITY
    with pytest.raises(T.EtacError) as ei:
        T.etac_step(ctx, None, T.make_step_args(4, None, indenters=out))
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG
    for bad in (dict(out_dtype=2), dict(out_env_stride=3 * 5696 - 1), dict(out_env_stride=-1)):
        with pytest.raises(T.EtacError) as ei:
            T.etac_step(ctx, None, T.make_step_args(4, out, indenters=out, **bad))
        assert ei.value.status == T.ETAC_ERR_INVALID_ARG
    with pytest.raises(T.EtacError) as ei:                               # fp32 output at an odd 2-byte address
        T.etac_step(ctx, None, T.make_step_args(4, out.data_ptr() + 2, indenters=out))
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG
    with pytest.raises(T.EtacError):
        T.etac_set_option(ctx, T.ETAC_OPT_ABLATION, 4)
    T.etac_step(ctx, None, T.make_step_args(0, out, indenters=out))       # no-op
    T.etac_destroy(ctx)


def test_full_size_config3_all_envs():
    """BASELINE.json's bench configuration (4096 envs, N = 5696, bf16) in the launch
    configuration bench.py times; the oracle checks EVERY environment element by element
    ("parity is checked on all envs for configs 1-4")."""
    wl = W.config3(0, 4096)
    gpu = run_gpu(wl)
    ref = run_oracle(wl)
    _report("cfg3 full", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="cfg3-full"))
    # properties that hold at any size: contact pairs = chosen patches; un-chosen patches are 0
    assert gpu["pairs"] == int(wl.meta["chosen"].sum())
    rows = ~np.repeat(wl.meta["chosen"], np.diff(wl.mesh.patch_offset), axis=1)
    assert np.all(gpu["U"][rows] == 0.0)
    act = gpu["mask"]
    nrm = wl.mesh.normal[None]
    np.testing.assert_array_equal(gpu["U"][act], (-gpu["delta"][..., None] * nrm)[act])   # P7 on every env


def _multi_indenter_hand(seed, n_envs, n_ind, posed):
    """Hand mesh (16 patches) with several indenters per environment pressed on random nodes:
    exercises the warp-per-(env, patch) S1 kernel with M > 1 (indenters staged per warp)."""
    base = W.config3(seed, n_envs)
    mesh = base.mesh
    rng = np.random.default_rng(100 + seed)
    ind = W._blank_indenters(n_envs, n_ind)
    for k in range(n_ind):
        c = rng.integers(0, mesh.n_nodes, size=n_envs)
        shape = rng.integers(1, 4, size=n_envs)                       # sphere / box / capsule
        size = rng.uniform(2.0, 5.0, n_envs)
        d = rng.uniform(0.1, 1.2, n_envs)
        centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, d, rng.uniform(0, 6.28, n_envs))
        use = rng.random(n_envs) < 0.8
        ind["type"][:, k] = np.where(use, shape, W.IND_NONE)
        ind["param"][:, k, 0] = size
        ind["param"][:, k, 1] = np.where(shape == W.IND_CAPSULE, rng.uniform(0.0, 4.0, n_envs), size)
        ind["param"][:, k, 2] = size
        ind["pose"][use, k, 0:3] = centre[use]
        ind["pose"][use, k, 3:7] = q[use]
    pose = None
    if posed:                                                         # one rigid motion per env for all patches
        pose = np.zeros((n_envs, mesh.n_patches, 7), np.float32)
        Rm = W.random_rotations(rng, n_envs)
        t = rng.uniform(-20, 20, (n_envs, 3))
        pose[:, :, 0:3] = t[:, None, :]
        pose[:, :, 3:7] = W.quat_from_matrix(Rm)[:, None, :]
        ind["pose"][..., 0:3] = np.einsum("eij,ekj->eki", Rm, ind["pose"][..., 0:3].astype(np.float64)) + t[:, None, :]
        qi = ind["pose"][..., 3:7].astype(np.float64)
        from scipy.spatial.transform import Rotation as Rot
        for e in range(n_envs):
            ind["pose"][e, :, 3:7] = (Rot.from_matrix(Rm[e]) * Rot.from_quat(qi[e])).as_quat()
    return W.Workload("hand_multi_ind", mesh, base.alpha, base.weights, n_envs, n_ind, ind, pose, "bf16")


@pytest.mark.parametrize("posed", [False, True])
def test_many_patches_several_indenters(posed):
    wl = _multi_indenter_hand(5, 29, 3, posed)
    gpu, ref = run_gpu(wl), run_oracle(wl)
    assert gpu["mask"].any()
    _report(f"hand M=3 posed={posed}", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="hand-multi"))
    assert gpu["pairs"] == int(ref["contact"].sum())
    gpu32 = run_gpu(wl, precision="fp32")
    compare(gpu32, ref, TOL["fp32"], resid_tol=1e-4, label="hand-multi-fp32")


@pytest.mark.parametrize("n_nodes,curved,frac", [(256, False, 0.05), (1024, True, 0.20), (1024, False, 0.01),
                                                 (4096, True, 0.01), (4096, False, 0.20), (8192, True, 0.20)])
def test_config5_dense_and_sparse_paths(n_nodes, curved, frac):
    """BASELINE.json configs[4] sweep points at a size the oracle finishes in seconds: the bf16
    context through the tensor-core contraction and through the gather form, the fp32 context
    through the fp32 gather kernel."""
    wl = W.config5(48, n_nodes, curved, frac, "bf16")
    ref = run_oracle(wl)
    assert ref["mask"].any()
    dense = run_gpu(wl, path=T.ETAC_PATH_DENSE)
    # 20 % contact on the curved sheet needs spheres of r > 100 mm: ulp(r) ~ 1e-5 in fp32
    _report(f"cfg5 N={n_nodes} dense", compare(dense, ref, TOL["bf16"], resid_tol=5e-2, label="cfg5-dense", delta_tol=1e-4))
    sparse = run_gpu(wl, path=T.ETAC_PATH_SPARSE)
    assert sparse["path"] == T.ETAC_PATH_SPARSE
    _report(f"cfg5 N={n_nodes} sparse bf16", compare(sparse, ref, TOL["bf16"], resid_tol=5e-2, label="cfg5-sparse16", delta_tol=1e-4))
    sparse32 = run_gpu(wl, path=T.ETAC_PATH_SPARSE, precision="fp32")
    _report(f"cfg5 N={n_nodes} sparse fp32", compare(sparse32, ref, TOL["fp32"], resid_tol=1e-4, label="cfg5-sparse32", delta_tol=1e-4))


def test_fp32_context_large_batch_all_envs():
    """An fp32 context beyond toy batch sizes (cfg-5 point N = 1024 curved, 5 %, E = 1024; the fp32 gather
    kernel's grid covers every (chunk, env)): every environment against the oracle at the fp32 tolerance."""
    wl = W.config5(1024, 1024, True, 0.05, "fp32")
    gpu, ref = run_gpu(wl), run_oracle(wl)
    assert gpu["path"] == T.ETAC_PATH_SPARSE
    _report("cfg5 fp32 E=1024", compare(gpu, ref, TOL["fp32"], resid_tol=1e-4, label="cfg5-fp32-1024", delta_tol=1e-4))


@pytest.mark.parametrize("frac", [0.01, 0.2])
def test_fp32_large_patch_shared_and_overflowing_active_lists(frac):
    """fp32 context, one patch of 8192 nodes, enough environments for the gather kernel to take several chunks of a
    patch per work item: at 1 % contact the chunks of an item share ONE compacted list of the patch's active nodes,
    at 20 % (about 1300 active nodes per environment) the list exceeds the cache and every chunk scans for itself.
    Sampled environments against the oracle at the fp32 tolerance; every row of every environment finite."""
    wl = W.config5(192, 8192, True, frac, "fp32")
    envs = [0, 1, 95, 191]
    gpu, ref = run_gpu(wl), run_oracle(wl, envs=envs)
    n_act = ref["mask"].sum(1)
    assert (n_act.max() > 1024) == (frac == 0.2) and n_act.min() > 0
    _report(f"cfg5 N=8192 fp32 frac={frac}", compare(gpu, ref, TOL["fp32"], envs=envs, resid_tol=1e-4, label="fp32-lists", delta_tol=1e-4))
    assert np.isfinite(gpu["U"]).all()


def test_full_size_config4_strided():
    """BASELINE.json configs[3] at full size (4096 envs, one dense K[8192 x 8192], bf16); the
    oracle checks every 16th environment (256 of them, so that every CTA's env tiles are hit) element by
    element; invariants hold on every environment."""
    wl = W.config4(0, 4096)
    import torch
    eng = T.Etac(wl, debug_outputs=False)
    try:
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        eng.out.fill_(float("nan"))
        U = eng.step(wl.n_envs, dev)
        torch.cuda.synchronize()
        envs = list(range(7, 4096, 16))
        ref = run_oracle(wl, envs=envs)
        Us = U[envs].cpu().numpy()
        umax = float(np.abs(ref["U"]).max())
        err = float(np.abs(Us - ref["U"]).max())
        print(f"[parity] cfg4 full: umax={umax:.3e} err={err:.3e} rel={err / umax:.3e}")
        assert err <= TOL["bf16"] * umax
        # active rows keep u^ = -delta n exactly (P7) on the sampled envs; everything finite everywhere
        act = ref["mask"]
        np.testing.assert_array_equal(Us[act], (-ref["delta32"][..., None] * wl.mesh.normal[None])[act])
        assert bool(torch.isfinite(U).all())
        assert T.etac_get_info(eng.ctx, T.ETAC_INFO_LAST_CONTACT_PAIRS) == int((np.abs(U.cpu().numpy()).sum((1, 2)) > 0).sum())
    finally:
        eng.close()


@pytest.mark.parametrize("n_envs,path", [(29, T.ETAC_PATH_DENSE), (97, T.ETAC_PATH_DENSE), (40, T.ETAC_PATH_SPARSE)])
def test_pointnet_residual_bf16(n_envs, path):
    """The paper's form of Phi: per-node encoder, max-pool over the patch,
    global MLP, decoder on [f_i; g'] -- two passes of the fused kernel against the oracle's
    residual_pointnet.  N(0, 0.15) weights so that the residual and its global part matter."""
    import dataclasses
    wl = dataclasses.replace(W.config3(4, n_envs), weights=W.make_pointnet_weights(3, 1, std=0.15))
    gpu, ref = run_gpu(wl, path=path), run_oracle(wl)
    assert gpu["launches"] == 5                      # S1 (cull, evaluate), encode + pool, global MLP, decode
    st = compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="pointnet")
    _report(f"pointnet E={n_envs}", st)
    # the global feature matters: with g' removed (per-node part only) the residual is different
    assert float(np.abs(ref["U"] - ref["analytic"]).max()) > 1e-2 * float(np.abs(ref["U"]).max())


@pytest.mark.parametrize("mesh_kind,n_envs", [("hand", 29), ("cap", 12)])
def test_pointnet_residual_fp32(mesh_kind, n_envs):
    """The paper's form of Phi on an fp32 context (k_pointnet_fp32.cu: fp32 SIMT, exact expf) at the fp32
    tolerance, on the hand mesh (16 patches) and on a single cap; N(0, 0.15) weights so that the residual and its
    global part matter; also its "Residual Network Only" and "Linear Decay Only" modes."""
    import dataclasses
    from oracle import etac_oracle as O
    base = W.config3(4, n_envs) if mesh_kind == "hand" else W.config2(4, n_envs)
    wl = dataclasses.replace(base, weights=W.make_pointnet_weights(3, 1, std=0.15))
    gpu, ref = run_gpu(wl, precision="fp32"), run_oracle(wl)
    assert gpu["launches"] == (5 if mesh_kind == "hand" else 4)     # S1 (hand: cull + evaluate), encode, global MLP, decode
    _report(f"pointnet fp32 {mesh_kind}", compare(gpu, ref, TOL["fp32"], resid_tol=1e-4, label="pointnet-fp32"))
    assert float(np.abs(ref["U"] - ref["analytic"]).max()) > 1e-2 * float(np.abs(ref["U"]).max())
    for mode, code in (("residual_only", T.ETAC_ABLATE_RESIDUAL_ONLY), ("linear_only", T.ETAC_ABLATE_LINEAR_ONLY)):
        m = O.model_from_workload(wl, resid_arch="pointnet")
        m.ablation = mode
        want = O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose)["U"]
        eng = T.Etac(wl, precision="fp32")
        try:
            T.etac_set_option(eng.ctx, T.ETAC_OPT_ABLATION, code)
            U = eng.step(wl.n_envs, eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)).cpu().numpy()
        finally:
            eng.close()
        assert np.abs(U - want).max() <= 1e-4 * np.abs(ref["U"]).max(), mode


def test_two_contexts_on_two_streams_are_independent():
    """include/etac.h: one in-flight stream per ctx, different ctxs are independent, a step only
    enqueues.  Two contexts (different meshes, precisions) stepped alternately on two streams
    without host synchronisation give the same results as each one alone; create/destroy loops
    leave nothing behind."""
    import torch
    wa, wb = W.config3(9, 33), W.config2(9, 21)
    ref_a, ref_b = run_gpu(wa)["U"], run_gpu(wb)["U"]
    ea, eb = T.Etac(wa), T.Etac(wb)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    da = ea.upload(indenters=wa.indenters, patch_pose=wa.patch_pose)
    db = eb.upload(indenters=wb.indenters, patch_pose=wb.patch_pose)
    torch.cuda.synchronize()
    for _ in range(5):
        with torch.cuda.stream(sa):
            ua = ea.step(wa.n_envs, da)
        with torch.cuda.stream(sb):
            ub = eb.step(wb.n_envs, db)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(ua.cpu().numpy(), ref_a)      # bit-identical: every step is stateless
    np.testing.assert_array_equal(ub.cpu().numpy(), ref_b)
    ea.close(), eb.close()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(8):
        T.Etac(wa).close()
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20)     # no leak across create/destroy


def _grid_workload(mesh_kind, n_envs, seed):
    """Objects given as SAMPLED signed-distance fields (ETAC_IND_GRID): a rounded box sampled at
    0.5 mm on a 41^3 grid, pressed on random nodes; half of the envs also get an analytic sphere."""
    rng = np.random.default_rng(300 + seed)
    base = W.config3(seed, n_envs) if mesh_kind == "hand" else W.config2(seed, n_envs)
    mesh = base.mesh
    h, n = 0.5, 41
    ax = -10.0 + h * np.arange(n)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    q = np.stack([np.abs(X) - 4.0, np.abs(Y) - 3.0, np.abs(Z) - 5.0], 0)             # box 4 x 3 x 5 ...
    vals = (np.linalg.norm(np.maximum(q, 0), axis=0) + np.minimum(q.max(0), 0) - 1.0).astype(np.float32)   # ... rounded by 1
    ind = W._blank_indenters(n_envs, 2)
    c = rng.integers(0, mesh.n_nodes, n_envs)
    d = rng.uniform(0.2, 1.4, n_envs)
    centre, quat = W._press_on_node(mesh.pos, mesh.normal, c, None, np.full(n_envs, 6.0), d, rng.uniform(0, 6.28, n_envs))
    ind["type"][:, 0] = T.ETAC_IND_GRID
    ind["param"][:, 0, 0] = 2.0                                                        # grid id
    ind["pose"][:, 0, 0:3], ind["pose"][:, 0, 3:7] = centre, quat
    c2 = rng.integers(0, mesh.n_nodes, n_envs)
    use = rng.random(n_envs) < 0.5
    cs, qs = W._press_on_node(mesh.pos, mesh.normal, c2, None, np.full(n_envs, 3.0), rng.uniform(0.1, 1.0, n_envs), np.zeros(n_envs))
    ind["type"][:, 1] = np.where(use, W.IND_SPHERE, W.IND_NONE)
    ind["param"][:, 1, 0] = 3.0
    ind["pose"][use, 1, 0:3], ind["pose"][use, 1, 3:7] = cs[use], qs[use]
    meta = {"grids": {2: (vals, (-10.0, -10.0, -10.0), h)}}
    return W.Workload("grid_sdf_" + mesh_kind, mesh, base.alpha, base.weights, n_envs, 2, ind, None, base.precision, meta)


@pytest.mark.parametrize("mesh_kind,n_envs", [("hand", 21), ("cap", 12)])
def test_sampled_sdf_grid_indenters(mesh_kind, n_envs):
    wl = _grid_workload(mesh_kind, n_envs, 1)
    gpu, ref = run_gpu(wl), run_oracle(wl)
    assert ref["mask"].any() and ref["mask"].sum() > 50
    tol = TOL[wl.precision]
    _report(f"grid sdf {mesh_kind}", compare(gpu, ref, tol, resid_tol=5e-2 if wl.precision == "bf16" else 1e-4,
                                             label="grid-sdf", delta_tol=1e-4))
    # the sampled field is close to the analytic rounded box it was sampled from (h^2 bound): the
    # penetrations differ by well under the grid spacing
    assert float(np.abs(ref["delta"]).max()) > 0.2


@pytest.mark.parametrize("shape_kind", ["box", "icosphere", "tetra"])
def test_mesh_to_sdf_grid_against_the_mesh_oracle(shape_kind):
    """etac_mesh_to_sdf_grid (objects given as triangle meshes) against oracle/etac_oracle_mesh.py on
    grids that are not cubes, with points inside, outside and close to the surface: fp32 brute force against float64,
    1e-5 of the scene's diagonal; the sign agrees wherever the point is further than that from the surface."""
    from oracle import etac_oracle_mesh as M
    V, Tr = {"box": lambda: W.box_mesh(4.0, 3.0, 5.0), "icosphere": lambda: W.icosphere(4.5, 2), "tetra": lambda: W.tetra_mesh(4.0)}[shape_kind]()
    shape, origin, h = (23, 19, 27), (-7.1, -6.3, -8.2), 0.61
    ref = M.mesh_sdf_grid(V, Tr, shape, origin, h)
    got = T.etac_mesh_to_sdf_grid(V, Tr, shape, origin, h).astype(np.float64)
    assert got.shape == ref.shape == (27, 19, 23) and (ref < 0).sum() > 200 and (ref > 0).sum() > 200
    diag = float(np.linalg.norm(np.asarray(shape) * h))
    err = float(np.abs(got - ref).max())
    print(f"[mesh grid {shape_kind}] {len(Tr)} triangles, {ref.size} points: max err {err:.3g} ({err / diag:.2e} of the diagonal)")
    assert err <= 1e-5 * diag
    far = np.abs(ref) > 1e-5 * diag
    assert np.array_equal(got[far] < 0, ref[far] < 0)
    with pytest.raises(T.EtacError):
        T.etac_mesh_to_sdf_grid(V, Tr + len(V), shape, origin, h)                    # vertex index out of range


def test_mesh_object_as_indenter_end_to_end():
    """A triangle-mesh object pressed on the fingertip cap: the GPU samples its SDF (etac_mesh_to_sdf_grid), the grid
    is registered as an ETAC_IND_GRID indenter and stepped; the oracle samples the same mesh with its own routine.
    The two grids differ by fp32 rounding (checked above), so masks may differ only where the oracle's penetration is
    below 1e-4 mm; displacements at the fp32 tolerance."""
    from oracle import etac_oracle_mesh as M
    import dataclasses
    rng = np.random.default_rng(77)
    base = W.config2(5, 10)
    mesh = base.mesh
    V, Tr = W.icosphere(5.0, 2)
    V = V * np.array([1.0, 0.8, 1.2])                                                 # an ellipsoid-like polyhedron
    shape, origin, h = (33, 29, 37), (-8.0, -7.0, -9.0), 0.5
    vals_ref = M.mesh_sdf_grid(V, Tr, shape, origin, h).astype(np.float32)
    n_envs = base.n_envs
    ind = W._blank_indenters(n_envs, 1)
    c = rng.integers(0, mesh.n_nodes, n_envs)
    centre, quat = W._press_on_node(mesh.pos, mesh.normal, c, None, np.full(n_envs, 4.0), rng.uniform(0.3, 1.2, n_envs),
                                    rng.uniform(0, 6.28, n_envs))
    ind["type"][:, 0], ind["param"][:, 0, 0] = T.ETAC_IND_GRID, 1.0
    ind["pose"][:, 0, 0:3], ind["pose"][:, 0, 3:7] = centre, quat
    wl = dataclasses.replace(base, indenters=ind, max_indenters=1, meta={"grids": {1: (vals_ref, origin, h)}})
    ref = run_oracle(wl)
    assert ref["mask"].sum() > 100
    eng = T.Etac(wl, debug_outputs=True)
    try:
        T.etac_set_sdf_grid(eng.ctx, 1, T.etac_mesh_to_sdf_grid(V, Tr, shape, origin, h), origin, h)   # the GPU-sampled field
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        U = eng.step(n_envs, dev).cpu().numpy()
        mask = eng.mask_bool(n_envs)
    finally:
        eng.close()
    differ = mask != ref["mask"]
    assert (ref["delta"][differ] < 1e-4).all() and differ.sum() <= 5
    umax = float(np.abs(ref["U"]).max())
    err = float(np.abs(U - ref["U"]).max())
    print(f"[mesh object] active nodes {int(ref['mask'].sum())}, masks differ at {int(differ.sum())}, max err {err:.3g} / {umax:.3g}")
    assert err <= 2 * TOL["fp32"] * umax                                              # two fp32 paths to the penetration


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_ablation_residual_only(precision):
    """Table II's "Residual Network Only" row as a run-time mode: passive rows get Phi_p alone."""
    import dataclasses
    from oracle import etac_oracle as O
    wl = dataclasses.replace(W.config3(11, 19), weights=W.make_weights(3, 2, std=0.2))
    m = O.model_from_workload(wl)
    m.ablation = "residual_only"
    ref = O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose)
    import torch
    eng = T.Etac(wl, precision=precision, debug_outputs=True)
    try:
        T.etac_set_option(eng.ctx, T.ETAC_OPT_ABLATION, T.ETAC_ABLATE_RESIDUAL_ONLY)
        U = eng.step(wl.n_envs, eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)).cpu().numpy()
    finally:
        eng.close()
    full = run_oracle(wl)
    assert np.abs(ref["U"] - full["U"]).max() > 0.1                      # the mode changes the answer
    tol = (1e-4 if precision == "fp32" else 5e-2) * np.abs(ref["U"][~ref["mask"]]).max()
    assert np.abs(U - ref["U"])[~ref["mask"]].max() <= tol
    np.testing.assert_allclose(U[ref["mask"]], full["U"][ref["mask"]], atol=2e-5)            # active rows keep u^


@pytest.mark.parametrize("kind,n_ind", [("hand", 1), ("hand", 3), ("few_patches", 2)])
def test_self_contact_between_links(kind, n_ind):
    """Self-contact: link collision shapes as indenters with skip_patch1, through the
    warp-per-pair S1 kernel with one and with several indenters and through the CTA-per-env kernel."""
    from parity_util import self_contact_workload
    if kind == "hand":
        wl = self_contact_workload(W.hand_mesh(), {p: 9.0 for p in range(5)}, 7, 23, n_ind)
    else:
        mesh = W.assemble([W.fib_cap(6.0, 72), W.flat_pad(10, 12, 1.0), W.fib_cap(5.0, 60)])
        wl = self_contact_workload(mesh, {0: 6.0, 2: 5.0}, 8, 17, n_ind)
    ref = run_oracle(wl)
    off = np.asarray(wl.mesh.patch_offset)
    for e in range(wl.n_envs):                                  # the skip is what keeps patch A free of its own link
        A, B = wl.meta["A"][e], wl.meta["B"][e]
        assert ref["mask"][e, off[B]:off[B + 1]].any()
        if n_ind == 1:
            assert not ref["mask"][e, off[A]:off[A + 1]].any()
    for precision in ("bf16", "fp32"):
        gpu = run_gpu(wl, precision=precision)
        _report(f"self-contact {kind} M={n_ind} {precision}",
                compare(gpu, ref, TOL[precision], resid_tol=5e-2 if precision == "bf16" else 1e-4, label="self-contact",
                        delta_tol=1e-4))       # world coordinates of a few hundred mm: ulp of the fp32 twin
        assert gpu["pairs"] == int(ref["contact"].sum())


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
@pytest.mark.parametrize("mode", ["linear_only", "no_propagation"])
def test_ablation_linear_only_and_no_propagation(precision, mode):
    """The other Table II rows as run-time modes of a context that has Phi: "Linear Decay Only"
     and the penalty displacement without propagation."""
    import dataclasses
    from oracle import etac_oracle as O
    wl = dataclasses.replace(W.config3(12, 21), weights=W.make_weights(3, 2, std=0.2))
    m = O.model_from_workload(wl)
    m.ablation = mode
    ref = O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose)
    eng = T.Etac(wl, precision=precision, debug_outputs=True)
    try:
        code = {"linear_only": T.ETAC_ABLATE_LINEAR_ONLY, "no_propagation": T.ETAC_ABLATE_NO_PROPAGATION}[mode]
        T.etac_set_option(eng.ctx, T.ETAC_OPT_ABLATION, code)
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        U = eng.step(wl.n_envs, dev).cpu().numpy()
        assert np.array_equal(eng.mask_bool(wl.n_envs), ref["mask"])
        T.etac_set_option(eng.ctx, T.ETAC_OPT_ABLATION, T.ETAC_ABLATE_FULL)      # and back
        U_full = eng.step(wl.n_envs, dev).cpu().numpy()
    finally:
        eng.close()
    full = run_oracle(wl)
    assert np.abs(ref["U"] - full["U"]).max() > 0.05                     # the mode changes the answer
    scale = np.abs(full["U"]).max()
    if mode == "no_propagation":
        assert np.all(U[~ref["mask"]] == 0)                              # nothing but the contact nodes moves
        np.testing.assert_allclose(U, ref["U"], rtol=0, atol=2e-5)
    else:
        assert np.abs(U - ref["U"]).max() <= TOL[precision] * scale
    assert np.abs(U_full - full["U"]).max() <= (5e-2 if precision == "bf16" else 1e-4) * scale


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
@pytest.mark.parametrize("path", ["dense", "sparse"])
def test_bf16_output_in_a_strided_observation_buffer(precision, path):
    """out_dtype = BF16 and out_env_stride: U lands, rounded to bf16, inside a wider per-env observation
    row (the n x 3 tensor is the policy observation); the rest of the row is untouched."""
    import torch
    if precision == "fp32" and path == "dense":
        pytest.skip("the dense contraction needs a bf16 context")
    wl = W.config3(14, 37)
    ref = run_oracle(wl)
    eng = T.Etac(wl, precision=precision)
    try:
        if path == "sparse":
            T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, T.ETAC_PATH_SPARSE)
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        N, E = eng.N, wl.n_envs
        stream = torch.cuda.current_stream().cuda_stream
        for dtype, code, pad_front, pad_back in ((torch.bfloat16, T.ETAC_OUT_BF16, 7, 5), (torch.float32, T.ETAC_OUT_F32, 3, 11)):
            stride = pad_front + 3 * N + pad_back
            obs = torch.full((E, stride), -7.0, dtype=dtype, device=eng.device)
            out = obs.data_ptr() + pad_front * obs.element_size()          # odd offsets: element alignment only
            T.etac_step(eng.ctx, stream, eng.args(E, dev, out=out, out_env_stride=stride, out_dtype=code))
            torch.cuda.synchronize()
            got = obs.float().cpu().numpy()
            assert np.all(got[:, :pad_front] == -7.0) and np.all(got[:, pad_front + 3 * N:] == -7.0)
            U = got[:, pad_front:pad_front + 3 * N].reshape(E, N, 3)
            packed = eng.step(E, dev).float().cpu().numpy()
            if dtype == torch.float32:
                assert np.array_equal(U, packed)                          # same kernels, other addresses
            else:                                                          # = the fp32 result rounded to bf16
                want = torch.from_numpy(packed).to(torch.bfloat16).float().numpy()
                assert np.array_equal(U, want)
            scale = np.abs(ref["U"]).max()
            assert np.abs(U - ref["U"]).max() <= (TOL[precision] + (2.0 ** -8 if dtype == torch.bfloat16 else 0)) * scale
    finally:
        eng.close()


def _backward_case(kind):
    import dataclasses
    if kind == "hand_bf16":
        wl = dataclasses.replace(W.config3(15, 19), weights=W.make_weights(3, 4, std=0.2))
        return wl, "bf16", T.ETAC_ACTIVE_PASSTHROUGH, True
    if kind == "pointnet_hand_bf16":
        wl = dataclasses.replace(W.config3(15, 19), weights=W.make_pointnet_weights(3, 4, std=0.12))
        return wl, "bf16", T.ETAC_ACTIVE_PASSTHROUGH, True
    mesh = W.assemble([W.fib_cap(6.0, 72), W.flat_pad(10, 20, 1.0), W.half_cylinder(5.0, 12.0, 9, 15)])   # ragged: 72, 200, 135
    rng = np.random.default_rng(31)
    E = 9
    ind = W._blank_indenters(E, 2)
    for k in range(2):
        c = rng.integers(0, mesh.n_nodes, size=E)
        size = rng.uniform(2.0, 4.0, E)
        centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, rng.uniform(0.2, 1.0, E), rng.uniform(0, 6.28, E))
        ind["type"][:, k], ind["param"][:, k, 0] = W.IND_SPHERE, size
        ind["pose"][:, k, 0:3], ind["pose"][:, k, 3:7] = centre, q
    alpha = np.asarray([0.45, 0.7, 0.55], np.float32)
    weights = W.make_pointnet_weights(9, 1, std=0.15) if kind.startswith("pointnet") else W.make_weights(9, 1, std=0.3)
    wl = W.Workload("grad_case", mesh, alpha, weights, E, 2, ind, None, "fp32")
    mode = T.ETAC_ACTIVE_PROPAGATE if kind.endswith("propagate") else T.ETAC_ACTIVE_PASSTHROUGH
    return wl, "fp32", mode, kind != "no_resid"


@pytest.mark.parametrize("kind", ["per_patch_alpha", "propagate", "no_resid", "hand_bf16", "pointnet", "pointnet_propagate",
                                  "pointnet_hand_bf16"])
def test_backward_against_the_gradient_oracle(kind):
    """etac_backward (calibration gradients of Eq. 3) against oracle/etac_oracle_grad.py
    (itself pinned by finite differences): dL/dalpha, dL/ddelta and dL/d(weights of Phi) -- the per-node MLP or the
    paper's PointNet -- for L = 0.5*||U - U*||^2.
    fp32 arithmetic, fp32 atomics across CTAs: 2e-5 of the largest entry of each tensor (measured: 1e-8 .. 6e-7)."""
    import torch
    from oracle import etac_oracle as O, etac_oracle_grad as OG
    wl, precision, mode, resid = _backward_case(kind)
    pointnet = "E1" in wl.weights
    m = O.model_from_workload(wl, resid_arch=("pointnet" if pointnet else "pernode") if resid else "none",
                              active_mode="propagate" if mode == T.ETAC_ACTIVE_PROPAGATE else "passthrough")
    U = O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose)["U"]
    G = U - np.random.default_rng(3).normal(0, 0.2, U.shape)
    ref = OG.backward(m, G, indenters=wl.indenters, patch_pose=wl.patch_pose)
    eng = T.Etac(wl, precision=precision, active_mode=mode, resid=resid)
    try:
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        d_G = torch.from_numpy(G.astype(np.float32)).to(eng.device)
        g_alpha = torch.full((len(wl.alpha),), 7.0, device=eng.device)
        n_w = T.ETAC_GRAD_WEIGHTS_POINTNET_LEN if pointnet else T.ETAC_GRAD_WEIGHTS_LEN
        g_w = torch.full((n_w,), 7.0, device=eng.device) if resid else None
        g_pen = torch.full((wl.n_envs, eng.N), 7.0, device=eng.device)
        stream = torch.cuda.current_stream().cuda_stream
        for _ in range(2):                                                # the outputs are overwritten, not accumulated
            T.etac_backward(eng.ctx, stream, wl.n_envs, d_G, g_alpha, g_w, grad_penetration=g_pen, **dev)
        torch.cuda.synchronize()
        got = {"alpha": g_alpha.cpu().numpy().astype(np.float64), "delta": g_pen.cpu().numpy().astype(np.float64)}
        if resid:
            got.update({k: v.astype(np.float64) for k, v in T.split_grad_weights(g_w.cpu().numpy()).items()})
        U_fwd = eng.step(wl.n_envs, dev).cpu().numpy()                    # the forward still works afterwards
    finally:
        eng.close()
    assert set(got) == set(ref)
    for k in ref:
        scale = np.abs(ref[k]).max()
        assert scale > 1e-4, k
        err = np.abs(got[k] - ref[k]).max()
        print(f"[backward {kind}] {k}: max|ref| {scale:.4g} max err {err:.3g} ({err / scale:.2e} rel)")
        assert err <= 2e-5 * scale, (k, err, scale)
    assert np.abs(U_fwd - U).max() <= (2e-2 if precision == "bf16" else 1e-4) * np.abs(U).max()


@pytest.mark.parametrize("resid_arch", ["pernode", "pointnet"])
def test_backward_pose_gradients_against_the_oracle(resid_arch):
    """etac_backward's dL/d(indenter poses) and dL/d(patch poses) (k_backward_pose.cu) against
    oracle/etac_oracle_grad.pose_gradients (pinned by central differences of the forward oracle): two patches under
    their own poses, sphere + tilted box + capsule + sampled grid in contact in every env; rows (dL/dt, dL/dtheta).
    fp32 with atomics: 2e-5 of the largest entry of each tensor, forces and torques apart (measured 7e-8 .. 6e-7)."""
    import dataclasses
    import torch
    from oracle import etac_oracle as O, etac_oracle_grad as OG
    from test_oracle_pins import pose_grad_case
    wl64, target = pose_grad_case(seed=92, n_envs=5)
    if resid_arch == "pointnet":
        wl64 = dataclasses.replace(wl64, weights=W.make_pointnet_weights(9, 1, std=0.2))
    m = O.model_from_workload(wl64, resid_arch=resid_arch)
    U = O.step(m, indenters=wl64.indenters, patch_pose=wl64.patch_pose)["U"]
    G = U - target
    g_delta = OG.backward(m, G, indenters=wl64.indenters, patch_pose=wl64.patch_pose)["delta"]
    ref = OG.pose_gradients(m, g_delta, wl64.indenters, wl64.patch_pose)
    ind = np.zeros(wl64.indenters.shape, dtype=W.INDENTER_DTYPE)             # the same numbers (fp32-representable) in the ABI's layout
    for f in ("type", "param", "pose", "skip_patch1"):
        ind[f] = wl64.indenters[f]
    wl = dataclasses.replace(wl64, indenters=ind, patch_pose=wl64.patch_pose.astype(np.float32))
    eng = T.Etac(wl, precision="fp32")
    try:
        dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
        d_G = torch.from_numpy(G.astype(np.float32)).to(eng.device)
        g_alpha = torch.empty(len(wl.alpha), device=eng.device)
        g_pen = torch.empty((wl.n_envs, eng.N), device=eng.device)
        g_ind = torch.full((wl.n_envs, wl.max_indenters, 6), 7.0, device=eng.device)
        g_patch = torch.full((wl.n_envs, eng.P, 6), 7.0, device=eng.device)
        stream = torch.cuda.current_stream().cuda_stream
        for _ in range(2):                                                    # overwritten, not accumulated
            T.etac_backward(eng.ctx, stream, wl.n_envs, d_G, g_alpha, None, grad_penetration=g_pen, grad_indenter_pose=g_ind,
                            grad_patch_pose=g_patch, **dev)
        torch.cuda.synchronize()
        got = {"indenter": g_ind.cpu().numpy().astype(np.float64), "patch": g_patch.cpu().numpy().astype(np.float64)}
        with pytest.raises(T.EtacError):                                      # needs dL/ddelta
            T.etac_backward(eng.ctx, stream, wl.n_envs, d_G, g_alpha, None, grad_indenter_pose=g_ind, **dev)
        with pytest.raises(T.EtacError):                                      # no poses in penetration input mode
            T.etac_backward(eng.ctx, stream, wl.n_envs, d_G, g_alpha, None, grad_penetration=g_pen, grad_patch_pose=g_patch,
                            penetration=g_pen)
        # without patch poses: the patch part is zero, the indenter part is that of identity poses
        ind_only = eng.upload(indenters=wl.indenters)
        T.etac_backward(eng.ctx, stream, wl.n_envs, d_G, g_alpha, None, grad_penetration=g_pen, grad_indenter_pose=g_ind,
                        grad_patch_pose=g_patch, **ind_only)
        torch.cuda.synchronize()
        assert not g_patch.any()
    finally:
        eng.close()
    for k in ("indenter", "patch"):
        for part, sl in (("force", slice(0, 3)), ("torque", slice(3, 6))):
            scale = np.abs(ref[k][..., sl]).max()
            err = np.abs(got[k][..., sl] - ref[k][..., sl]).max()
            print(f"[backward pose {resid_arch}] {k} {part}: max|ref| {scale:.4g} max err {err:.3g} ({err / scale:.2e} rel)")
            assert scale > 1e-2 and err <= 2e-5 * scale, (k, part, err, scale)
    assert ((np.abs(ref["indenter"]).max(axis=2) > 0).sum(axis=0) >= 4).all()  # every indenter type is in contact in >= 4 of 5 envs


@pytest.mark.parametrize("first_seed", [0, 40, 80])
def test_randomised_parity_sweep(first_seed):
    """40 seeded random workloads per parameter (parity_util.random_case: patch counts and sizes incl. the large-patch
    path, env counts over several tiles, indenter types, poses, both forms of Phi or none, both precisions, dense and
    gather paths, both active-row modes), two steps each on one context, against the oracle at the usual tolerances."""
    for seed in range(first_seed, first_seed + 40):
        wl, arch, prec, path, mode = random_case(seed)
        resid = arch != "none"
        gpu = run_gpu(wl, precision=prec, path=path, resid=resid, active_mode=mode, steps=2)
        ref = run_oracle(wl, resid=resid, active_mode="propagate" if mode == T.ETAC_ACTIVE_PROPAGATE else "passthrough")
        label = f"random{seed} sizes {np.diff(wl.mesh.patch_offset).tolist()} E {wl.n_envs} {arch} {prec} path {path} mode {mode}"
        if np.abs(ref["U"]).max() == 0:
            assert not gpu["U"].any(), label
            continue
        compare(gpu, ref, TOL[prec], label=label, delta_tol=1e-4)


@pytest.mark.parametrize("seeds", [range(0, 25), (134, 163, 169)])
def test_results_do_not_depend_on_batch_size_or_output_layout(seeds):
    """On random workloads (parity_util.random_case; the three single seeds are fp32 contexts whose batch size switches
    the gather kernel between shared and per-chunk active lists): the first E' < E environments stepped alone give the
    bits they give inside the full batch, on a context with spare max_envs; the bf16 / strided outputs are the fp32
    result rounded / moved, and the padding of the observation rows is untouched."""
    import torch
    for seed in seeds:
        wl, arch, prec, path, mode = random_case(seed)
        rng = np.random.default_rng(seed + 99)
        E = wl.n_envs
        E_run = int(rng.integers(1, E + 1))
        eng = T.Etac(wl, precision=prec, active_mode=mode, resid=arch != "none", max_envs=E + int(rng.integers(0, 9)))
        try:
            T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, path)
            dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
            stream = torch.cuda.current_stream().cuda_stream
            full = eng.step(E, dev).clone()
            part = eng.step(E_run, dev).clone()
            assert torch.equal(part, full[:E_run]), (seed, prec, E, E_run, float((part - full[:E_run]).abs().max()))
            N = eng.N
            for dtype, code in ((torch.bfloat16, T.ETAC_OUT_BF16), (torch.float32, T.ETAC_OUT_F32)):
                pf, pb = int(rng.integers(0, 9)), int(rng.integers(0, 9))
                stride = pf + 3 * N + pb
                obs = torch.full((E, stride), -7.0, dtype=dtype, device=eng.device)
                out = obs.data_ptr() + pf * obs.element_size()
                T.etac_step(eng.ctx, stream, eng.args(E, dev, out=out, out_env_stride=stride, out_dtype=code))
                torch.cuda.synchronize()
                got = obs.float()
                assert bool((got[:, :pf] == -7.0).all()) and bool((got[:, pf + 3 * N:] == -7.0).all()), (seed, "padding")
                want = full if dtype == torch.float32 else full.to(torch.bfloat16).float()
                assert torch.equal(got[:, pf:pf + 3 * N].reshape(E, N, 3), want), (seed, str(dtype))
        finally:
            eng.close()


def test_randomised_penetration_sweep():
    """Penetration input mode on 60 random workloads: random per-node penetrations with 0 / 0.2 / 2 / 20 / 90 % of the
    nodes in contact (negatives clamp; sometimes an env without contact), against the oracle."""
    for seed in range(60):
        wl, arch, prec, path, mode = random_case(seed)
        rng = np.random.default_rng(seed + 31)
        E, N = min(wl.n_envs, 40), wl.mesh.n_nodes
        frac = rng.choice([0.0, 0.002, 0.02, 0.2, 0.9])
        pen = np.where(rng.random((E, N)) < frac, rng.uniform(0.0, 1.2, (E, N)), rng.uniform(-1.0, 0.0, (E, N))).astype(np.float32)
        if rng.random() < 0.3:
            pen[rng.integers(0, E)] = -0.5
        resid = arch != "none"
        gpu = run_gpu(wl, precision=prec, path=path, resid=resid, active_mode=mode, penetration=pen, n_envs=E)
        ref = run_oracle(wl, resid=resid, active_mode="propagate" if mode == T.ETAC_ACTIVE_PROPAGATE else "passthrough", penetration=pen)
        label = f"random{seed} sizes {np.diff(wl.mesh.patch_offset).tolist()} E {E} frac {frac} {arch} {prec} path {path} mode {mode}"
        if np.abs(ref["U"]).max() == 0:
            assert not gpu["U"].any(), label
            continue
        compare(gpu, ref, TOL[prec], label=label, delta_tol=1e-4)


def test_randomised_workspace_reuse():
    """60 random workloads: input set A, then set B (the envs in another order, 30 % of the indenters gone, fewer envs)
    on ONE context gives the bits of B on a fresh context -- nothing of A survives in the per-step workspaces."""
    import torch
    for seed in range(60):
        wl, arch, prec, path, mode = random_case(seed)
        rng = np.random.default_rng(seed + 7)
        E = wl.n_envs
        perm = rng.permutation(E)
        E_b = int(rng.integers(1, E + 1))
        ind_b = wl.indenters[perm].copy()
        ind_b["type"][rng.random(ind_b.shape) < 0.3] = 0
        pose_b = None if wl.patch_pose is None else wl.patch_pose[perm].copy()

        def run(first_a):
            eng = T.Etac(wl, precision=prec, active_mode=mode, resid=arch != "none")
            try:
                T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, path)
                if first_a:
                    eng.step(E, eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose))
                return eng.step(E_b, eng.upload(indenters=ind_b, patch_pose=pose_b)).clone()
            finally:
                eng.close()
        assert torch.equal(run(False), run(True)), (seed, arch, prec, path, mode)


def test_randomised_backward_sweep():
    """etac_backward incl. the pose gradients on the random workloads of modest size (<= 1500 nodes, <= 12 envs) among the
    first 300 seeds, against the gradient oracle: 1e-4 of the largest entry of every tensor."""
    import torch
    from oracle import etac_oracle as O, etac_oracle_grad as OG
    n = 0
    for seed in range(300):
        wl, arch, prec, path, mode = random_case(seed)
        if wl.mesh.n_nodes > 1500 or wl.n_envs > 12:
            continue
        m = O.model_from_workload(wl, resid_arch=arch, active_mode="propagate" if mode == T.ETAC_ACTIVE_PROPAGATE else "passthrough")
        U = O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose)["U"]
        if np.abs(U).max() == 0:
            continue
        G = U - np.random.default_rng(seed).normal(0, 0.2, U.shape)
        ref = dict(OG.backward(m, G, indenters=wl.indenters, patch_pose=wl.patch_pose))
        ref.update(OG.pose_gradients(m, ref["delta"], wl.indenters, wl.patch_pose))
        eng = T.Etac(wl, precision=prec, active_mode=mode, resid=arch != "none")
        try:
            dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
            d_G = torch.from_numpy(G.astype(np.float32)).to(eng.device)
            g_alpha = torch.empty(len(wl.alpha), device=eng.device)
            n_w = T.ETAC_GRAD_WEIGHTS_POINTNET_LEN if arch == "pointnet" else T.ETAC_GRAD_WEIGHTS_LEN
            g_w = torch.empty(n_w, device=eng.device) if arch != "none" else None
            g_pen = torch.empty((wl.n_envs, eng.N), device=eng.device)
            g_ind = torch.empty((wl.n_envs, wl.max_indenters, 6), device=eng.device)
            g_patch = torch.empty((wl.n_envs, eng.P, 6), device=eng.device)
            T.etac_backward(eng.ctx, torch.cuda.current_stream().cuda_stream, wl.n_envs, d_G, g_alpha, g_w, grad_penetration=g_pen,
                            grad_indenter_pose=g_ind, grad_patch_pose=g_patch, **dev)
            torch.cuda.synchronize()
            got = {"alpha": g_alpha.cpu().numpy(), "delta": g_pen.cpu().numpy(), "indenter": g_ind.cpu().numpy(), "patch": g_patch.cpu().numpy()}
            if g_w is not None:
                got.update(T.split_grad_weights(g_w.cpu().numpy()))
        finally:
            eng.close()
        for k in ref:
            scale = np.abs(ref[k]).max()
            if scale < 1e-6:
                assert np.abs(got[k]).max() < 1e-4, (seed, k)
                continue
            err = np.abs(got[k].astype(np.float64) - ref[k]).max() / scale
            assert err < 1e-4, (seed, k, err, scale, arch, prec)
        n += 1
    assert n >= 15, n


def test_pose_gradients_recover_an_indenter_pose_from_a_tactile_target():
    """Differentiability end to end (Table I): the displacement field of a sphere pressed into the cap at
    a hidden position is the target; Adam on dL/dt of the indenter (etac_backward's pose gradients), starting 0.5 mm
    off (sideways and in depth), finds the position again to 1e-3 mm although the contact set changes along the way.
    ETAC_ACTIVE_PROPAGATE context: with the mask M_p of Eq. 2 a node's row jumps from the propagated value to
    u^ = -delta n ~ 0 when it enters contact, so the loss is discontinuous in the pose and a descent stalls at the jumps
    (measured on the same case: it ends 0.05-0.8 mm off); without the mask the field is continuous in delta."""
    import torch
    wl = W.config2(21, 4)
    ind = wl.indenters.copy()
    ind["type"][:, 1:] = 0                                                  # one sphere per env
    ind["type"][:, 0] = 1
    ind["param"][:, 0, 0] = 4.0
    c = np.nonzero(wl.mesh.normal[:, 2] > 0.8)[0][[3, 17, 40, 71]]
    t_star = (wl.mesh.pos[c] + wl.mesh.normal[c] * (4.0 - 0.9)).astype(np.float32)   # pressed 0.9 mm into node c
    ind["pose"][:, 0, 0:3] = t_star
    ind["pose"][:, 0, 3:7] = [0, 0, 0, 1]
    eng = T.Etac(wl, precision="fp32", active_mode=T.ETAC_ACTIVE_PROPAGATE)
    try:
        stream = torch.cuda.current_stream().cuda_stream
        target = eng.step(wl.n_envs, eng.upload(indenters=ind)).clone()
        assert float(target.abs().max()) > 0.5
        t = t_star.astype(np.float64) + np.asarray([[0.4, -0.3, 0.15], [-0.5, 0.2, 0.1], [0.3, 0.4, -0.2], [-0.2, -0.45, 0.25]])
        err0 = np.linalg.norm(t - t_star, axis=1)
        g_alpha = torch.empty(len(wl.alpha), device=eng.device)
        g_pen = torch.empty((wl.n_envs, eng.N), device=eng.device)
        g_ind = torch.empty((wl.n_envs, wl.max_indenters, 6), device=eng.device)
        m1, m2, losses = np.zeros_like(t), np.zeros_like(t), []
        for it in range(1, 201):
            ind["pose"][:, 0, 0:3] = t.astype(np.float32)
            dev = eng.upload(indenters=ind)
            G = eng.step(wl.n_envs, dev) - target
            losses.append(0.5 * float((G * G).sum()))
            T.etac_backward(eng.ctx, stream, wl.n_envs, G.contiguous(), g_alpha, None, grad_penetration=g_pen,
                            grad_indenter_pose=g_ind, **dev)
            g = g_ind[:, 0, 0:3].cpu().numpy().astype(np.float64)
            m1, m2 = 0.9 * m1 + 0.1 * g, 0.999 * m2 + 0.001 * g * g
            t = t - 0.02 * (m1 / (1 - 0.9 ** it)) / (np.sqrt(m2 / (1 - 0.999 ** it)) + 1e-12)
    finally:
        eng.close()
    err = np.linalg.norm(t - t_star, axis=1)
    print(f"[pose recovery] |t - t*| {err0.round(3)} -> {err.round(4)} mm; loss {losses[0]:.4g} -> {losses[-1]:.4g}")
    assert (err < 1e-3).all() and losses[-1] < 1e-6 * losses[0]


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_update_params_equals_a_fresh_context(precision):
    """etac_update_params (a gradient-descent step of Eq. 3 writes alpha and Phi back): the context then
    gives bit for bit what a context created with the new parameters gives."""
    import dataclasses
    wl_a = W.config3(16, 11)
    wl_b = dataclasses.replace(wl_a, alpha=np.asarray([0.8], np.float32), weights=W.make_weights(3, 9, std=0.15))
    dev_kw = dict(indenters=wl_a.indenters, patch_pose=wl_a.patch_pose)
    eng_b = T.Etac(wl_b, precision=precision)
    U_b = eng_b.step(wl_b.n_envs, eng_b.upload(**dev_kw)).cpu().numpy()
    eng_b.close()
    eng = T.Etac(wl_a, precision=precision)
    try:
        dev = eng.upload(**dev_kw)
        U_a = eng.step(wl_a.n_envs, dev).cpu().numpy()
        T.etac_update_params(eng.ctx, alpha=wl_b.alpha, weights=wl_b.weights)
        U_ab = eng.step(wl_a.n_envs, dev).cpu().numpy()
        T.etac_update_params(eng.ctx, alpha=wl_a.alpha)                      # alpha alone, back
        T.etac_update_params(eng.ctx, weights=wl_a.weights)                  # weights alone, back
        U_aa = eng.step(wl_a.n_envs, dev).cpu().numpy()
        with pytest.raises(T.EtacError):
            T.etac_update_params(eng.ctx, alpha=np.asarray([0.5, 0.6], np.float32))   # n_alpha differs
        with pytest.raises(T.EtacError):
            T.etac_update_params(eng.ctx, alpha=np.asarray([-1.0], np.float32))
    finally:
        eng.close()
    assert np.abs(U_a - U_b).max() > 1e-2
    assert np.array_equal(U_ab, U_b) and np.array_equal(U_aa, U_a)


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_update_params_pointnet_equals_a_fresh_context(precision):
    """etac_update_params on an ETAC_RESID_POINTNET context: all ten arrays of the paper's Phi
    restaged in place (bf16 image, fp32 copies, global MLP, output layer) give bit for bit the step of a context
    created with them; the per-node arrays are refused there, and the PointNet arrays on a per-node context."""
    import dataclasses
    base = W.config3(17, 11) if precision == "bf16" else W.config2(17, 11)
    wl_a = dataclasses.replace(base, weights=W.make_pointnet_weights(3, 6, std=0.15))
    wl_b = dataclasses.replace(wl_a, alpha=(base.alpha * 1.3).astype(np.float32), weights=W.make_pointnet_weights(3, 7, std=0.12))
    dev_kw = dict(indenters=wl_a.indenters, patch_pose=wl_a.patch_pose)
    eng_b = T.Etac(wl_b, precision=precision)
    U_b = eng_b.step(wl_b.n_envs, eng_b.upload(**dev_kw)).cpu().numpy()
    eng_b.close()
    eng = T.Etac(wl_a, precision=precision)
    try:
        dev = eng.upload(**dev_kw)
        U_a = eng.step(wl_a.n_envs, dev).cpu().numpy()
        T.etac_update_params(eng.ctx, alpha=wl_b.alpha, weights=wl_b.weights)
        U_ab = eng.step(wl_a.n_envs, dev).cpu().numpy()
        T.etac_update_params(eng.ctx, weights=wl_a.weights)
        T.etac_update_params(eng.ctx, alpha=wl_a.alpha)
        U_aa = eng.step(wl_a.n_envs, dev).cpu().numpy()
        with pytest.raises(T.EtacError) as ei:
            T.etac_update_params(eng.ctx, weights=W.make_weights(3, 9))      # per-node arrays on a PointNet context
        assert ei.value.status == T.ETAC_ERR_UNSUPPORTED
        part = dict(wl_b.weights)
        p = T.etac_params()
        p.struct_size = C.sizeof(T.etac_params)
        e1 = np.ascontiguousarray(part["E1"])
        p.E1 = e1.ctypes.data_as(C.POINTER(C.c_float))                       # one of ten
        assert T.load().etac_update_params(eng.ctx, C.byref(p)) == T.ETAC_ERR_INVALID_ARG
        p = T.etac_params()                                                  # a caller built before the PointNet arrays
        p.struct_size = T.etac_params.E1.offset
        assert T.load().etac_update_params(eng.ctx, C.byref(p)) == T.ETAC_OK
        assert np.array_equal(eng.step(wl_a.n_envs, dev).cpu().numpy(), U_a)
    finally:
        eng.close()
    eng = T.Etac(base, precision=precision)                                  # per-node context
    try:
        with pytest.raises(T.EtacError) as ei:
            T.etac_update_params(eng.ctx, weights=wl_b.weights)
        assert ei.value.status == T.ETAC_ERR_UNSUPPORTED
    finally:
        eng.close()
    assert np.abs(U_a - U_b).max() > 1e-2
    assert np.array_equal(U_ab, U_b) and np.array_equal(U_aa, U_a)


def test_calibration_of_the_pointnet_residual_lowers_the_loss():
    """Eq. (3) with the paper's Phi end to end on synthetic data: targets from a teacher with its own PointNet weights
    and alpha; Adam on all ten weight arrays and alpha (gradients from etac_backward, written back with
    etac_update_params) from another random start lowers 1/2 ||U - U*||^2 by more than 100x in 150 steps."""
    import dataclasses
    import torch
    base = W.config2(18, 12)
    wl_t = dataclasses.replace(base, weights=W.make_pointnet_weights(3, 8, std=0.15))
    dev_kw = dict(indenters=wl_t.indenters, patch_pose=wl_t.patch_pose)
    teacher = T.Etac(wl_t, precision="fp32")
    target = teacher.step(wl_t.n_envs, teacher.upload(**dev_kw)).clone()
    teacher.close()
    w = {k: v.astype(np.float64) for k, v in W.make_pointnet_weights(3, 9, std=0.1).items()}
    a = wl_t.alpha.astype(np.float64) * 0.8
    eng = T.Etac(dataclasses.replace(wl_t, alpha=a.astype(np.float32), weights={k: v.astype(np.float32) for k, v in w.items()}),
                 precision="fp32")
    try:
        dev = eng.upload(**dev_kw)
        stream = torch.cuda.current_stream().cuda_stream
        g_alpha = torch.empty(a.size, device=eng.device)
        g_w = torch.empty(T.ETAC_GRAD_WEIGHTS_POINTNET_LEN, device=eng.device)
        theta = {"alpha": a, **w}
        m1 = {k: np.zeros_like(v) for k, v in theta.items()}
        m2 = {k: np.zeros_like(v) for k, v in theta.items()}
        lr = {k: 3e-3 for k in theta}
        lr["alpha"] = 0.01
        losses = []
        for it in range(1, 151):
            G = eng.step(wl_t.n_envs, dev) - target
            losses.append(0.5 * float((G * G).sum()))
            T.etac_backward(eng.ctx, stream, wl_t.n_envs, G.contiguous(), g_alpha, g_w, **dev)
            grads = {k: v.astype(np.float64) for k, v in T.split_grad_weights(g_w.cpu().numpy()).items()}
            grads["alpha"] = g_alpha.cpu().numpy().astype(np.float64)
            for k in theta:
                m1[k] = 0.9 * m1[k] + 0.1 * grads[k]
                m2[k] = 0.999 * m2[k] + 0.001 * grads[k] ** 2
                theta[k] = theta[k] - lr[k] * (m1[k] / (1 - 0.9 ** it)) / (np.sqrt(m2[k] / (1 - 0.999 ** it)) + 1e-12)
            theta["alpha"] = np.maximum(theta["alpha"], 0.05)
            T.etac_update_params(eng.ctx, alpha=theta["alpha"].astype(np.float32),
                                 weights={k: v.astype(np.float32) for k, v in theta.items() if k != "alpha"})
    finally:
        eng.close()
    print(f"[calibration pointnet] alpha {theta['alpha']} vs {wl_t.alpha}; loss {losses[0]:.4g} -> {min(losses):.4g} (last {losses[-1]:.4g})")
    assert losses[-1] < 0.01 * losses[0]


def test_calibration_recovers_alpha_of_a_synthetic_teacher():
    """Eq. (3) end to end on synthetic data (the paper's FEM data is not available): displacements of a
    teacher with hidden alpha* (one per patch) are the targets; Adam on dL/dalpha from etac_backward, written
    back with etac_update_params, recovers alpha* from a start 30-40 % off."""
    import dataclasses
    import torch
    wl, precision, mode, _ = _backward_case("per_patch_alpha")
    a_star = wl.alpha.astype(np.float64)
    dev_kw = dict(indenters=wl.indenters, patch_pose=wl.patch_pose)
    teacher = T.Etac(wl, precision=precision)
    target = teacher.step(wl.n_envs, teacher.upload(**dev_kw)).clone()
    teacher.close()
    a = a_star * np.asarray([0.65, 1.35, 0.7])
    eng = T.Etac(dataclasses.replace(wl, alpha=a.astype(np.float32)), precision=precision)
    try:
        dev = eng.upload(**dev_kw)
        stream = torch.cuda.current_stream().cuda_stream
        g_alpha = torch.empty(3, device=eng.device)
        m1, m2, losses = np.zeros(3), np.zeros(3), []
        for it in range(1, 121):
            G = eng.step(wl.n_envs, dev) - target
            losses.append(0.5 * float((G * G).sum()))
            T.etac_backward(eng.ctx, stream, wl.n_envs, G.contiguous(), g_alpha, None, **dev)
            g = g_alpha.cpu().numpy().astype(np.float64)
            m1, m2 = 0.9 * m1 + 0.1 * g, 0.999 * m2 + 0.001 * g * g
            a = a - 0.02 * (m1 / (1 - 0.9 ** it)) / (np.sqrt(m2 / (1 - 0.999 ** it)) + 1e-12)
            T.etac_update_params(eng.ctx, alpha=a.astype(np.float32))
    finally:
        eng.close()
    print(f"[calibration] alpha {a} vs {a_star}; loss {losses[0]:.4g} -> {losses[-1]:.4g}")
    assert np.abs(a - a_star).max() < 0.02 and losses[-1] < 1e-3 * losses[0]


def test_step_is_capturable_in_a_cuda_graph():
    """etac_step only enqueues (no sync, no allocation, no host copy): it can be captured in a
    CUDA graph and replayed; the replays give the eager result bit for bit."""
    import torch
    for wl in (W.config2(13, 16), W.config3(13, 40), W.config4(13, 40)):      # fp32; 16-env tile; clusters + bucketed S1
        eng = T.Etac(wl)
        try:
            dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
            eager = eng.step(wl.n_envs, dev).clone()
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            side = torch.cuda.Stream()
            with torch.cuda.stream(side):
                eng.step(wl.n_envs, dev)                      # warm-up on the capture stream
                torch.cuda.synchronize()
                with torch.cuda.graph(g, stream=side):
                    eng.step(wl.n_envs, dev)
            for _ in range(3):
                eng.out.fill_(float("nan"))
                g.replay()
            torch.cuda.synchronize()
            assert torch.equal(eng.out[: wl.n_envs], eager)
        finally:
            eng.close()


def test_sfu_rate_microbenchmark_is_plausible():
    """bench.py's "alu" roofline divides by this live measurement: it must be a whole-device rate of the order
    of 16 results per clock and SM (four sub-partitions x four lanes), not a launch-bound or optimised-away one."""
    import torch
    ops_s, per_clk_sm = T.etac_measure_sfu_rate(torch.cuda.current_stream().cuda_stream)
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    assert 8.0 <= per_clk_sm <= 17.0, per_clk_sm
    assert ops_s > 1e9 * n_sm


@pytest.mark.parametrize("n_nodes,curved,frac,path", [(1024, False, 0.05, T.ETAC_PATH_DENSE),
                                                     (1024, False, 0.05, T.ETAC_PATH_SPARSE),
                                                     (8192, True, 0.01, T.ETAC_PATH_DENSE)])
def test_config5_largest_batch_sampled(n_nodes, curved, frac, path):
    """BASELINE.json configs[4] at its largest batch (16,384 envs; N = 8192 is its largest mesh too): every
    output of the step comes back, the oracle checks a sample of environments one by one,
    and the properties that hold at any size are checked on all of them."""
    E = 16384
    wl = W.config5(E, n_nodes, curved, frac, "bf16")
    gpu = run_gpu(wl, path=path)
    assert gpu["path"] == path
    envs = [0, 5461, 10923, E - 1] if n_nodes > 4096 else list(range(0, E, 683)) + [E - 1]
    ref = run_oracle(wl, envs=envs)
    _report(f"cfg5 E={E} N={n_nodes} path={path}",
            compare(gpu, ref, TOL["bf16"], envs=envs, resid_tol=5e-2, label="cfg5-max", delta_tol=1e-4))
    # every env: active rows keep u^ = -delta n exactly (P7), mask <=> delta > 0, active-node counts, pairs
    act = gpu["mask"]
    assert np.array_equal(act, gpu["delta"] > 0.0)
    np.testing.assert_array_equal(gpu["U"][act], (-gpu["delta"][..., None] * wl.mesh.normal[None])[act])
    assert np.array_equal(gpu["active_count"], act.sum(1))
    assert gpu["pairs"] == int(act.any(1).sum())


@pytest.mark.parametrize("cfg,n_envs,group_bytes", [("cfg4", 40, 1 << 10), ("cfg4", 40, 1700 << 10), ("cfg3", 200, 120 << 10)])
def test_grouped_item_order_is_only_scheduling(cfg, n_envs, group_bytes):
    """ETAC_OPT_L2_GROUP_BYTES forced small: the fused kernel's grouped item order (groups of 1 env tile; of 2 with
    a ragged last group; several patches with different tile counts) against the oracle on every env, and bit for
    bit against the plain order."""
    wl = W.config4(3, n_envs) if cfg == "cfg4" else W.config3(3, n_envs)
    ref = run_oracle(wl)
    plain = run_gpu(wl)
    grouped = run_gpu(wl, group_bytes=group_bytes)
    _report(f"{cfg} grouped {group_bytes}", compare(grouped, ref, TOL["bf16"], resid_tol=5e-2, label="grouped", delta_tol=1e-4))
    assert np.array_equal(grouped["U"], plain["U"]) and np.array_equal(grouped["analytic"], plain["analytic"])
    with pytest.raises(T.EtacError):
        eng = T.Etac(wl)
        try:
            T.etac_set_option(eng.ctx, T.ETAC_OPT_L2_GROUP_BYTES, 0)
        finally:
            eng.close()


@pytest.mark.parametrize("out_bf16", [False, True])
def test_big_patch_instantiation_pointnet_and_linear_only(out_bf16):
    """One patch of 8192 nodes takes the big-patch instantiation of the fused kernel (grouped item order, u_lin
    parked in shared memory, one pipeline stage fewer) at any batch size: its PointNet decode pass, its
    no-residual form and its bf16-output store against the oracle (the per-node form is in the cfg-4 tests)."""
    import dataclasses
    import torch
    base = W.config4(5, 19)                           # two env tiles, the second ragged
    wl = dataclasses.replace(base, weights=W.make_pointnet_weights(3, 2, std=0.15))
    ref = run_oracle(wl)
    if not out_bf16:
        gpu = run_gpu(wl)
        assert gpu["launches"] == 6      # S1 (evaluate, bucket scatter), encode + pool, global MLP, tile k-block masks, decode
        _report("big-patch pointnet", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="big-pointnet", delta_tol=1e-4))
        lin, ref_lin = run_gpu(base, resid=False), run_oracle(base, resid=False)
        _report("big-patch linear", compare(lin, ref_lin, TOL["bf16"], label="big-linear", delta_tol=1e-4))
    else:
        eng = T.Etac(wl)
        try:
            dev = eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)
            out16 = torch.full((wl.n_envs, eng.N, 3), float("nan"), dtype=torch.bfloat16, device="cuda")
            T.etac_step(eng.ctx, torch.cuda.current_stream().cuda_stream,
                        T.make_step_args(wl.n_envs, out16, indenters=dev["indenters"], patch_pose=dev.get("patch_pose"),
                                         out_dtype=T.ETAC_OUT_BF16))
            torch.cuda.synchronize()
            U = out16.float().cpu().numpy()
        finally:
            eng.close()
        umax = float(np.abs(ref["U"]).max())
        assert np.isfinite(U).all() and np.abs(U - ref["U"]).max() <= (TOL["bf16"] + 2.0 ** -8) * umax


@pytest.mark.parametrize("kind", ["dense", "gather16", "fp32", "pointnet", "big_patch"])
def test_workspace_reuse_across_changing_contact_sets(kind):
    """One context stepped with input set A, then set B (other contacts, other (env, patch) pairs), then the
    first third of B's environments: every result equals, bit for bit, what a fresh context gives for the
    same inputs -- the per-step workspace (U^ slot rows, active lists, delta, env lists, pooled features)
    carries nothing from one step to the next."""
    import dataclasses
    import torch
    E = 61
    if kind == "big_patch":
        wa, wb = W.config4(21, E), W.config4(22, E)
    else:
        wa, wb = W.config3(21, E), W.config3(22, E)
    pw = W.make_pointnet_weights(3, 5, std=0.15) if kind == "pointnet" else wa.weights
    wa, wb = dataclasses.replace(wa, weights=pw), dataclasses.replace(wb, weights=pw)   # one model, two input sets
    precision = "fp32" if kind == "fp32" else "bf16"
    path = T.ETAC_PATH_SPARSE if kind == "gather16" else T.ETAC_PATH_AUTO
    n_small = E // 3

    def fresh(wl, n):
        eng = T.Etac(wl, precision=precision, max_envs=E)
        try:
            T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, path)
            eng.out.fill_(float("nan"))
            out = eng.step(n, eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)).cpu().numpy()
        finally:
            eng.close()
        return out

    want_b, want_small = fresh(wb, E), fresh(wb, n_small)
    eng = T.Etac(wa, precision=precision, max_envs=E)
    try:
        T.etac_set_option(eng.ctx, T.ETAC_OPT_PATH, path)
        da = eng.upload(indenters=wa.indenters, patch_pose=wa.patch_pose)
        db = eng.upload(indenters=wb.indenters, patch_pose=wb.patch_pose)
        eng.step(E, da)
        eng.out.fill_(float("nan"))
        got_b = eng.step(E, db).cpu().numpy()
        eng.step(E, da)
        eng.out.fill_(float("nan"))
        got_small = eng.step(n_small, db).cpu().numpy()
        rest = eng.out[n_small:E].cpu().numpy()
    finally:
        eng.close()
    assert np.isfinite(got_b).all()
    assert np.array_equal(got_b, want_b)
    assert np.array_equal(got_small, want_small)
    assert np.isnan(rest).all()                       # rows of environments >= n_envs are not touched
    ref = run_oracle(wb)
    assert np.abs(got_b - ref["U"]).max() <= TOL[precision] * np.abs(ref["U"]).max()


def test_residual_only_without_a_residual_network_is_zero_on_passive_rows():
    """ETAC_ABLATE_RESIDUAL_ONLY on a context created without Phi: U_p = Phi_p = 0 on the passive rows,
    active rows keep u^ -- the same answer from the fp32 and the bf16 context (and from the oracle)."""
    from oracle import etac_oracle as O
    wl = W.config3(23, 13)
    m = O.model_from_workload(wl, resid_arch="none")
    m.ablation = "residual_only"
    ref = O.step(m, indenters=wl.indenters, patch_pose=wl.patch_pose)
    assert np.all(ref["U"][~ref["mask"]] == 0)
    for precision in ("fp32", "bf16"):
        eng = T.Etac(wl, precision=precision, resid=False)
        try:
            T.etac_set_option(eng.ctx, T.ETAC_OPT_ABLATION, T.ETAC_ABLATE_RESIDUAL_ONLY)
            U = eng.step(wl.n_envs, eng.upload(indenters=wl.indenters, patch_pose=wl.patch_pose)).cpu().numpy()
        finally:
            eng.close()
        assert np.all(U[~ref["mask"]] == 0), precision
        np.testing.assert_allclose(U[ref["mask"]], ref["U"][ref["mask"]], rtol=0, atol=2e-5)


@pytest.mark.parametrize("pattern", ["disjoint", "clustered", "spread"])
def test_block_sparse_contraction_on_a_large_patch(pattern):
    """Large patches take the block-sparse form of the dense contraction (Omega is (n-m) x m): S1
    records which 64-node k-blocks hold an active node, buckets the environments by contact position, and the
    TMA / MMA warps skip the k-blocks no environment of a 32-env tile touches.  Penetration input on a 64 x 64 pad
    (N = 4096, 64 k-blocks), 77 environments = three tiles, the last ragged: "disjoint" = every environment touches
    ONE k-block of its own (no two environments of a tile share one: the union has as many blocks as the tile has
    environments), "clustered" = all contacts inside four neighbouring k-blocks (almost everything is skipped),
    "spread" = nodes in contact all over the pad (nothing can be skipped).  Against the oracle on every env."""
    mesh = W.assemble([W.flat_pad(64, 64, 1.0)])
    E, N = 77, mesh.n_nodes
    rng = np.random.default_rng({"disjoint": 1, "clustered": 2, "spread": 3}[pattern])
    pen = np.zeros((E, N), np.float32)
    for e in range(E):
        if pattern == "disjoint":
            blk = (e * 29) % 64
            idx = blk * 64 + rng.choice(64, size=rng.integers(1, 9), replace=False)
        elif pattern == "clustered":
            idx = 20 * 64 + rng.choice(256, size=rng.integers(3, 40), replace=False)
        else:
            idx = rng.choice(N, size=rng.integers(30, 300), replace=False)
        pen[e, idx] = rng.uniform(0.05, 1.0, len(idx))
    pen[5] = 0.0                                    # an environment without contact in the middle of a tile
    wl = W.Workload("block_sparse", mesh, np.float32([0.5]), W.make_weights(8, 3, std=0.1), E, 0,
                    np.zeros((E, 0), dtype=W.INDENTER_DTYPE), None, "bf16")
    ref = run_oracle(wl, penetration=pen)
    gpu = run_gpu(wl, penetration=pen)
    assert gpu["path"] == T.ETAC_PATH_DENSE and gpu["pairs"] == E - 1
    _report(f"block-sparse {pattern}", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="block-sparse"))
    assert np.all(gpu["U"][5] == 0)


@pytest.mark.parametrize("n_envs", [1, 70])
def test_two_large_patches_bucketed(n_envs):
    """Two patches of 2048 nodes (a flat pad and a curved sheet, own alpha each) with sphere indenters: the per-env S1
    kernel in bucket mode + scatter over SEVERAL patches, the 32-env tile with a ragged last tile (and a single
    environment), an environment that touches only one of the two patches."""
    mesh = W.assemble([W.flat_pad(32, 64, 1.0), W.cyl_sheet(40.0, 32.0 / 40.0, 32, 64, 1.0)])
    rng = np.random.default_rng(77 + n_envs)
    ind = W._blank_indenters(n_envs, 2)
    off = np.asarray(mesh.patch_offset)
    pose = np.zeros((n_envs, 2, 7), np.float32)
    pose[:, :, 6] = 1.0
    pose[:, 1, 0] = 500.0                                              # the sheet sits 0.5 m away from the pad
    for k in range(2):
        c = rng.integers(off[k], off[k + 1], size=n_envs)
        size = rng.uniform(3.0, 12.0, n_envs)
        centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, rng.uniform(0.1, 1.2, n_envs), np.zeros(n_envs))
        ind["type"][:, k] = W.IND_SPHERE
        ind["param"][:, k, 0] = size
        ind["pose"][:, k, 0:3] = centre + pose[:, k, 0:3]
        ind["pose"][:, k, 3:7] = q
    if n_envs > 3:
        ind["type"][3, 1] = W.IND_NONE                                 # env 3 touches the pad only
    wl = W.Workload("two_large", mesh, np.float32([0.5, 0.35]), W.make_weights(8, 5, std=0.1), n_envs, 2, ind, pose, "bf16")
    gpu, ref = run_gpu(wl), run_oracle(wl)
    _report(f"two large patches E={n_envs}", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="two-large", delta_tol=1e-4))
    assert gpu["pairs"] == int(ref["contact"].sum()) and gpu["launches"] == 4      # S1 evaluate + scatter, tile masks, fused


@pytest.mark.parametrize("kind,n_envs", [("pair", 40), ("pair", 1), ("tile16", 40)])
def test_patch_sizes_that_are_not_multiples_of_eight(kind, n_envs):
    """Patches whose node counts are odd: every patch after the first starts at an odd node index, while TMA boxes of
    the U^ operand have to start on 16-byte boundaries (the operand rows are padded per patch).
    "pair": the 32-env instantiation runs as clusters of two CTAs that share the U^ tile of a PAIR of node blocks; a
    patch of 2139 nodes (17 blocks of 128, the last one ragged: the pair's second CTA has a block beyond the patch)
    beside a patch of 100 nodes (one block: the second CTA has no block at all) and one of 384 (three blocks).
    "tile16": the 16-env instantiation on patches of 35, 2015 and 81 nodes."""
    if kind == "pair":
        parts = [W.flat_pad(31, 69, 1.0), W.flat_pad(10, 10, 1.0), W.cyl_sheet(40.0, 16.0 / 40.0, 16, 24, 1.0)]
    else:
        parts = [W.flat_pad(5, 7, 1.0), W.flat_pad(31, 65, 1.0), W.flat_pad(9, 9, 1.0)]
    mesh = W.assemble(parts)
    rng = np.random.default_rng(99 + n_envs)
    ind = W._blank_indenters(n_envs, 3)
    off = np.asarray(mesh.patch_offset)
    pose = np.zeros((n_envs, 3, 7), np.float32)
    pose[:, :, 6] = 1.0
    pose[:, 1, 0], pose[:, 2, 0] = 400.0, 800.0
    for k in range(3):
        c = rng.integers(off[k], off[k + 1], size=n_envs)
        size = rng.uniform(2.0, 9.0, n_envs)
        centre, q = W._press_on_node(mesh.pos, mesh.normal, c, None, size, rng.uniform(0.1, 1.0, n_envs), np.zeros(n_envs))
        ind["type"][:, k] = W.IND_SPHERE
        ind["param"][:, k, 0] = size
        ind["pose"][:, k, 0:3] = centre + pose[:, k, 0:3]
        ind["pose"][:, k, 3:7] = q
    if n_envs > 5:
        ind["type"][5, 1 if kind == "tile16" else 0] = W.IND_NONE      # env 5 does not touch the large patch
    wl = W.Workload("odd_sizes", mesh, np.float32([0.5, 0.4, 0.3]), W.make_weights(8, 6, std=0.1), n_envs, 3, ind, pose, "bf16")
    gpu, ref = run_gpu(wl), run_oracle(wl)
    _report(f"odd patch sizes ({kind}) E={n_envs}", compare(gpu, ref, TOL["bf16"], resid_tol=5e-2, label="odd-sizes", delta_tol=1e-4))
    assert gpu["pairs"] == int(ref["contact"].sum())
    assert gpu["launches"] == (4 if kind == "pair" else 2)             # the 32-env tile: S1 evaluate + scatter, tile masks, fused
