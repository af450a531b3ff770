"""etac_propagate_noalloc (include/etac_noalloc.h): the entry point that allocates nothing (scratch in a static
__device__ array) against the existing context path -- an ETAC_PREC_FP32 context without a residual network in
penetration input mode -- on two calls in a row that share the scratch, and its size limit.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.  Needs nothing from the
tests before it and leaves nothing behind: passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W
from parity_util import TOL, run_gpu

pytestmark = pytest.mark.gpu


def _penetration(rng, mesh, n_envs, n_bumps, radius):
    """Seeded synthetic penetration: per env `n_bumps` smooth bumps of up to 0.8 mm around random nodes, negative
    (= no contact, clamped by the method) elsewhere; env 1 has no contact at all."""
    pen = np.full((n_envs, mesh.n_nodes), -0.05, np.float32)
    for e in range(n_envs):
        for c in rng.integers(0, mesh.n_nodes, size=n_bumps):
            r = np.linalg.norm(mesh.pos - mesh.pos[c], axis=1)
            pen[e] = np.maximum(pen[e], rng.uniform(0.2, 0.8) * (1.0 - (r / radius) ** 2))
    if n_envs > 1:
        pen[1] = -0.05
    return pen


def test_noalloc_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    wl = W.config2(3, 48)                                              # one patch, 1024 nodes, fp32
    assert len(wl.mesh.patch_offset) == 2 and wl.n_envs * wl.mesh.n_nodes <= T.ETAC_NOALLOC_MAX_ENTRIES
    rng = np.random.default_rng(2024)
    N, E = wl.mesh.n_nodes, wl.n_envs
    # the second call has FEWER active nodes per environment than the first: entries the first call left in the
    # shared scratch beyond the new counts must not be read
    pens = [_penetration(rng, wl.mesh, E, 3, 6.0), _penetration(rng, wl.mesh, E, 1, 3.0)]
    assert (pens[0] > 0).sum() > 2 * (pens[1] > 0).sum() > 0
    refs = [run_gpu(wl, precision="fp32", resid=False, penetration=p) for p in pens]   # the existing path
    dev = torch.device("cuda:0")
    pos = torch.from_numpy(np.ascontiguousarray(wl.mesh.pos, np.float32)).to(dev)
    nrm = torch.from_numpy(np.ascontiguousarray(wl.mesh.normal, np.float32)).to(dev)
    d_pens = [torch.from_numpy(p).to(dev) for p in pens]
    outs = [torch.full((E, N, 3), float("nan"), device=dev) for _ in pens]
    stream = torch.cuda.current_stream().cuda_stream
    for d_pen, out in zip(d_pens, outs):                               # back to back on one stream, no sync in between
        T.etac_propagate_noalloc(stream, E, N, float(wl.alpha[0]), pos, nrm, d_pen, out)
    torch.cuda.synchronize()
    for k, (out, ref) in enumerate(zip(outs, refs)):
        got = out.cpu().numpy()
        assert np.isfinite(got).all(), f"call {k}: unwritten output"
        scale = np.abs(ref["U"]).max()
        err = np.abs(got - ref["U"]).max()
        print(f"[noalloc] call {k}: max|u| {scale:.4g} max err {err:.3g} ({err / scale:.2e} rel)")
        assert scale > 0.1 and err <= TOL["fp32"] * scale
        assert not got[1].any()                                       # the environment without contact is exactly 0
        act = pens[k] > 0
        n32 = wl.mesh.normal.astype(np.float32).astype(np.float64)    # active rows are u^ = -delta n, one fp32 rounding
        assert np.array_equal(got[act], (-pens[k][act].astype(np.float64)[:, None] * n32[np.nonzero(act)[1]]).astype(np.float32))


def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    dev = torch.device("cuda:0")
    t = torch.zeros(8, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    with pytest.raises(T.EtacError) as ei:
        T.etac_propagate_noalloc(stream, 1024, 1024, 0.5, t, t, t, t)  # 2^20 entries > ETAC_NOALLOC_MAX_ENTRIES
    assert ei.value.status == T.ETAC_ERR_CAPACITY and "ETAC_NOALLOC_MAX_ENTRIES" in str(ei.value)
    with pytest.raises(T.EtacError) as ei:
        T.etac_propagate_noalloc(stream, T.ETAC_NOALLOC_MAX_ENVS + 1, 1, 0.5, t, t, t, t)
    assert ei.value.status == T.ETAC_ERR_CAPACITY and "ETAC_NOALLOC_MAX_ENVS" in str(ei.value)
    with pytest.raises(T.EtacError) as ei:
        T.etac_propagate_noalloc(stream, 2, 4, 0.5, t, None, t, t)
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG
    T.etac_propagate_noalloc(stream, 0, 4, 0.5, None, None, None, None)   # empty: a no-op
    torch.cuda.synchronize()
