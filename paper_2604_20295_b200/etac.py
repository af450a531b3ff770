"""Thin ctypes binding of the C ABI in include/etac.h -- argument marshalling only.

Every step of the hot path (S1 contact detection, S2 propagation, S3 residual MLP, S4 combine;
PAPER.md:L77-L102) runs in the CUDA kernels of libetac.so.  There is no Python or CPU fallback:
if the library is missing, ``load()`` raises.  PyTorch is used by callers for device memory and
streams only; this module accepts raw device pointers (ints) or torch tensors.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libetac.so")

ETAC_OK, ETAC_ERR_INVALID_ARG, ETAC_ERR_UNSUPPORTED, ETAC_ERR_ALLOC, ETAC_ERR_CUDA, ETAC_ERR_CAPACITY = range(6)
ETAC_IND_NONE, ETAC_IND_SPHERE, ETAC_IND_BOX, ETAC_IND_CAPSULE, ETAC_IND_GRID = range(5)
ETAC_KERNEL_EXP_L2 = 0
ETAC_RESID_NONE, ETAC_RESID_PERNODE_MLP, ETAC_RESID_POINTNET = range(3)
ETAC_PREC_FP32, ETAC_PREC_BF16 = 0, 1
ETAC_ACTIVE_PASSTHROUGH, ETAC_ACTIVE_PROPAGATE = 0, 1
ETAC_IN_INDENTERS, ETAC_IN_PENETRATION = 0, 1
ETAC_OPT_PATH, ETAC_OPT_ABLATION, ETAC_OPT_L2_GROUP_BYTES = 1, 2, 3
ETAC_ABLATE_FULL, ETAC_ABLATE_RESIDUAL_ONLY, ETAC_ABLATE_LINEAR_ONLY, ETAC_ABLATE_NO_PROPAGATION = range(4)
ETAC_OUT_F32, ETAC_OUT_BF16 = 0, 1
ETAC_PATH_AUTO, ETAC_PATH_DENSE, ETAC_PATH_SPARSE = 0, 1, 2
(ETAC_INFO_N_NODES, ETAC_INFO_N_PATCHES, ETAC_INFO_MAX_ENVS, ETAC_INFO_DEVICE_BYTES, ETAC_INFO_LAST_PATH,
 ETAC_INFO_LAST_LAUNCHES, ETAC_INFO_LAST_CONTACT_PAIRS, ETAC_INFO_SM_COUNT) = range(1, 9)

EXPORTS = ["etac_create", "etac_destroy", "etac_step", "etac_set_option", "etac_get_info", "etac_last_error",
           "etac_patches_from_adjacency", "etac_abi_version", "etac_time_steps", "etac_set_sdf_grid", "etac_backward", "etac_update_params",
           "etac_measure_sfu_rate", "etac_propagate_noalloc", "etac_mesh_to_sdf_grid"]
ETAC_NOALLOC_MAX_ENTRIES, ETAC_NOALLOC_MAX_ENVS = 262144, 4096

_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)


class etac_indenter(C.Structure):
    _fields_ = [("type", C.c_int32), ("param", C.c_float * 3), ("pose", C.c_float * 7), ("skip_patch1", C.c_int32)]


class etac_model_desc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_nodes", C.c_int32), ("node_pos", _fp), ("node_normal", _fp),
                ("n_patches", C.c_int32), ("patch_offset", _ip), ("adj_rowptr", _ip), ("adj_col", _ip),
                ("kernel_type", C.c_int32), ("n_alpha", C.c_int32), ("alpha", _fp),
                ("resid_arch", C.c_int32), ("resid_hidden", C.c_int32),
                ("W1", _fp), ("b1", _fp), ("W2", _fp), ("b2", _fp), ("W3", _fp), ("b3", _fp),
                ("E1", _fp), ("e1", _fp), ("E2", _fp), ("e2", _fp), ("G1", _fp), ("g1", _fp),
                ("D1", _fp), ("d1", _fp), ("D2", _fp), ("d2", _fp),
                ("max_envs", C.c_int32), ("max_indenters", C.c_int32), ("precision", C.c_int32),
                ("active_mode", C.c_int32), ("device", C.c_int32)]


class etac_step_args(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_envs", C.c_int32), ("input_mode", C.c_int32),
                ("d_indenters", C.c_void_p), ("d_patch_pose", C.c_void_p), ("d_penetration", C.c_void_p),
                ("d_out", C.c_void_p), ("d_penetration_out", C.c_void_p), ("d_mask_out", C.c_void_p),
                ("d_analytic_out", C.c_void_p), ("d_contact_out", C.c_void_p), ("d_active_count_out", C.c_void_p),
                ("out_env_stride", C.c_int64), ("out_dtype", C.c_int32), ("reserved", C.c_int32)]


class etac_backward_args(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_envs", C.c_int32), ("input_mode", C.c_int32),
                ("d_indenters", C.c_void_p), ("d_patch_pose", C.c_void_p), ("d_penetration", C.c_void_p),
                ("d_grad_out", C.c_void_p), ("d_grad_alpha", C.c_void_p), ("d_grad_weights", C.c_void_p),
                ("d_grad_penetration", C.c_void_p), ("d_grad_indenter_pose", C.c_void_p), ("d_grad_patch_pose", C.c_void_p)]


class etac_params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_alpha", C.c_int32), ("alpha", _fp),
                ("W1", _fp), ("b1", _fp), ("W2", _fp), ("b2", _fp), ("W3", _fp), ("b3", _fp),
                ("E1", _fp), ("e1", _fp), ("E2", _fp), ("e2", _fp), ("G1", _fp), ("g1", _fp),
                ("D1", _fp), ("d1", _fp), ("D2", _fp), ("d2", _fp)]


ETAC_GRAD_WEIGHTS_LEN = 4995
GRAD_WEIGHTS_LAYOUT = (("W1", (64, 9)), ("b1", (64,)), ("W2", (64, 64)), ("b2", (64,)), ("W3", (3, 64)), ("b3", (3,)))
ETAC_GRAD_WEIGHTS_POINTNET_LEN = 17411
GRAD_WEIGHTS_POINTNET_LAYOUT = (("E1", (64, 9)), ("e1", (64,)), ("E2", (64, 64)), ("e2", (64,)), ("G1", (64, 64)), ("g1", (64,)),
                                ("D1", (64, 128)), ("d1", (64,)), ("D2", (3, 64)), ("d2", (3,)))

_lib = None


def load() -> C.CDLL:
    """dlopen libetac.so (built by ``python -m paper_2604_20295_b200.build``).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2604_20295_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.etac_create.argtypes = [C.POINTER(etac_model_desc), C.POINTER(C.c_void_p)]
        lib.etac_destroy.argtypes = [C.c_void_p]
        lib.etac_step.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(etac_step_args)]
        lib.etac_set_option.argtypes = [C.c_void_p, C.c_int32, C.c_int64]
        lib.etac_get_info.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int64)]
        lib.etac_last_error.argtypes = [C.c_void_p]
        lib.etac_last_error.restype = C.c_char_p
        lib.etac_patches_from_adjacency.argtypes = [C.c_int32, _ip, _ip, _ip, C.c_int32, _ip]
        lib.etac_abi_version.restype = C.c_int32
        lib.etac_time_steps.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(etac_step_args), C.c_int32, _fp, _fp]
        lib.etac_update_params.argtypes = [C.c_void_p, C.POINTER(etac_params)]
        lib.etac_backward.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(etac_backward_args)]
        lib.etac_measure_sfu_rate.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.etac_set_sdf_grid.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, _fp, C.c_float, _fp]
        lib.etac_propagate_noalloc.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p,
                                               C.c_void_p, C.c_char_p, C.c_int32]
        lib.etac_mesh_to_sdf_grid.argtypes = [C.c_int32, C.c_int32, _fp, C.c_int32, _ip, C.c_int32, C.c_int32, C.c_int32, _fp, C.c_float, _fp]
        for name in EXPORTS:
            getattr(lib, name)
        _lib = lib
    return _lib


class EtacError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"etac status {status}: {msg}")
        self.status = status


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


def _p(a, t):
    return None if a is None else a.ctypes.data_as(t)


def _dptr(x):
    """torch tensor / int / None -> raw device address."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    return x.data_ptr()


# ------------------------------------------------------------------ same names as the C ABI
def etac_create(node_pos, node_normal, alpha, *, patch_offset=None, adj_rowptr=None, adj_col=None, weights=None,
                max_envs=1, max_indenters=1, precision=ETAC_PREC_FP32, active_mode=ETAC_ACTIVE_PASSTHROUGH,
                device=0, resid_arch=None, resid_hidden=64) -> int:
    lib = load()
    pos, nrm, al = _f32(node_pos), _f32(node_normal), _f32(np.atleast_1d(alpha))
    off, rp, col = _i32(patch_offset), _i32(adj_rowptr), _i32(adj_col)
    w = {k: _f32(v) for k, v in (weights or {}).items()}
    if resid_arch is None:
        resid_arch = ETAC_RESID_NONE if not weights else (ETAC_RESID_POINTNET if "E1" in w else ETAC_RESID_PERNODE_MLP)
    d = etac_model_desc()
    d.struct_size = C.sizeof(etac_model_desc)
    d.n_nodes = pos.shape[0]
    d.node_pos, d.node_normal = _p(pos, _fp), _p(nrm, _fp)
    d.n_patches = 0 if off is None else off.shape[0] - 1
    d.patch_offset, d.adj_rowptr, d.adj_col = _p(off, _ip), _p(rp, _ip), _p(col, _ip)
    d.kernel_type = ETAC_KERNEL_EXP_L2
    d.n_alpha, d.alpha = al.shape[0], _p(al, _fp)
    d.resid_arch, d.resid_hidden = resid_arch, resid_hidden
    for k in ("W1", "b1", "W2", "b2", "W3", "b3", "E1", "e1", "E2", "e2", "G1", "g1", "D1", "d1", "D2", "d2"):
        setattr(d, k, _p(w.get(k), _fp))
    d.max_envs, d.max_indenters = max_envs, max_indenters
    d.precision, d.active_mode, d.device = precision, active_mode, device
    ctx = C.c_void_p()
    st = lib.etac_create(C.byref(d), C.byref(ctx))
    if st != ETAC_OK:
        raise EtacError(st, (lib.etac_last_error(None) or b"").decode())
    return ctx.value


def etac_destroy(ctx) -> None:
    st = load().etac_destroy(ctx)
    if st != ETAC_OK:
        raise EtacError(st, "etac_destroy")


def make_step_args(n_envs, out, *, indenters=None, patch_pose=None, penetration=None, penetration_out=None,
                   mask_out=None, analytic_out=None, contact_out=None, active_count_out=None,
                   out_env_stride=0, out_dtype=ETAC_OUT_F32) -> etac_step_args:
    a = etac_step_args()
    a.struct_size = C.sizeof(etac_step_args)
    a.n_envs = n_envs
    a.input_mode = ETAC_IN_PENETRATION if penetration is not None else ETAC_IN_INDENTERS
    a.d_indenters, a.d_patch_pose, a.d_penetration = _dptr(indenters), _dptr(patch_pose), _dptr(penetration)
    a.d_out, a.d_penetration_out = _dptr(out), _dptr(penetration_out)
    a.d_mask_out, a.d_analytic_out = _dptr(mask_out), _dptr(analytic_out)
    a.d_contact_out, a.d_active_count_out = _dptr(contact_out), _dptr(active_count_out)
    a.out_env_stride, a.out_dtype, a.reserved = out_env_stride, out_dtype, 0
    return a


def _check(ctx, st):
    if st != ETAC_OK:
        raise EtacError(st, (load().etac_last_error(ctx) or b"").decode())


def etac_step(ctx, stream, args: etac_step_args) -> None:
    _check(ctx, load().etac_step(ctx, stream, C.byref(args)))


def etac_set_option(ctx, key, value) -> None:
    _check(ctx, load().etac_set_option(ctx, key, value))


def etac_get_info(ctx, key) -> int:
    v = C.c_int64()
    _check(ctx, load().etac_get_info(ctx, key, C.byref(v)))
    return v.value


def etac_set_sdf_grid(ctx, grid_id, values, origin, spacing) -> None:
    """values: [nz, ny, nx] fp32 samples (x fastest), origin [3], spacing."""
    v = _f32(values)
    nz, ny, nx = v.shape
    o = _f32(np.asarray(origin, dtype=np.float32).reshape(3))
    _check(ctx, load().etac_set_sdf_grid(ctx, int(grid_id), nx, ny, nz, _p(o, _fp), C.c_float(float(spacing)), _p(v, _fp)))


def etac_last_error(ctx=None) -> str:
    return (load().etac_last_error(ctx) or b"").decode()


def etac_abi_version() -> int:
    return load().etac_abi_version()


def etac_patches_from_adjacency(n_nodes, adj_rowptr, adj_col):
    rp, col = _i32(adj_rowptr), _i32(adj_col)
    off = np.zeros(n_nodes + 1, dtype=np.int32)
    n = C.c_int32()
    st = load().etac_patches_from_adjacency(n_nodes, _p(rp, _ip), _p(col, _ip), _p(off, _ip), n_nodes + 1, C.byref(n))
    if st != ETAC_OK:
        raise EtacError(st, "etac_patches_from_adjacency")
    return off[: n.value + 1].copy()


def etac_backward(ctx, stream, n_envs, grad_out, grad_alpha, grad_weights=None, *, indenters=None, patch_pose=None,
                  penetration=None, grad_penetration=None, grad_indenter_pose=None, grad_patch_pose=None) -> None:
    """dL/dalpha, dL/d(weights of Phi) and optionally dL/ddelta, dL/d(indenter poses) [E, M, 6], dL/d(patch poses)
    [E, P, 6] of one step from dL/dU (device tensors / addresses; marshalling only)."""
    a = etac_backward_args()
    a.struct_size = C.sizeof(etac_backward_args)
    a.n_envs = n_envs
    a.input_mode = ETAC_IN_PENETRATION if penetration is not None else ETAC_IN_INDENTERS
    a.d_indenters, a.d_patch_pose, a.d_penetration = _dptr(indenters), _dptr(patch_pose), _dptr(penetration)
    a.d_grad_out, a.d_grad_alpha, a.d_grad_weights = _dptr(grad_out), _dptr(grad_alpha), _dptr(grad_weights)
    a.d_grad_penetration = _dptr(grad_penetration)
    a.d_grad_indenter_pose, a.d_grad_patch_pose = _dptr(grad_indenter_pose), _dptr(grad_patch_pose)
    _check(ctx, load().etac_backward(ctx, stream, C.byref(a)))


def etac_update_params(ctx, alpha=None, weights=None) -> None:
    """Replace alpha and / or the weights of the context's residual network in place: {"W1": ..., ..., "b3": ...} on a
    per-node MLP context, {"E1": ..., ..., "d2": ...} on a PointNet context."""
    p = etac_params()
    p.struct_size = C.sizeof(etac_params)
    keep = []
    if alpha is not None:
        a = np.ascontiguousarray(alpha, dtype=np.float32).reshape(-1)
        keep.append(a)
        p.n_alpha, p.alpha = a.size, a.ctypes.data_as(_fp)
    if weights is not None:
        names = ("E1", "e1", "E2", "e2", "G1", "g1", "D1", "d1", "D2", "d2") if "E1" in weights else ("W1", "b1", "W2", "b2", "W3", "b3")
        for k in names:
            w = np.ascontiguousarray(weights[k], dtype=np.float32)
            keep.append(w)
            setattr(p, k, w.ctypes.data_as(_fp))
    _check(ctx, load().etac_update_params(ctx, C.byref(p)))


def etac_mesh_to_sdf_grid(vertices, triangles, shape, origin, spacing, device=0):
    """Closed triangle mesh -> sampled SDF values [nz, ny, nx] fp32 (the layout of etac_set_sdf_grid); shape = (nx, ny, nz)."""
    v, t, o = _f32(vertices), _i32(triangles), _f32(origin)
    nx, ny, nz = (int(x) for x in shape)
    out = np.empty((nz, ny, nx), np.float32)
    st = load().etac_mesh_to_sdf_grid(int(device), v.shape[0], _p(v, _fp), t.shape[0], _p(t, _ip), nx, ny, nz, _p(o, _fp),
                                      C.c_float(float(spacing)), _p(out, _fp))
    if st != ETAC_OK:
        raise EtacError(st, load().etac_last_error(None).decode())
    return out


def etac_propagate_noalloc(stream, n_envs, n_nodes, alpha, pos, normal, penetration, out) -> None:
    """include/etac_noalloc.h: analytic propagation + mask of one patch, no allocation (device fp32 tensors)."""
    err = C.create_string_buffer(256)
    st = load().etac_propagate_noalloc(stream, n_envs, n_nodes, alpha, _dptr(pos), _dptr(normal), _dptr(penetration), _dptr(out),
                                       err, len(err))
    if st != ETAC_OK:
        raise EtacError(st, err.value.decode())


def split_grad_weights(flat):
    """[4995] -> {"W1": [64, 9], "b1": [64], ...} or [17411] -> {"E1": [64, 9], ...} (PointNet): views in the order
    of etac_backward_args.d_grad_weights."""
    out, o = {}, 0
    for name, shape in (GRAD_WEIGHTS_POINTNET_LAYOUT if flat.shape[0] == ETAC_GRAD_WEIGHTS_POINTNET_LEN else GRAD_WEIGHTS_LAYOUT):
        n = int(np.prod(shape))
        out[name] = flat[o:o + n].reshape(shape)
        o += n
    return out


def etac_time_steps(ctx, stream, args: etac_step_args, iters: int, per_kernel: bool = False):
    ms = C.c_float()
    mk = (C.c_float * 2)()
    _check(ctx, load().etac_time_steps(ctx, stream, C.byref(args), iters, C.byref(ms), mk if per_kernel else None))
    return (ms.value, [mk[0], mk[1]]) if per_kernel else ms.value


def etac_measure_sfu_rate(stream):
    """(results/s, results per clock and SM at the nominal maximum clock) of the special-function pipe."""
    a, b = C.c_double(), C.c_double()
    st = load().etac_measure_sfu_rate(stream, C.byref(a), C.byref(b))
    if st != 0:
        raise EtacError(st, "etac_measure_sfu_rate")
    return a.value, b.value


# ------------------------------------------------------------------ convenience wrapper (marshalling only)
class Etac:
    """Owns one etac_ctx built from a workloads.Workload-like object and its device buffers
    (torch tensors).  ``step()`` enqueues on torch's current stream and returns the output tensor."""

    def __init__(self, wl, *, precision=None, active_mode=ETAC_ACTIVE_PASSTHROUGH, device=0, resid=True,
                 max_envs=None, debug_outputs=False):
        import torch
        self.torch = torch
        self.wl = wl
        self.device = torch.device("cuda", device)
        prec = {"fp32": ETAC_PREC_FP32, "bf16": ETAC_PREC_BF16}[precision or wl.precision]
        self.max_envs = max_envs or wl.n_envs
        m = wl.mesh
        self.ctx = etac_create(m.pos, m.normal, wl.alpha, patch_offset=m.patch_offset, adj_rowptr=m.adj_rowptr,
                               adj_col=m.adj_col, weights=wl.weights if resid else None, max_envs=self.max_envs,
                               max_indenters=wl.max_indenters, precision=prec, active_mode=active_mode, device=device)
        for gid, (values, origin, spacing) in getattr(wl, "meta", {}).get("grids", {}).items():
            etac_set_sdf_grid(self.ctx, gid, values, origin, spacing)
        self.N, self.P = m.n_nodes, m.n_patches
        E = self.max_envs
        self.out = torch.empty((E, self.N, 3), dtype=torch.float32, device=self.device)
        self.debug = debug_outputs
        if debug_outputs:
            self.pen_out = torch.empty((E, self.N), dtype=torch.float32, device=self.device)
            self.mask_out = torch.empty((E, (self.N + 31) // 32), dtype=torch.int32, device=self.device)
            self.analytic = torch.empty((E, self.N, 3), dtype=torch.float32, device=self.device)
            self.contact = torch.empty((E, self.P), dtype=torch.uint8, device=self.device)
            self.active_count = torch.empty((E,), dtype=torch.int32, device=self.device)

    def upload(self, indenters=None, patch_pose=None, penetration=None):
        t = self.torch
        dev = {}
        if indenters is not None:
            dev["indenters"] = t.from_numpy(np.ascontiguousarray(indenters).view(np.uint8).reshape(-1)).to(self.device)
        if patch_pose is not None:
            dev["patch_pose"] = t.from_numpy(np.ascontiguousarray(patch_pose, dtype=np.float32)).to(self.device)
        if penetration is not None:
            dev["penetration"] = t.from_numpy(np.ascontiguousarray(penetration, dtype=np.float32)).to(self.device)
        return dev

    def args(self, n_envs, dev, out=None, **opts):
        """Step arguments; `out` (a CUDA tensor: fp32 or bf16, possibly a wider observation buffer)
        together with out_env_stride / out_dtype in `opts` replaces the engine's packed fp32 output."""
        kw = dict(dev)
        kw.update(opts)
        if self.debug:
            kw.update(penetration_out=self.pen_out, mask_out=self.mask_out, analytic_out=self.analytic,
                      contact_out=self.contact, active_count_out=self.active_count)
        return make_step_args(n_envs, self.out if out is None else out, **kw)

    def step(self, n_envs, dev):
        stream = self.torch.cuda.current_stream(self.device).cuda_stream
        etac_step(self.ctx, stream, self.args(n_envs, dev))
        return self.out[:n_envs]

    def mask_bool(self, n_envs):
        """[E, N] bool from the packed mask words (debug outputs)."""
        w = self.mask_out[:n_envs].cpu().numpy().view(np.uint32)
        bits = (w[:, :, None] >> np.arange(32, dtype=np.uint32)) & 1
        return bits.reshape(n_envs, -1)[:, : self.N].astype(bool)

    def close(self):
        if self.ctx:
            etac_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
