"""CPU-side checks of the C-ABI library: it loads without a GPU, exports every symbol that
include/etac.h declares, validates arguments before touching CUDA, and its host-only logic
(patch derivation from the mesh adjacency) is right.  No compute calls."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2604_20295_b200 import build as B
from paper_2604_20295_b200 import etac as T
from paper_2604_20295_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return T.load()


def test_exports_match_header(lib):
    import glob
    hdr = "".join(open(h).read() for h in sorted(glob.glob(os.path.join(ROOT, "include", "*.h"))))
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(etac_[a-z_]+)\s*\(", hdr))
    assert declared == set(T.EXPORTS)
    product = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "etac.h")).read(), flags=re.S)
    assert "etac_time_steps" not in product and "etac_measure_sfu_rate" not in product   # etac_bench.h only
    for name in declared:
        assert getattr(lib, name) is not None
    assert lib.etac_abi_version() == 7
    assert C.sizeof(T.etac_indenter) == 48 == W.INDENTER_DTYPE.itemsize


def test_struct_layouts_match_header():
    # field order of the ctypes mirrors == order of declaration in the header
    hdr = open(os.path.join(ROOT, "include", "etac.h")).read()
    body = hdr[hdr.index("typedef struct {\n  uint32_t struct_size;        /*"): hdr.index("} etac_model_desc;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"[\*\s](\w+)\s*[;,]", body)
    assert names == [f[0] for f in T.etac_model_desc._fields_]
    body = hdr[hdr.index("typedef struct {\n  uint32_t struct_size;               /*"): hdr.index("} etac_step_args;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"[\*\s](\w+)\s*;", body)
    assert names == [f[0] for f in T.etac_step_args._fields_]


def test_create_validates_before_cuda(lib):
    wl = W.config1()
    m = wl.mesh
    with pytest.raises(T.EtacError) as ei:
        T.etac_create(m.pos, m.normal, [-1.0], patch_offset=m.patch_offset)
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG and "alpha" in str(ei.value)
    with pytest.raises(T.EtacError) as ei:
        T.etac_create(m.pos, m.normal, [0.5], patch_offset=np.int32([0, 100, 50, 256]))
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG
    with pytest.raises(T.EtacError) as ei:
        T.etac_create(m.pos, m.normal, [0.5], patch_offset=m.patch_offset, weights=wl.weights,
                      resid_arch=T.ETAC_RESID_POINTNET, precision=T.ETAC_PREC_BF16)
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG and "PointNet" in str(ei.value)     # per-node weights only
    with pytest.raises(T.EtacError) as ei:
        T.etac_create(m.pos, m.normal, [0.5], patch_offset=m.patch_offset, max_envs=0)
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG
    # an edge crossing a declared patch boundary is rejected
    with pytest.raises(T.EtacError) as ei:
        T.etac_create(m.pos, m.normal, [0.5], patch_offset=np.int32([0, 128, 256]), adj_rowptr=m.adj_rowptr,
                      adj_col=m.adj_col)
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG and "crosses" in str(ei.value)
    # ABI guard
    d = T.etac_model_desc()
    d.struct_size = 4
    ctx = C.c_void_p()
    assert lib.etac_create(C.byref(d), C.byref(ctx)) == T.ETAC_ERR_INVALID_ARG and not ctx.value
    assert lib.etac_destroy(None) == T.ETAC_OK
    assert lib.etac_step(None, None, None) == T.ETAC_ERR_INVALID_ARG


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    wl = W.config1()
    with pytest.raises(T.EtacError) as ei:
        T.etac_create(wl.mesh.pos, wl.mesh.normal, wl.alpha, patch_offset=wl.mesh.patch_offset, weights=wl.weights)
    assert ei.value.status == T.ETAC_ERR_CUDA and "no CPU fallback" in str(ei.value)


def test_patches_from_adjacency(lib):
    hand = W.hand_mesh()
    off = T.etac_patches_from_adjacency(hand.n_nodes, hand.adj_rowptr, hand.adj_col)
    assert np.array_equal(off, hand.patch_offset) and len(off) == 17
    # no edges: every node is its own patch
    off = T.etac_patches_from_adjacency(5, np.zeros(6, np.int32), np.zeros(0, np.int32))
    assert list(off) == [0, 1, 2, 3, 4, 5]
    # components 0-2 and 1: node 1 interrupts the range {0,2} -> unsupported
    rp, col = np.int32([0, 1, 1, 2]), np.int32([2, 0])
    with pytest.raises(T.EtacError) as ei:
        T.etac_patches_from_adjacency(3, rp, col)
    assert ei.value.status == T.ETAC_ERR_UNSUPPORTED
    with pytest.raises(T.EtacError) as ei:
        T.etac_patches_from_adjacency(3, rp, np.int32([7, 0]))
    assert ei.value.status == T.ETAC_ERR_INVALID_ARG
