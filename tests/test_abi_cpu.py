"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/ks.h declares;
host-side logic that needs no GPU (argument validation happens before any CUDA call)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2606_28565_b200 import binding as B
from paper_2606_28565_b200 import build as ksbuild
from paper_2606_28565_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    ksbuild.build()
    return B.load()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "ks.h")).read()
    declared = set(re.findall(r"\b(ks_[a-z_]+)\s*\(", hdr))
    assert {"ks_create", "ks_load_heads", "ks_load_grid", "ks_predict_kernels", "ks_compose_steps",
            "ks_destroy"} <= declared
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layouts_match_header():
    assert C.sizeof(B.ks_hw_spec) == 44
    assert C.sizeof(B.ks_step_params) == 20
    assert C.sizeof(B.ks_desc_batch) == 32 + 8 * B.KS_MAX_COLS + 8
    assert (C.sizeof(B.ks_sched_config), C.sizeof(B.ks_model_desc), C.sizeof(B.ks_sched_stats),
            C.sizeof(B.ks_sim_stats)) == (24, 36, 72, 64)


def test_status_strings(lib):
    assert B.status_string(B.KS_OK) == "KS_OK" and B.status_string(B.KS_ESTATE) == "KS_ESTATE"


def test_null_and_bad_arguments_fail_before_cuda(lib):
    assert lib.ks_create(None, 0, None) == B.KS_EINVAL
    assert lib.ks_destroy(None) == B.KS_OK
    assert lib.ks_predict_kernels(None, None, 0, None, 0, 0, 0, None, None, None, None) == B.KS_EINVAL
    assert lib.ks_set_gelu_mode(None, 0) == B.KS_EINVAL
    p = B.make_step_params(W.STEP_PARAMS_ZERO)
    assert lib.ks_compose_steps(None, None, None, None, 0, 0, 0, C.byref(p), None, 0, 0, None, None) == B.KS_EINVAL


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    assert lib.ks_create(C.byref(h), 0, None) == B.KS_ECUDA and not h.value
    with pytest.raises(B.KsError):
        B.Context(0)


def test_marshalling_of_batches():
    w = W.config2(n=1000)
    b = B.make_batch(w.buckets[1])
    assert (b.family, b.n, b.col_dtype, b.n_cols, b.attn_hq, b.attn_hkv, b.attn_head_dim) == (2, 300, 0, 3, 32, 8, 128)
    assert b.cols[0] == w.buckets[1].cols[0].ctypes.data and not b.cols[3]
    b1 = B.make_batch(W.config1().buckets[0])
    assert b1.col_dtype == B.KS_COL_F32
    bad = W.Bucket(0, [np.zeros(4, np.int64)] * 3)
    with pytest.raises(TypeError):
        B.make_batch(bad)
