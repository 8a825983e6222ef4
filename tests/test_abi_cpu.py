"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/ks.h declares;
host-side logic that needs no GPU (argument validation happens before any CUDA call)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2606_28565_b200 import binding as B
from paper_2606_28565_b200 import build as ksbuild
import workloads as W

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


def test_struct_layouts_match_header(tmp_path):
    """Sizes and field offsets of every ABI struct as gcc lays include/ks.h out, against the ctypes mirrors."""
    import subprocess
    structs = {"ks_hw_spec": B.ks_hw_spec, "ks_desc_batch": B.ks_desc_batch, "ks_step_params": B.ks_step_params,
               "ks_sched_config": B.ks_sched_config, "ks_model_desc": B.ks_model_desc,
               "ks_sched_stats": B.ks_sched_stats, "ks_sim_stats": B.ks_sim_stats}
    lines = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{os.path.join(ROOT, "include", "ks.h")}"',
             'int main(void) {']
    for name, cls in structs.items():
        lines.append(f'  printf("{name} %zu\\n", sizeof({name}));')
        for fld, _ in cls._fields_:
            lines.append(f'  printf("{name}.{fld} %zu\\n", offsetof({name}, {fld}));')
    lines += ['  printf("KS_MAX_MODEL_SLOTS %d\\nKS_SLOT_FAMILY %d\\nKS_HEAD_LOG_ETA %d\\n", (int)KS_MAX_MODEL_SLOTS, '
              '(int)KS_SLOT_FAMILY, (int)KS_HEAD_LOG_ETA);', '  return 0;', '}']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-o", str(exe), str(src)])
    got = dict(line.split() for line in subprocess.check_output([str(exe)], text=True).splitlines())
    for name, cls in structs.items():
        assert int(got[name]) == C.sizeof(cls), name
        for fld, _ in cls._fields_:
            assert int(got[f"{name}.{fld}"]) == getattr(cls, fld).offset, f"{name}.{fld}"
    assert (int(got["KS_MAX_MODEL_SLOTS"]), int(got["KS_SLOT_FAMILY"]), int(got["KS_HEAD_LOG_ETA"])) == \
           (B.KS_MAX_MODEL_SLOTS, B.KS_SLOT_FAMILY, B.KS_HEAD_LOG_ETA)
    assert (W.SLOT_LM_HEAD, W.SLOT_ATTN_PREFILL, W.SLOT_ATTN_DECODE, W.SLOT_RMSNORM, W.SLOT_SILU_MUL, W.SLOT_ROPE,
            W.SLOT_KV_WRITE, W.SLOT_EMBEDDING, W.SLOT_RESIDUAL_ADD) == tuple(range(5, 14))


def test_status_strings(lib):
    assert B.status_string(B.KS_OK) == "KS_OK" and B.status_string(B.KS_ESTATE) == "KS_ESTATE"


def test_null_and_bad_arguments_fail_before_cuda(lib):
    assert lib.ks_create(None, 0, None) == B.KS_EINVAL
    assert lib.ks_destroy(None) == B.KS_OK
    assert lib.ks_predict_kernels(None, None, 0, None, 0, 0, 0, None, None, None, None) == B.KS_EINVAL
    assert lib.ks_set_gelu_mode(None, 0) == B.KS_EINVAL
    assert lib.ks_set_head_output(None, 0, 0) == B.KS_EINVAL
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
    assert b.model_slot == B.KS_SLOT_FAMILY                          # no slot named: the family's
    assert B.make_batch(W.config_families(n=800).buckets[3]).model_slot == W.SLOT_ATTN_DECODE
    b1 = B.make_batch(W.config1().buckets[0])
    assert b1.col_dtype == B.KS_COL_F32
    bad = W.Bucket(0, [np.zeros(4, np.int64)] * 3)
    with pytest.raises(TypeError):
        B.make_batch(bad)
