"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/festina_eval.h declares; struct layouts agree between the header and the numpy dtypes."""
from __future__ import annotations

import os
import re
import subprocess
import tempfile

import pytest

import paper_2606_30391_b200 as fs
from paper_2606_30391_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "festina_eval.h")


def test_library_exports_every_declared_symbol():
    fs.build_library()
    L = fs.lib()
    text = open(HEADER).read()
    declared = set(re.findall(r"\b(fs_[a-z_]+)\s*\(", text))
    assert declared == set(fs.SYMBOLS), declared ^ set(fs.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    assert L.fs_strerror(0) == b"ok" and L.fs_strerror(-4) != b"unknown"


def test_struct_sizes_match_header():
    """Compile a C program against the header and compare sizeof with the numpy record dtypes."""
    src = r'''
#include <stdio.h>
#include "festina_eval.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu\n", sizeof(fs_tenant), sizeof(fs_gpu_state),
         sizeof(fs_request), sizeof(fs_model_info), sizeof(fs_placement), sizeof(fs_local_cfg),
         sizeof(fs_consol_out), sizeof(fs_dims), sizeof(fs_params));
  return 0;
}'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "t.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "t")
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        got = [int(x) for x in subprocess.check_output([exe]).split()]
    want = [synth.TENANT_DT.itemsize, synth.GPU_STATE_DT.itemsize, synth.REQUEST_DT.itemsize,
            synth.MODEL_INFO_DT.itemsize, synth.PLACEMENT_DT.itemsize, synth.LOCAL_CFG_DT.itemsize,
            synth.CONSOL_DT.itemsize, 16, 16]
    assert got == want


def test_no_cpu_fallback_without_a_device():
    """Without a CUDA device fs_create fails with FS_ERR_CUDA; nothing computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(fs.FestinaError) as e:
        fs.Festina(0)
    assert e.value.code == fs.FS_ERR_CUDA


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_30391_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "festina_oracle" not in text, f


def test_static_plan_entry_point_validates_before_it_touches_cuda():
    """fs_replace_plan_static (the no-allocation entry point): bad counts and a size beyond the built-in scratch array
    are refused from the host-visible arguments alone; without a device a well-formed call fails with FS_ERR_CUDA."""
    import ctypes as C
    import torch
    L = fs.lib()
    one = (C.c_int32 * 4)()
    buf = (C.c_uint8 * 64)()
    assert L.fs_replace_plan_static(-1, buf, 8, 1.0, one, one, None) == fs.FS_ERR_ARG
    assert L.fs_replace_plan_static(1, None, 8, 1.0, one, one, None) == fs.FS_ERR_ARG
    assert L.fs_replace_plan_static(1, buf, 0, 1.0, one, one, None) == fs.FS_ERR_ARG          # s_eff < 1
    assert L.fs_replace_plan_static(1, buf, 33, 1.0, one, one, None) == fs.FS_ERR_ARG         # s_eff > FS_MAX_S
    assert L.fs_replace_plan_static(fs.FS_PLAN_STATIC_MAX_N + 1, buf, 8, 1.0, one, one, None) == fs.FS_ERR_SHAPE
    text = open(HEADER).read()
    assert re.search(r"#define\s+FS_PLAN_STATIC_MAX_N\s+%d\b" % fs.FS_PLAN_STATIC_MAX_N, text)
    if not torch.cuda.is_available():
        assert L.fs_replace_plan_static(0, None, 8, 1.0, None, one, None) == fs.FS_ERR_CUDA
