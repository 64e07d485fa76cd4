"""No-GPU checks of the C-ABI boundary: the library loads, exports every symbol include/msas.h declares, the host
helpers compute the documented values, and argument validation rejects bad tables before any CUDA call."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2604_02945_b200 import build
    build.build()
    from paper_2604_02945_b200 import binding
    return binding


def test_exports_match_header(B):
    hdr = open(os.path.join(ROOT, "include", "msas.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mas_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    for name in declared:
        assert hasattr(B.lib, name), name


def test_struct_layouts(B):
    assert C.sizeof(B.mas_segment) == 32 and C.sizeof(B.mas_params) == 40 and C.sizeof(B.mas_segment_out) == 36
    assert C.sizeof(B.mas_outputs) == 80


def test_host_helpers(B):
    assert B.lib.mas_version() == 100
    p = B.default_params()
    assert (round(p.lambda_spatial, 6), round(p.lambda_temp, 6), round(p.tau_s, 6), p.kappa, p.cut, p.select_mode) == (0.6, 0.4, 0.3, 10.0, 0.5, 0)
    assert B.keep_count(576, 0.25) == 144 and B.keep_count(18432, 0.15) == 2765 and B.keep_count(1500, 0.40) == 600
    assert B.keep_count(10, 0.0) == 1 and B.keep_count(10, 2.0) == 10
    assert B.lib.mas_status_string(2).decode().startswith("unsupported")


def test_validation_before_cuda(B):
    segs, n = B.make_segments([(0, 1, 1, 576, 144), (1, 2, 4, 100, 50)])
    ok, nbytes = B.workspace_bytes(segs, 2, [0, 16, 48], 4096, B.MAS_BF16)
    assert ok == B.MAS_OK and nbytes > n * 17
    assert B.workspace_bytes(segs, 2, [0, 16, 48], 4100, B.MAS_BF16)[0] == B.MAS_ERR_UNSUPPORTED      # d % 8
    assert B.workspace_bytes(segs, 2, [0, 16, 48], 4100, B.MAS_F32)[0] == B.MAS_OK                    # d % 4 is fine for fp32
    assert B.workspace_bytes(segs, 2, [0, 16, 16], 4096, B.MAS_BF16)[0] == B.MAS_ERR_UNSUPPORTED      # L = 0
    assert B.workspace_bytes(segs, 2, [0, 16, 16 + 129], 4096, B.MAS_BF16)[0] == B.MAS_ERR_UNSUPPORTED  # L > 128
    assert B.workspace_bytes(segs, 2, [1, 16, 48], 4096, B.MAS_BF16)[0] == B.MAS_ERR_INVALID_ARG
    segs[1].row0 = 577                                                                                 # gap in the tiling
    assert B.workspace_bytes(segs, 2, [0, 16, 48], 4096, B.MAS_BF16)[0] == B.MAS_ERR_INVALID_ARG
    segs[1].row0 = 576
    segs[1].request = 5
    assert B.workspace_bytes(segs, 2, [0, 16, 48], 4096, B.MAS_BF16)[0] == B.MAS_ERR_INVALID_ARG
    # keep_k is validated at plan creation (needs params): no CUDA call is reached
    segs, _ = B.make_segments([(0, 1, 1, 576, 577)])
    h = C.c_void_p()
    q = np.array([0, 4], np.int64)
    prm = B.default_params()
    st = B.lib.mas_plan_create(C.byref(h), segs, 1, q.ctypes.data_as(C.POINTER(C.c_int64)), 1, 64, B.MAS_BF16, C.byref(prm),
                               C.c_void_p(256), 1 << 30, None)
    assert st == B.MAS_ERR_INVALID_ARG
    prm.lambda_spatial = 0.9
    segs[0].keep_k = 10
    st = B.lib.mas_plan_create(C.byref(h), segs, 1, q.ctypes.data_as(C.POINTER(C.c_int64)), 1, 64, B.MAS_BF16, C.byref(prm),
                               C.c_void_p(256), 1 << 30, None)
    assert st == B.MAS_ERR_INVALID_ARG                                                                  # lambda_sp + lambda_t > 1
    prm = B.default_params()
    st = B.lib.mas_plan_create(C.byref(h), segs, 1, q.ctypes.data_as(C.POINTER(C.c_int64)), 1, 64, B.MAS_BF16, C.byref(prm),
                               C.c_void_p(256), 16, None)
    assert st == B.MAS_ERR_WORKSPACE


def test_product_does_not_import_oracle():
    # the product path must never route through oracle/
    pkg = os.path.join(ROOT, "paper_2604_02945_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "mas_ref_" not in src and "mas_oracle" not in src, f
