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


def _segments_of(kind, rng):
    """(rows, q_off) descriptor tables with the shapes of the five BASELINE.json configs (no token data needed)."""
    rows, L = [], []
    if kind == "images":
        for r in range(64):
            rows.append((r, 1, 1, 576, 144)); L.append(int(rng.integers(16, 65)))
    elif kind == "video":
        for r in range(8):
            rows.append((r, 2, 32, 576, 2765)); L.append(48)
    elif kind == "audio":
        for r in range(16):
            rows.append((r, 1, 1, 576, 144)); rows.append((r, 3, 1500, 1, 600)); L.append(64)
    elif kind == "ragged":
        for r in range(256):
            n = int(rng.integers(144, 2881))
            rows.append((r, 1, 1, n, 1) if rng.integers(2) else (r, 2, 5, n // 5, 1)); L.append(int(rng.integers(8, 129)))
    elif kind == "tiny":
        rows, L = [(0, 1, 1, 7, 1), (1, 2, 3, 5, 2)], [3, 128]
    return rows, np.concatenate([[0], np.cumsum(L)]).astype(np.int64)


@pytest.mark.parametrize("kind", ["images", "video", "audio", "ragged", "tiny"])
def test_score_schedule_covers_every_row_once_and_is_balanced(B, kind):
    rng = np.random.default_rng(7)
    rows, q_off = _segments_of(kind, rng)
    t = B.score_schedule(rows, q_off, 4096, B.MAS_BF16, 148)
    N = sum(r[2] * r[3] for r in rows)
    assert len(t) > 0
    cov = np.zeros(N, np.int32)
    seg_of_row = np.concatenate([np.full(r[2] * r[3], k) for k, r in enumerate(rows)])
    row0, P_of, q0_of = np.cumsum([0] + [r[2] * r[3] for r in rows]), [r[3] if r[2] > 1 else 0 for r in rows], [int(q_off[r[0]]) for r in rows]
    for cta, rs, n, q0, L, pd, key, _ in t:
        k = seg_of_row[rs]
        # 256 = a double tile (non-temporal segments only); 384 = a tall one (three accumulator halves 64 TMEM columns apart:
        # needs L <= 64; cut only from short segments)
        tall_ok = not pd and L <= 64 and rows[k][2] * rows[k][3] <= 768
        assert 1 <= n <= (128 if pd else 384 if tall_ok else 256) and 0 <= cta < 148
        cov[rs:rs + n] += 1
        pd_expected = P_of[k]
        assert seg_of_row[rs + n - 1] == k                       # a tile never straddles a segment
        assert q0 == q0_of[k] and L == q_off[rows[k][0] + 1] - q_off[rows[k][0]] and pd == P_of[k]
        assert key == (min(max(P_of[k] - (rs - row0[k]), 0), n) if pd else 0)   # rows of frame 0 have no previous frame
    assert cov.min() == 1 and cov.max() == 1                     # every row exactly once
    assert np.all(np.diff(t[:, 0]) >= 0)                         # grouped per CTA, CTAs in order
    for c in np.unique(t[:, 0]):
        assert np.all(np.diff(t[t[:, 0] == c, 1]) > 0)           # ascending rows inside a CTA
    if N >= 148 * 128:
        # the schedule balances bytes pulled into the SM, not rows: token rows (+25 % when a previous-frame tile rides
        # along), 0.7 per padded query row, a per-tile constant (csrc/k_score_tc.cuh TcCost)
        rows16 = (t[:, 2] + 15) // 16 * 16
        has_prev = (t[:, 5] > 0) & (t[:, 6] < t[:, 2])
        cost = rows16 * (1.0 + 0.25 * has_prev) + 0.7 * ((t[:, 4] + 15) // 16 * 16) + 50.0
        load = np.bincount(t[:, 0], weights=cost, minlength=148)
        assert load.max() <= 1.2 * load.mean()     # a batch of 64 images is only ~1.4 tiles per CTA
        if len(t) >= 4 * 148:   # rows follow the cost only where a CTA holds several tiles (else one tall tile vs several short ones)
            assert np.bincount(t[:, 0], weights=rows16, minlength=148).max() <= 1.3 * rows16.sum() / 148


def test_score_schedule_rejects_bad_descriptors_and_generic_shapes(B):
    rows, q_off = [(0, 1, 1, 576, 144)], np.array([0, 32], np.int64)
    assert len(B.score_schedule(rows, q_off, 1024, B.MAS_F32)) == 0          # fp32 takes the generic path
    assert len(B.score_schedule(rows, q_off, 1000, B.MAS_BF16)) == 0         # d % 64 != 0 too
    with pytest.raises(B.MasError):
        B.score_schedule(rows, np.array([0, 0], np.int64), 1024, B.MAS_BF16)  # L = 0
