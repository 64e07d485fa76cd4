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


def _block_sweeps(t, nk):
    """(scored row range, first K-chunk, end K-chunk) of every block of a schedule record (include/msas.h, mas_score_schedule):
    the last block joins at k0, block 0 leaves at k1 (a one-block record: [k0, k1)), the blocks in between are swept over all of K."""
    cta, row0, n, nb, stride, mode, prev, halo = [int(v) for v in t[:8]]
    k0, k1 = int(t[12]), int(t[13])
    out = []
    for b in range(nb):
        if mode == 0:
            lo, hi = row0 + b * stride, row0 + min(n, (b + 1) * stride)
        elif mode == 1:
            lo, hi = row0 + b * stride, row0 + b * stride + n
        else:   # window b: 128 rows from row0 + b * stride on, scored from `prev` on (the record's first window: from `halo` on)
            lo, hi = row0 + b * stride + (halo if b == 0 else prev), row0 + min(n, b * stride + 128)
        out.append(((lo, hi), k0 if b == nb - 1 else 0, k1 if b == 0 else nk))
    return out


@pytest.mark.parametrize("kind", ["images", "video", "audio", "ragged", "tiny"])
def test_score_schedule_covers_every_row_once_and_is_balanced(B, kind):
    rng = np.random.default_rng(7)
    rows, q_off = _segments_of(kind, rng)
    d = 4096
    t = B.score_schedule(rows, q_off, d, B.MAS_BF16, 148)
    N = sum(r[2] * r[3] for r in rows)
    assert len(t) > 0
    nk = d // 64
    cov = np.zeros(N, np.int32)                                  # K-chunks swept per row: every row needs all nk of them, once
    owned = np.zeros(N, np.int32)                                # tiles that WRITE the row's results
    seg_of_row = np.concatenate([np.full(r[2] * r[3], k) for k, r in enumerate(rows)])
    row0_of, q0_of = np.cumsum([0] + [r[2] * r[3] for r in rows]), [int(q_off[r[0]]) for r in rows]
    maxL = int(np.diff(q_off).max())
    n_slots = min(10, 512 // ((maxL + 15) // 16 * 16))           # TMEM accumulator slots of pad16(longest query block) columns
    cost = np.zeros(148)
    split_open = None                                            # (rows, next k0, owner record) of a block being shared along K
    prev_nb, prev_epi = 0, 0.0
    for rec in t:
        cta, r0, n, nb, stride, mode, prev, halo, q0, L, seg, part0, k0, k1, n_wait, peer = [int(v) for v in rec]
        T, P = rows[seg][2], rows[seg][3]
        assert 0 <= cta < 148 and 1 <= nb <= n_slots
        assert q0 == q0_of[seg] and L == q_off[rows[seg][0] + 1] - q_off[rows[seg][0]]
        assert mode == (0 if T == 1 else 1 if P >= 64 else 2)
        assert 0 <= k0 < nk and 0 < k1 <= nk and k0 % 2 == 0 and k1 % 2 == 0   # two K-slices per chunk at d % 128 == 0
        if mode == 0:
            assert stride % 8 == 0 and stride <= 128 and prev == 0 and halo == 0 and nb == -(-n // stride)   # blocks of one height
            assert (r0 - row0_of[seg]) % 8 == 0                                                   # cut at whole 8-row swizzle atoms
        elif mode == 1:
            assert stride == P and prev == P and 1 <= n <= 128 and halo in (0, 1)
            t0 = (r0 - row0_of[seg]) // P
            assert halo == (1 if t0 > 0 else 0) and t0 + nb <= T          # frame t0 - 1 exists iff halo
            assert (r0 - row0_of[seg]) % P + n <= P                        # the patch rows of one frame
        else:
            assert stride == 128 - P and prev == P and halo in (0, P)
            assert halo == (0 if r0 == row0_of[seg] else P)               # only a segment's first window starts without predecessors
            assert nb == (1 if n <= 128 else -(-(n - 128) // stride) + 1)
            assert n - (nb - 1) * stride > P                               # the last window scores at least one row
        sweeps = _block_sweeps(rec, nk)
        for (lo, hi), ka, kb in sweeps:
            assert lo < hi and seg_of_row[lo] == seg and seg_of_row[hi - 1] == seg    # a tile never straddles a segment
            assert 0 <= ka < kb <= nk
            cov[lo:hi] += kb - ka
            if kb == nk:
                owned[lo:hi] += 1
        mine = t[t[:, 0] == cta]
        # K-split: a block shared along K is the last block of its owner (the part that ends at chunk nk; last tile of its CTA) and
        # the first block of the first tile of every CTA that follows, in descending K, until chunk 0 is reached
        if k1 < nk:
            assert split_open is not None and sweeps[0][0] == split_open[0] and k1 == split_open[1] and cta == split_open[2] + 1
            assert np.array_equal(rec, mine[0])
            split_open[1], split_open[2], split_open[3] = sweeps[0][1], cta, split_open[3] - 1
            if sweeps[0][1] == 0:
                assert split_open[3] == 0
                split_open = None
        if k0 > 0 and (nb > 1 or k1 == nk):
            assert split_open is None and n_wait >= 1 and peer == cta + 1 and np.array_equal(rec, mine[-1])
            split_open = [sweeps[-1][0], k0, cta, n_wait]
        else:
            assert n_wait == 0 and peer == -1
        # cost model of csrc/k_score_tc.cuh (TcCost), about microseconds: a block 14 + 0.025 h (x 1.28 in a frame walk, x 1.7 for a window
        # of a short-frame segment) by its share of K; per tile (by its share of K) 0.055 per padded query row and 0.077 per row of a
        # halo chunk; 1.5 per tile; and the wait for accumulator slots the CTA's previous tile still holds (0.35 + 0.013 columns each)
        share = sum(kb - ka for _, ka, kb in sweeps) / nk          # in blocks
        h = rows[seg][3] / -(-rows[seg][3] // 128) if mode == 0 else n if mode == 1 else 128
        blocks = share * (1.0, 1.28, 1.7)[mode] * (14 + 0.025 * h)
        tile_share = share if nb == 1 else 1.0
        Lpad = (L + 15) // 16 * 16
        first_of_cta = np.array_equal(rec, mine[0])
        wait = 0.0 if first_of_cta else prev_epi * max(0, prev_nb + nb - n_slots)
        cost[cta] += blocks + tile_share * (0.055 * Lpad + (0.077 * n if mode == 1 and (halo or k1 < nk) else 0)) + 1.5 + wait
        prev_nb, prev_epi = nb, 0.35 + 0.013 * Lpad
    assert split_open is None
    assert cov.min() == nk and cov.max() == nk                   # every K-chunk of every row swept exactly once
    assert owned.min() == 1 and owned.max() == 1                 # and its results written by exactly one tile
    assert np.all(np.diff(t[:, 0]) >= 0)                         # grouped per CTA, CTAs in order
    if N >= 148 * 128:
        # equal cost per CTA: K-split fills every CTA to the common target
        assert np.count_nonzero(cost) >= 140 and cost.max() <= 1.10 * cost.sum() / 148, (cost.max(), cost.sum() / 148)


def test_score_schedule_rider_variant_and_small_devices(B):
    """Few SMs, and a long single-frame segment: tiles of up to 4 blocks (L = 128), every K-chunk of every row once."""
    rows, q_off = [(0, 1, 1, 5000, 10), (1, 2, 9, 100, 10), (2, 3, 700, 1, 10)], np.array([0, 64, 70, 198], np.int64)
    for sms in (1, 3, 148):
        t = B.score_schedule(rows, q_off, 128, B.MAS_BF16, sms)
        cov = np.zeros(5000 + 900 + 700, np.int32)
        for rec in t:
            assert int(rec[3]) <= 4                              # L = 128 somewhere: four 128-column accumulator slots
            for (lo, hi), ka, kb in _block_sweeps(rec, 2):
                cov[lo:hi] += kb - ka
        assert cov.min() == 2 and cov.max() == 2 and t[:, 0].max() < sms      # d = 128: two K-chunks


def test_score_schedule_rejects_bad_descriptors_and_generic_shapes(B):
    rows, q_off = [(0, 1, 1, 576, 144)], np.array([0, 32], np.int64)
    assert len(B.score_schedule(rows, q_off, 1024, B.MAS_F32)) == 0          # fp32 takes the generic path
    assert len(B.score_schedule(rows, q_off, 1000, B.MAS_BF16)) == 0         # d % 64 != 0 too
    with pytest.raises(B.MasError):
        B.score_schedule(rows, np.array([0, 0], np.int64), 1024, B.MAS_BF16)  # L = 0
