"""Pins of the CPU oracle against what the paper and the mathematics fix (SPEC.md, SURVEY.md §8(c) "Pins").
No GPU.  Each test is chosen so that a plausible mistake in oracle/mas_oracle.cpp (dropped term, wrong sign or index,
transposed operand, wrong normalisation) fails it.  Expected values come from tests/golden/closed_forms.txt (hand
expansions of the paper's equations), from brute force written independently here, or from numpy float64."""
import math
import os

import numpy as np
import pytest

from oracle import mas_ref as O
from paper_2604_02945_b200 import synth

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            GOLD[k.strip()] = float(v)


def seg1(T, P, k=1, req=0, mod=1):
    return O.make_segments([(req, mod, T, P, k)])[0]


def f32(a):
    return np.ascontiguousarray(a, np.float32)


# ---------------------------------------------------------------- S0 / S3: dot products, norms, cosine
def test_dot_products_hand_expanded():
    X = f32([[1, 2, 3, 4], [0, -1, 2, -3]])
    Q = f32([[1, 0, -1, 2], [2, 2, 2, 2], [-1, 3, 0, 1]])
    rel, S = O.crossmodal(seg1(1, 2), [0, 3], X, Q, want_S=True)
    exp = np.array([[GOLD["S_00"], GOLD["S_01"], GOLD["S_02"]], [GOLD["S_10"], GOLD["S_11"], GOLD["S_12"]]])
    assert np.array_equal(S, exp)          # a transposed operand or wrong stride breaks this
    xn = np.array([math.sqrt(30), math.sqrt(14)])
    qn = np.array([math.sqrt(6), 4.0, math.sqrt(11)])
    cos = exp / xn[:, None] / qn[None, :]
    assert np.allclose(rel, cos.max(axis=1), rtol=0, atol=1e-15)
    assert rel[1] < 0                       # max of all-negative cosines stays negative (no clamp at 0)


def test_cosine_closed_forms_and_zero_rows():
    X = f32([[1, 0], [1, 1], [0, 0]])
    Q = f32([[1, 0], [0, 1]])
    rel = O.crossmodal(seg1(1, 3), [0, 2], X, Q)
    assert rel[0] == 1.0
    assert abs(rel[1] - GOLD["cos_11_vs_axes"]) < 1e-15
    assert rel[2] == 0.0                    # G18: zero row -> cos := 0
    rel = O.crossmodal(seg1(1, 3), [0, 2], X, f32([[0, 0], [0, -1]]))
    assert rel[0] == 0.0 and rel[1] == 0.0  # zero query contributes cos 0, which beats -1/sqrt2


def test_crossmodal_matches_numpy_float64_and_bf16_decoding():
    rng = np.random.default_rng(7)
    N, L, d = 12, 5, 40
    Xf = rng.standard_normal((N, d)).astype(np.float32)
    Qf = rng.standard_normal((2 * L, d)).astype(np.float32)
    Xb, Qb = synth.f32_to_bf16_bits(Xf), synth.f32_to_bf16_bits(Qf)
    segs, _ = O.make_segments([(0, 1, 1, 7, 1), (1, 1, 1, 5, 1)])
    rel, S = O.crossmodal(segs, [0, L, 2 * L], Xb, Qb, want_S=True)
    X64 = synth.bf16_bits_to_f32(Xb).astype(np.float64)
    Q64 = synth.bf16_bits_to_f32(Qb).astype(np.float64)
    for (lo, hi, q0) in [(0, 7, 0), (7, 12, L)]:      # each request uses only its own queries
        Sx = X64[lo:hi] @ Q64[q0:q0 + L].T
        assert np.allclose(S[lo:hi, :L], Sx, rtol=1e-13, atol=1e-13)
        cos = Sx / np.linalg.norm(X64[lo:hi], axis=1)[:, None] / np.linalg.norm(Q64[q0:q0 + L], axis=1)[None, :]
        assert np.allclose(rel[lo:hi], cos.max(axis=1), rtol=1e-13)


def test_query_permutation_and_duplicate_query_are_bit_invariant():
    w = synth.batched_images(seed=11, R=2, d=64, L_lo=6, L_hi=6)
    segs, _ = O.make_segments(w.segments)
    prm = O.default_params()
    a = O.forward(segs, w.q_off, prm, w.X, w.Q, want_Y=False)
    perm = np.concatenate([np.random.default_rng(1).permutation(6), 6 + np.random.default_rng(2).permutation(6)])
    b = O.forward(segs, w.q_off, prm, w.X, w.Q[perm], want_Y=False)
    for k in ("rel", "mas_tok", "m_spatial", "keep_mask", "kept_idx"):
        assert np.array_equal(a[k], b[k]), k
    # appending a duplicate query to every request changes nothing
    Q2 = np.concatenate([w.Q[0:6], w.Q[0:1], w.Q[6:12], w.Q[7:8]])
    c = O.forward(segs, np.array([0, 7, 14]), prm, w.X, Q2, want_Y=False)
    for k in ("rel", "mas_tok", "keep_mask"):
        assert np.array_equal(a[k], c[k]), k


# ---------------------------------------------------------------- S1: RMS, standardise, sigmoid, rho
def test_spatial_two_rows_closed_form():
    X = f32([[1, -1, 1, -1], [3, 3, -3, -3]])       # RMS 1 and 3
    s = O.rms(seg1(1, 2), X)
    assert np.array_equal(s, [1.0, 3.0])
    m, mas, out = O.fuse(seg1(1, 2), O.default_params(), s, np.zeros(2), np.zeros(2))
    assert abs(m[0] - GOLD["sigmoid_minus1"]) < 1e-15 and abs(m[1] - GOLD["sigmoid_plus1"]) < 1e-15
    assert out[0].rho_spatial == GOLD["rho_two_rows"]
    assert out[0].mean_s == 2.0 and out[0].std_s == 1.0


def test_spatial_constant_segment_and_strict_threshold():
    s = np.full(5, 2.5)
    m, _, out = O.fuse(seg1(1, 5), O.default_params(), s, np.zeros(5), np.zeros(5))
    assert np.all(m == 0.5) and out[0].rho_spatial == 0.0           # G18: den_s floor, z -> 0
    m, _, out = O.fuse(seg1(1, 5), O.default_params(tau_s=0.5), s, np.zeros(5), np.zeros(5))
    assert out[0].rho_spatial == 0.0                                 # strict '<' (G12): M == tau is not below
    s0 = np.zeros(4)
    m, _, out = O.fuse(seg1(1, 4), O.default_params(), s0, np.zeros(4), np.zeros(4))
    assert np.all(m == 0.5)                                          # den_s = 0 -> z = 0


def test_spatial_statistics_bruteforce():
    rng = np.random.default_rng(3)
    s = np.abs(rng.standard_normal(257)) + 0.1
    prm = O.default_params()
    m, _, out = O.fuse(seg1(1, 257), prm, s, np.zeros(257), rng.standard_normal(257))
    z = (s - s.mean()) / s.std()
    assert abs(z.mean()) < 1e-12 and abs(z.var() - 1) < 1e-12
    assert np.allclose(m, 1 / (1 + np.exp(-z)), rtol=1e-13)
    assert np.all((m > 0) & (m < 1))
    assert out[0].rho_spatial == np.count_nonzero(m < 0.3) / 257
    assert 0 < out[0].rho_spatial < 1
    # RMS itself against numpy on random bf16 data
    Xb = synth.f32_to_bf16_bits(rng.standard_normal((9, 24)).astype(np.float32))
    x64 = synth.bf16_bits_to_f32(Xb).astype(np.float64)
    assert np.allclose(O.rms(seg1(1, 9), Xb), np.sqrt((x64 ** 2).mean(axis=1)), rtol=1e-14)


# ---------------------------------------------------------------- S2: temporal change
def test_temporal_closed_forms():
    a = [1.0, 2.0, -3.0, 0.5]
    rows = [a, a,                       # identical -> 0 exactly
            [-v for v in a],            # opposite of previous -> 1
            [-2 * v for v in a],        # doubled -> 1/3
            [0, 0, 0, 0],               # one zero row -> 1
            [0, 0, 0, 0],               # both zero -> 0 (G18)
            [3, 0, 0, 0], [0, 3, 0, 0]]  # orthogonal equal norm -> 1/sqrt2
    g = O.temporal(seg1(8, 1), f32(rows))
    assert g[0] == 1.0                                   # keyframe G6
    assert g[1] == 0.0
    assert g[2] == GOLD["gamma_opposite"]
    assert abs(g[3] - GOLD["gamma_doubled"]) < 1e-15
    assert g[4] == 1.0 and g[5] == 0.0
    assert g[6] == 1.0                                   # previous row is zero
    assert abs(g[7] - GOLD["gamma_orthogonal_equal_norm"]) < 1e-15


def test_temporal_indexing_frame_major_and_single_frame():
    # T=3 frames x P=2 patches: row (t,p) compares with (t-1,p), not with the adjacent row
    X = f32([[1, 0], [0, 1],      # t=0
             [1, 0], [0, -1],     # t=1: p0 identical, p1 opposite
             [2, 0], [0, -1]])    # t=2: p0 doubled, p1 identical
    g = O.temporal(seg1(3, 2), X)
    assert list(g[:2]) == [1.0, 1.0]
    assert g[2] == 0.0 and g[3] == 1.0
    assert abs(g[4] - 1 / 3) < 1e-15 and g[5] == 0.0
    assert np.all(O.temporal(seg1(1, 6), X) == 0.0)      # T = 1: not applicable
    # two segments: the second must not look into the first
    segs, _ = O.make_segments([(0, 1, 1, 2, 1), (0, 2, 2, 2, 1)])
    g = O.temporal(segs, X)
    assert list(g) == [0, 0, 1, 1, g[4], g[5]] and abs(g[4] - 1 / 3) < 1e-15 and g[5] == 0.0


def test_temporal_equal_norm_is_sin_half_angle_and_range():
    rng = np.random.default_rng(5)
    d = 6
    for _ in range(20):
        u = rng.standard_normal(d); u /= np.linalg.norm(u)
        v = rng.standard_normal(d); v /= np.linalg.norm(v)
        X = np.stack([u, v]).astype(np.float32)
        x64 = X.astype(np.float64)
        g = O.temporal(seg1(2, 1), X)[1]
        # general definition in float64 (norms are equal only up to fp32 rounding, so use the full formula) ...
        exp = np.linalg.norm(x64[1] - x64[0]) / (np.linalg.norm(x64[1]) + np.linalg.norm(x64[0]))
        assert abs(g - exp) < 1e-14 and 0 <= g <= 1
        # ... and the closed form sin(theta/2) for (nearly) equal norms
        cos = x64[0] @ x64[1] / np.linalg.norm(x64[0]) / np.linalg.norm(x64[1])
        assert abs(g - math.sqrt((1 - cos) / 2)) < 1e-6


def test_temporal_ar1_statistical_law():
    # AR(1) x_t = rho x_{t-1} + sqrt(1-rho^2) n: E|x_t - x_{t-1}|^2 = 2(1-rho)|x|^2 -> gamma ~ sqrt(2(1-rho))/2
    rng = np.random.default_rng(9)
    for rho, expect in ((0.95, 0.158), (0.9, 0.224)):
        d, T = 512, 200
        x = np.empty((T, d), np.float32)
        x[0] = rng.standard_normal(d)
        for t in range(1, T):
            x[t] = rho * x[t - 1] + math.sqrt(1 - rho * rho) * rng.standard_normal(d)
        g = O.temporal(seg1(T, 1), x)[1:]
        assert abs(g.mean() - expect) < 0.05 * expect


# ---------------------------------------------------------------- softmax / Eq. 7
def _fuse_segments(rows, s, gamma, rel, **kw):
    segs, n = O.make_segments(rows)
    return O.fuse(segs, O.default_params(**kw), s, gamma, rel)


def test_softmax_identities():
    rng = np.random.default_rng(2)
    rows = [(0, 1, 1, 4, 1), (0, 3, 3, 2, 1), (0, 2, 2, 3, 1), (1, 1, 1, 5, 1)]
    n = 4 + 6 + 6 + 5
    s, gam, rel = rng.random(n) + 0.5, rng.random(n), rng.standard_normal(n) * 0.1
    _, _, out = _fuse_segments(rows, s, gam, rel)
    beta = O.seg_out_array(out, "beta")
    assert abs(beta[:3].sum() - 1) < 1e-15 and beta[3] == 1.0      # one segment -> beta = 1
    alpha = np.array([rel[0:4].mean(), rel[4:10].mean(), rel[10:16].mean()])
    e = np.exp(10 * alpha)
    assert np.allclose(beta[:3], e / e.sum(), rtol=1e-13)          # kappa = 10 (G20)
    assert np.allclose(O.seg_out_array(out, "alpha_mean")[:3], alpha, rtol=1e-14)
    # shift invariance: adding a constant to every rel leaves beta unchanged; equal alpha -> 1/n
    _, _, out2 = _fuse_segments(rows, s, gam, rel + 0.25)
    assert np.allclose(O.seg_out_array(out2, "beta"), beta, rtol=1e-12)
    _, _, out3 = _fuse_segments(rows, s, gam, np.full(n, 0.3))
    assert np.allclose(O.seg_out_array(out3, "beta")[:3], 1 / 3, rtol=1e-15)


def test_eq7_special_cases():
    # single image segment: beta = 1, a = 0 -> MAS = lambda_sp * rho
    s = np.array([1.0, 3.0])
    _, _, out = _fuse_segments([(0, 1, 1, 2, 1)], s, np.zeros(2), np.zeros(2))
    assert abs(out[0].mas - GOLD["mas_single_image_rho_half"]) < 1e-15
    # single video segment, all frames identical (gamma = 0 beyond the keyframe) -> lambda_sp*rho + lambda_t
    s = np.array([1.0, 3.0, 1.0, 3.0, 1.0, 3.0])
    gam = np.array([1, 1, 0, 0, 0, 0.0])
    _, _, out = _fuse_segments([(0, 2, 3, 2, 1)], s, gam, np.zeros(6))
    assert out[0].gamma_avg == 0.0                                  # keyframe excluded (G6/G7)
    assert abs(out[0].mas - GOLD["mas_static_video_rho_half"]) < 1e-15
    # gamma_avg is the mean over frames t>=1 of per-frame patch means
    gam = np.array([1, 1, 0.2, 0.4, 0.6, 1.0])
    _, _, out = _fuse_segments([(0, 2, 3, 2, 1)], s, gam, np.zeros(6))
    assert abs(out[0].gamma_avg - 0.55) < 1e-15
    assert abs(out[0].mas - (1 - (1 - 0.6 * 0.5 - 0.4 * (1 - 0.55)))) < 1e-15
    # lambda weights are not swapped
    _, _, out = _fuse_segments([(0, 2, 3, 2, 1)], s, gam, np.zeros(6), lambda_spatial=0.9, lambda_temp=0.1)
    assert abs(out[0].mas - (0.9 * 0.5 + 0.1 * 0.45)) < 1e-15


def test_fuse_gain_bias_kappa_worked_example():
    """spatial_gain / spatial_bias / rel_gain / rel_bias / kappa away from their defaults (reading G2, G20): the hand-worked case of
    tests/golden/closed_forms.txt (fusep_*).  Swapping the two gains, or a sign error on a bias, changes every value below."""
    rows = [(0, 1, 1, 2, 1), (0, 1, 1, 2, 1)]
    s = np.array([1.0, 3.0, 2.0, 2.0])
    rel = np.array([0.1, 0.3, 0.5, 0.7])
    m, mas, out = _fuse_segments(rows, s, np.zeros(4), rel, spatial_gain=2.0, spatial_bias=-0.5, rel_gain=0.5, rel_bias=0.25, kappa=3.0)
    assert np.allclose(m, [GOLD["fusep_M_A0"], GOLD["fusep_M_A1"], GOLD["fusep_M_B"], GOLD["fusep_M_B"]], rtol=0, atol=1e-15)
    assert np.allclose(mas[:2], [GOLD["fusep_mas_A0"], GOLD["fusep_mas_A1"]], rtol=0, atol=1e-15)
    assert out[0].rho_spatial == 0.5 and out[1].rho_spatial == 0.0
    assert abs(out[0].beta - GOLD["fusep_beta_A"]) < 1e-15 and abs(out[0].beta + out[1].beta - 1) < 1e-15
    assert abs(out[0].mas - GOLD["fusep_mas_seg_A"]) < 1e-15 and abs(out[1].mas - GOLD["fusep_mas_seg_B"]) < 1e-15
    # the relevance sigmoid of the worked case, recovered from MAS_i = 1 - g (1 - lambda_sp (1 - M)) at T = 1
    g = (1 - mas[:2]) / (1 - 0.6 * (1 - m[:2]))
    assert np.allclose(g, [GOLD["fusep_g_A0"], GOLD["fusep_g_A1"]], rtol=0, atol=1e-15)


def test_fuse_nondefault_params_against_numpy_float64():
    """Every parameter of mas_ref_fuse away from its default, three segments of one request plus a single-segment request, against
    the formulas of SPEC S1 / S3 / S4 evaluated with numpy in float64."""
    rng = np.random.default_rng(11)
    rows = [(0, 1, 1, 7, 1), (0, 2, 4, 5, 1), (0, 3, 9, 1, 1), (1, 2, 3, 4, 1)]
    sizes = [T * P for (_, _, T, P, _) in rows]
    n = sum(sizes)
    s, gam, rel = rng.random(n) + 0.3, rng.random(n), 0.2 * rng.standard_normal(n)
    prm = dict(lambda_spatial=0.55, lambda_temp=0.35, tau_s=0.42, kappa=3.0, spatial_gain=2.0, spatial_bias=-0.5, rel_gain=0.5, rel_bias=0.25)
    m, mas, out = _fuse_segments(rows, s, gam, rel, **prm)
    sig = lambda u: 1.0 / (1.0 + np.exp(-u))
    r0, alphas, rhos, gavgs = 0, [], [], []
    for (_, _, T, P, _), nk in zip(rows, sizes):
        sl = slice(r0, r0 + nk)
        z = (s[sl] - s[sl].mean()) / s[sl].std()
        M = sig(2.0 * z - 0.5)
        g = sig(0.5 * (rel[sl] - rel[sl].mean()) / rel[sl].std() + 0.25)
        a = 1.0 if T > 1 else 0.0
        assert np.allclose(m[sl], M, rtol=1e-13, atol=0)
        assert np.allclose(mas[sl], 1 - g * (1 - 0.55 * (1 - M) - a * 0.35 * (1 - gam[sl])), rtol=1e-13, atol=0)
        alphas.append(rel[sl].mean()); rhos.append(np.count_nonzero(M < 0.42) / nk)
        gavgs.append(gam[sl].reshape(T, P)[1:].mean(axis=1).mean() if T > 1 else 0.0)
        r0 += nk
    e = np.exp(3.0 * np.array(alphas[:3]))
    beta = list(e / e.sum()) + [1.0]
    for k, (_, _, T, P, _) in enumerate(rows):
        a = 1.0 if T > 1 else 0.0
        assert abs(out[k].rho_spatial - rhos[k]) < 1e-15 and abs(out[k].gamma_avg - gavgs[k]) < 1e-14
        assert abs(out[k].beta - beta[k]) < 1e-13
        assert abs(out[k].mas - (1 - beta[k] * (1 - 0.55 * rhos[k] - a * 0.35 * (1 - gavgs[k])))) < 1e-13
    # the two gains are not interchangeable, nor are the two biases
    m2, mas2, _ = _fuse_segments(rows, s, gam, rel, **dict(prm, spatial_gain=0.5, rel_gain=2.0))
    assert not np.allclose(m2, m) and not np.allclose(mas2, mas)
    m3, mas3, _ = _fuse_segments(rows, s, gam, rel, **dict(prm, spatial_bias=0.25, rel_bias=-0.5))
    assert not np.allclose(m3, m) and not np.allclose(mas3, mas)


def test_per_token_mas_formula_ranges_and_monotonicity():
    rng = np.random.default_rng(4)
    n = 64
    s, gam, rel = rng.random(n) + 0.2, rng.random(n), rng.standard_normal(n)
    gam[:8] = 1.0
    rows = [(0, 2, 8, 8, 1)]
    m, mas, out = _fuse_segments(rows, s, gam, rel)
    g = 1 / (1 + np.exp(-(rel - rel.mean()) / rel.std()))
    exp = 1 - g * (1 - 0.6 * (1 - m) - 0.4 * (1 - gam))
    assert np.allclose(mas, exp, rtol=1e-13)
    assert np.all((mas >= 0) & (mas <= 1)) and 0 <= out[0].mas <= 1
    # T = 1: temporal term dropped even if a gamma array is supplied
    m1, mas1, _ = _fuse_segments([(0, 1, 1, 64, 1)], s, gam, rel)
    assert np.allclose(mas1, 1 - g * (1 - 0.6 * (1 - m1)), rtol=1e-13)
    # raising gamma_i (more change) never raises MAS_i; extreme token -> MAS near 0
    gam2 = gam.copy(); gam2[20] = min(1.0, gam[20] + 0.3)
    _, mas2, _ = _fuse_segments(rows, s, gam2, rel)
    assert mas2[20] <= mas[20] and np.array_equal(np.delete(mas2, 20), np.delete(mas, 20))
    s3, rel3 = s.copy(), rel.copy()
    s3[5] = 100.0; rel3[5] = 100.0
    g3 = gam.copy(); g3[5] = 1.0
    _, mas3, _ = _fuse_segments(rows, s3, g3, rel3)
    assert mas3[5] < 1e-3 and mas3[5] == mas3.min()


# ---------------------------------------------------------------- S5: selection and compaction
def test_keep_count_rule():
    assert O.keep_count(576, 0.25) == 144 and O.keep_count(18432, 0.15) == 2765 and O.keep_count(1500, 0.40) == 600
    assert O.keep_count(10, 0.0) == 1 and O.keep_count(10, 2.0) == 10 and O.keep_count(7, 0.5) == 4
    for n in (1, 5, 144, 577, 2880):
        for r in (0.1, 0.15, 0.25, 0.4, 1.0):
            assert O.keep_count(n, r) == synth.keep_count(n, r)


def test_topk_bruteforce_with_ties():
    rng = np.random.default_rng(8)
    rows = [(0, 1, 1, 9, 4), (0, 1, 1, 1, 1), (1, 2, 2, 5, 10), (2, 1, 1, 7, 3)]
    segs, n = O.make_segments(rows)
    vals = rng.integers(0, 4, n).astype(np.float64) / 4          # heavy ties
    X = rng.standard_normal((n, 8)).astype(np.float32)
    prm = O.default_params()
    mask, idx, off, Y, out = O.select_compact(segs, prm, X, vals)
    r0 = 0
    exp_idx = []
    for (_, _, T, P, k) in rows:
        ns = T * P
        order = sorted(range(r0, r0 + ns), key=lambda i: (vals[i], i))[:k]   # brute force: (MAS, index) order
        exp_idx += sorted(order)
        r0 += ns
    total = len(exp_idx)
    assert list(idx[:total]) == exp_idx
    assert list(off) == [0, 4, 5, 15, 18]
    assert [o.n_kept for o in out] == [4, 1, 10, 3]
    exp_mask = np.zeros(n, np.uint8); exp_mask[exp_idx] = 1
    assert np.array_equal(mask, exp_mask)
    assert np.array_equal(Y[:total], X[exp_idx])                  # byte-exact rows
    # explicit tie case: equal scores -> lower index wins
    segs, _ = O.make_segments([(0, 1, 1, 5, 2)])
    mask, idx, off, _, _ = O.select_compact(segs, prm, X[:5], np.array([0.5, 0.2, 0.5, 0.2, 0.2]))
    assert list(idx[:2]) == [1, 3] and list(mask) == [0, 1, 0, 1, 0]


def test_threshold_mode_and_cap_overflow():
    rng = np.random.default_rng(10)
    rows = [(0, 1, 1, 6, 6), (1, 1, 1, 5, 5), (2, 1, 1, 4, 4)]
    segs, n = O.make_segments(rows)
    vals = np.array([0.5, 0.50001, 0.1, 0.9, 0.5, 0.0, 0.9, 0.8, 0.7, 0.6, 0.51, 0.3, 0.5, 0.2, 1.0])
    Xb = synth.f32_to_bf16_bits(rng.standard_normal((n, 16)).astype(np.float32))
    prm = O.default_params(select_mode=1, cut=0.5)
    mask, idx, off, Y, out = O.select_compact(segs, prm, Xb, vals)
    exp = [i for i in range(n) if vals[i] <= 0.5]                 # inclusive (G17)
    assert exp == [0, 2, 4, 5, 11, 12, 13]
    assert list(idx[:len(exp)]) == exp and list(off) == [0, 4, 4, 7]   # a segment may keep 0 tokens
    assert np.array_equal(Y[:len(exp)], Xb[exp])
    # cap smaller than the total: nothing past the cap, true total still reported
    mask2, idx2, off2, Y2, _ = O.select_compact(segs, prm, Xb, vals, cap_rows=5)
    assert list(idx2) == exp[:5] and off2[-1] == 7 and np.array_equal(mask2, mask)


# ---------------------------------------------------------------- whole-pass invariances
def test_power_of_two_scaling_is_bit_invariant():
    w = synth.video(seed=21, R=2, T=4, P=12, d=64, L=5)
    segs, _ = O.make_segments(w.segments)
    prm = O.default_params()
    a = O.forward(segs, w.q_off, prm, w.X, w.Q, want_Y=False)
    Xs = synth.f32_to_bf16_bits(synth.bf16_bits_to_f32(w.X) * np.float32(4.0))
    Qs = synth.f32_to_bf16_bits(synth.bf16_bits_to_f32(w.Q) * np.float32(0.25))
    b = O.forward(segs, w.q_off, prm, Xs, Qs, want_Y=False)
    for k in ("m_spatial", "gamma", "rel", "mas_tok", "keep_mask", "kept_idx"):
        assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(O.seg_out_array(a["seg_out"], "mas"), O.seg_out_array(b["seg_out"], "mas"))


def test_row_permutation_of_image_segment():
    w = synth.batched_images(seed=22, R=1, d=48, L_lo=4, L_hi=4)
    segs, n = O.make_segments(w.segments)
    prm = O.default_params()
    a = O.forward(segs, w.q_off, prm, w.X, w.Q, want_Y=False)
    perm = np.random.default_rng(0).permutation(n)
    b = O.forward(segs, w.q_off, prm, w.X[perm], w.Q, want_Y=False)
    for k in ("m_spatial", "rel", "mas_tok"):
        assert np.allclose(a[k][perm], b[k], rtol=1e-11, atol=1e-13), k
    for f in ("rho_spatial", "alpha_mean", "beta", "mas"):
        assert np.allclose(O.seg_out_array(a["seg_out"], f), O.seg_out_array(b["seg_out"], f), rtol=1e-11), f


def test_forward_equals_staged_composition_and_static_patches_are_zero():
    w = synth.video(seed=23, R=2, T=5, P=576, d=32, L=6)
    segs, n = O.make_segments(w.segments)
    prm = O.default_params()
    full = O.forward(segs, w.q_off, prm, w.X, w.Q)
    gam = O.temporal(segs, w.X)
    assert np.array_equal(full["gamma"], gam)
    # static background patches are bit copies (unless the salient block touched them in either frame) -> gamma == 0
    P = 576
    for r in range(2):
        static = w.meta["static"][r]
        base = r * 5 * P
        for t in range(1, 5):
            rows = base + t * P + np.nonzero(static)[0]
            same = np.all(w.X[rows] == w.X[rows - P], axis=1)
            assert same.sum() > 0.4 * P
            assert np.all(gam[rows[same]] == 0.0)
            assert np.all(gam[rows[~same]] > 0.0)
    m, mas, out = O.fuse(segs, prm, O.rms(segs, w.X), gam, O.crossmodal(segs, w.q_off, w.X, w.Q))
    assert np.array_equal(mas, full["mas_tok"]) and np.array_equal(m, full["m_spatial"])
    mask, idx, off, Y, _ = O.select_compact(segs, prm, w.X, mas)
    assert np.array_equal(mask, full["keep_mask"]) and np.array_equal(idx, full["kept_idx"]) and np.array_equal(Y, full["Y"])
    # structural checks on the selection
    for k, (_, _, T, Pn, kk) in enumerate(w.segments):
        sl = idx[off[k]:off[k + 1]]
        assert len(sl) == kk and np.all(np.diff(sl) > 0)
        assert sl.min() >= segs[k].row0 and sl.max() < segs[k].row0 + T * Pn
    assert mask.sum() == off[-1]


def test_planted_salient_tokens_are_preferentially_kept():
    # sanity of the instantiation (not parity): salient, query-aligned rows should mostly survive the 25 % top-k
    w = synth.batched_images(seed=24, R=3, d=256)
    segs, _ = O.make_segments(w.segments)
    r = O.forward(segs, w.q_off, O.default_params(), w.X, w.Q, want_Y=False)
    kept = r["keep_mask"].astype(bool)
    recall = (kept & w.salient).sum() / max(1, min(w.salient.sum(), kept.sum()))
    assert recall > 0.6


# ---------------------------------------------------------------- NEXT-1: literal LSH probe (Eq. 5)
def test_lsh_hand_expanded_bits():
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")):
        if line.startswith("lsh_"):
            k, v = line.split("#")[0].split("=")
            gold[k.strip()] = float(v)
    R = np.zeros((64, 4), np.float32)
    R[0], R[1], R[2], R[3] = (1, 1, 1, 1), (-1, 0, 0, 0), (2, 1, 5, 0), (0, 0, 0, -1)
    X = np.array([[1, -2, 0, 3], [-1, 2, 0, -3]], np.float32)
    segs = seg1(2, 1)
    sig, g, proj = O.temporal_lsh(segs, X, R, want_proj=True)
    low4 = (sig & np.uint64(15)).astype(int)
    assert low4[0] == int(gold["lsh_bits_x"]) and low4[1] == int(gold["lsh_bits_negx"])
    assert np.all((sig >> np.uint64(4)) == np.uint64((1 << 60) - 1))          # zero rows of R project to 0 -> bit set
    assert list(proj[0, :4]) == [2, -1, 0, -3]
    assert g[0] == 1.0 and g[1] == gold["lsh_gamma_x_vs_negx_4hashes"]         # keyframe; 3 of 64 bits differ


def test_lsh_identical_negated_scaled_and_single_frame():
    rng = np.random.default_rng(5)
    d, P = 32, 6
    R = rng.standard_normal((64, d)).astype(np.float32)
    f0 = rng.standard_normal((P, d)).astype(np.float32)
    X = np.concatenate([f0, f0, -f0, 4.0 * f0]).astype(np.float32)            # frames: x, x, -x, 4x
    segs = seg1(4, P)
    sig, g = O.temporal_lsh(segs, X, R)
    assert np.all(g[:P] == 1.0)                                                # keyframe (G6)
    assert np.all(g[P:2 * P] == 0.0)                                           # identical rows -> identical signatures
    assert np.all(g[2 * P:3 * P] == 1.0)                                       # negation flips every (non-zero) projection
    assert np.all(g[3 * P:] == 1.0) and np.array_equal(sig[3 * P:], sig[:P])   # 4x has x's signature; vs -x all differ
    segs1 = seg1(1, 4 * P)
    assert np.all(O.temporal_lsh(segs1, X, R)[1] == 0.0)                       # T = 1: term not applicable
    assert np.all(np.abs(g * 64 - np.round(g * 64)) == 0)                      # multiples of 1 / K


def test_lsh_collision_law_theta_over_pi():
    """Sign random projections collide with probability 1 - theta / pi (Goemans-Williamson / Charikar): E[gamma] = theta / pi."""
    rng = np.random.default_rng(9)
    d, P = 24, 3000
    R = rng.standard_normal((64, d)).astype(np.float32)
    for theta in (0.3, 1.0, 2.2):
        a = rng.standard_normal((P, d)); a /= np.linalg.norm(a, axis=1, keepdims=True)
        b = rng.standard_normal((P, d)); b -= (b * a).sum(1, keepdims=True) * a; b /= np.linalg.norm(b, axis=1, keepdims=True)
        X = np.concatenate([a, np.cos(theta) * a + np.sin(theta) * b]).astype(np.float32)
        segs = seg1(2, P)
        g = O.temporal_lsh(segs, X, R)[1][P:]
        # the 64 hashes are shared by all pairs, so average over pairs AND hashes: tolerance from the spread over hashes
        assert abs(g.mean() - theta / np.pi) < 0.03, (theta, g.mean())


# ---------------------------------------------------------------- NEXT-4: draft-confidence entropy (Eq. 9-10)
def test_entropy_closed_forms():
    V = 1000
    uni = np.full((1, V), 3.25, np.float32)
    onehot = np.full((1, V), -1e4, np.float32); onehot[0, 17] = 0.0
    k, a, b = 10, 2.0, -1.0                                    # k logits at a, V - k at b: closed form below
    two = np.full((1, V), b, np.float32); two[0, :k] = a
    L = np.concatenate([uni, onehot, two])
    H, flag = O.draft_entropy(L, theta_conf=1.0)
    assert abs(H[0] - np.log(V)) < 1e-12                       # uniform: log V
    assert abs(H[1]) < 1e-12                                   # one-hot: 0
    Z = k * np.exp(a) + (V - k) * np.exp(b)
    pa, pb = np.exp(a) / Z, np.exp(b) / Z
    assert abs(H[2] - (-(k * pa * np.log(pa) + (V - k) * pb * np.log(pb)))) < 1e-12
    assert list(flag) == [0, 1, int(H[2] <= 1.0)]              # Eq. 10: speculate iff H <= theta


def test_entropy_of_masked_logits():
    """-inf logits (filtered drafts) carry no probability: 0 ln 0 = 0 (SPEC NEXT-4).  k survivors at equal logits -> ln k; one -> 0."""
    L = np.full((3, 300), -np.inf, np.float32)
    L[0, 10:14] = 1.5
    L[1, 299] = -3.0
    L[2, ::3] = 0.25
    H, flag = O.draft_entropy(L, 1.0)
    assert abs(H[0] - math.log(4)) < 1e-15 and H[1] == 0.0 and abs(H[2] - math.log(100)) < 1e-13
    assert list(flag) == [0, 1, 0]
    Hb, _ = O.draft_entropy(synth.f32_to_bf16_bits(L), 1.0)
    assert np.allclose(Hb, H, rtol=0, atol=1e-14)


def test_entropy_matches_scipy_and_is_shift_invariant():
    from scipy.special import softmax
    from scipy.stats import entropy
    rng = np.random.default_rng(3)
    L = (rng.standard_normal((6, 4097)) * np.array([[0.1], [1], [3], [6], [10], [0.5]])).astype(np.float32)
    H, _ = O.draft_entropy(L, 2.0)
    want = np.array([entropy(softmax(row.astype(np.float64))) for row in L])
    assert np.allclose(H, want, rtol=1e-12, atol=1e-12)
    H2, _ = O.draft_entropy((L + 8.0).astype(np.float32), 2.0)       # + 8 is exact for these magnitudes? compare loosely
    assert np.allclose(H, H2, rtol=1e-5)
    Lb = synth.f32_to_bf16_bits(L)
    Hb, _ = O.draft_entropy(Lb, 2.0)
    wantb = np.array([entropy(softmax(row.astype(np.float64))) for row in synth.bf16_bits_to_f32(Lb)])
    assert np.allclose(Hb, wantb, rtol=1e-12, atol=1e-12)            # bf16 decoding


# ---------------------------------------------------------------- NEXT-3: adaptive retention from Eq. 11's constraint
def test_adaptive_retention_rule():
    """keep_k = ceil((1 - MAS_s) N_s) clamped to [1, N_s] (beta_m >= 1 - MAS_m), ties and order as in top-k."""
    n = 10
    X = np.arange(n * 4, dtype=np.float32).reshape(n, 4)
    mas_tok = np.array([0.5, 0.1, 0.9, 0.1, 0.3, 0.7, 0.2, 0.8, 0.4, 0.6])
    prm = O.default_params(select_mode=2)
    for seg_mas, want_k in ((0.3, 7), (1.0, 1), (0.0, 10), (0.25, 8), (0.95, 1), (0.9, 1), (0.89, 2)):
        mask, idx, off, Y, out = O.select_compact(seg1(1, n), prm, X, mas_tok, seg_mas=[seg_mas])
        assert int(off[1]) == want_k == int(mask.sum()) == out[0].n_kept
        assert want_k >= (1.0 - seg_mas) * n - 1e-9 and want_k - 1 < max((1.0 - seg_mas) * n, 1)      # smallest admissible retention
        order = sorted(range(n), key=lambda i: (mas_tok[i], i))[:want_k]                               # same order as top-k
        assert list(idx[:want_k]) == sorted(order)
        assert np.array_equal(Y[:want_k], X[sorted(order)])


# ---------------------------------------------------------------- NEXT-2: learned heads (Eq. 3, Eq. 6 with supplied weights)
def _heads_weights(d, hidden, w_sp, W1z, W1p, b1, w2):
    W = np.zeros((64, d), np.float32)
    Wp = np.zeros((64, d), np.float32)
    B1 = np.zeros(64)
    W2 = np.zeros(64)
    W[0] = w_sp
    W[1:1 + hidden] = W1z
    Wp[1:1 + hidden] = W1p
    B1[1:1 + hidden] = b1
    W2[1:1 + hidden] = w2
    W[1 + hidden:] = 7.0          # rows past `hidden` are ignored
    Wp[0] = -3.0                  # so is row 0 of Wp
    B1[0] = 5.0
    W2[0] = 5.0
    return W, Wp, B1, W2


def test_learned_heads_worked_example():
    segs, n = O.make_segments([(0, 1, 1, 2, 1), (0, 2, 2, 1, 1)])
    X = f32([[1, 0], [0, 2], [2, 2], [-2, 0]])
    Q = f32([[1, 1], [3, -1]])
    W, Wp, b1, w2 = _heads_weights(2, 2, [1, -1], [[1, 0], [0, 1]], [[0.5, 0], [0, 1]], [-1.25, 0.25], [2, 3])
    m, out = O.learned_heads(segs, [0, 2], O.default_params(), X, Q, [0, 0, 1, 0.25], W, Wp, b1, w2, 0.0, -0.5, 2)
    assert np.allclose(m, [GOLD["heads_M_u1"], GOLD["heads_M_um2"], 0.5, GOLD["heads_M_um2"]], rtol=0, atol=1e-15)
    assert out[0].rho_spatial == 0.5 == out[1].rho_spatial
    assert out[0].alpha_mean == GOLD["heads_alpha_A"] and out[1].alpha_mean == GOLD["heads_alpha_B"]
    assert abs(out[0].beta - GOLD["heads_beta_A"]) < 1e-15 and abs(out[0].beta + out[1].beta - 1.0) < 1e-15
    assert out[0].gamma_avg == 0.0 and out[1].gamma_avg == 0.25
    assert abs(out[0].mas - GOLD["heads_mas_A"]) < 1e-14 and abs(out[1].mas - GOLD["heads_mas_B"]) < 1e-14


def test_learned_heads_special_cases_and_numpy():
    rng = np.random.default_rng(5)
    d, hidden = 24, 5
    rows = [(0, 1, 1, 30, 1), (0, 2, 3, 7, 1), (1, 1, 1, 11, 1)]
    segs, n = O.make_segments(rows)
    X = rng.standard_normal((n, d)).astype(np.float32)
    Q = rng.standard_normal((9, d)).astype(np.float32)
    q_off = [0, 4, 9]
    gamma = rng.random(n)
    w_sp = rng.standard_normal(d).astype(np.float32) * 0.3
    W1z, W1p = rng.standard_normal((hidden, d)).astype(np.float32), rng.standard_normal((hidden, d)).astype(np.float32)
    b1, w2 = rng.standard_normal(hidden), rng.standard_normal(hidden)
    W, Wp, B1, W2 = _heads_weights(d, hidden, w_sp, W1z, W1p, b1, w2)
    prm = O.default_params()
    m, out = O.learned_heads(segs, q_off, prm, X, Q, gamma, W, Wp, B1, W2, 0.1, -0.2, hidden)
    # library routines in float64: matrix products and column means
    X64, Q64 = X.astype(np.float64), Q.astype(np.float64)
    assert np.allclose(m, 1.0 / (1.0 + np.exp(-(X64 @ w_sp.astype(np.float64) + 0.1))), rtol=1e-13, atol=0)
    r0 = 0
    alphas = []
    for k, (req, _, T, P, _) in enumerate(rows):
        nk = T * P
        z = X64[r0:r0 + nk].mean(axis=0)
        p = Q64[q_off[req]:q_off[req + 1]].mean(axis=0)
        pre = W1z.astype(np.float64) @ z + W1p.astype(np.float64) @ p + b1
        alphas.append(float(w2 @ np.maximum(pre, 0.0) - 0.2))
        assert abs(out[k].alpha_mean - alphas[-1]) < 1e-12
        assert out[k].rho_spatial == np.count_nonzero(m[r0:r0 + nk] < 0.3) / nk
        r0 += nk
    e = np.exp(np.array(alphas[:2]) - max(alphas[:2]))
    assert abs(out[0].beta - e[0] / e.sum()) < 1e-14 and out[2].beta == 1.0          # request 1 has one segment
    assert abs(out[1].gamma_avg - gamma[30 + 7:30 + 21].reshape(2, 7).mean(axis=1).mean()) < 1e-15
    # token order inside a single-frame segment does not matter (means), the map is permuted with it
    perm = rng.permutation(30)
    X2 = X.copy()
    X2[:30] = X[:30][perm]
    m2, out2 = O.learned_heads(segs, q_off, prm, X2, Q, gamma, W, Wp, B1, W2, 0.1, -0.2, hidden)
    assert np.array_equal(m2[:30], m[:30][perm]) and abs(out2[0].alpha_mean - out[0].alpha_mean) < 1e-12
    # w_sp = 0: M = sigmoid(b_sp) everywhere, rho is 0 or 1 by the strict compare
    W0 = W.copy()
    W0[0] = 0
    for b, rho in ((math.log(0.3 / 0.7) - 1e-9, 1.0), (math.log(0.3 / 0.7) + 1e-9, 0.0)):
        m0, out0 = O.learned_heads(segs, q_off, prm, X, Q, gamma, W0, Wp, B1, W2, b, -0.2, hidden)
        assert np.allclose(m0, 1.0 / (1.0 + math.exp(-b)), rtol=1e-15) and all(o.rho_spatial == rho for o in out0)
    # a dead hidden layer (every unit clipped): alpha = b2 for every segment -> uniform beta
    Bd = B1.copy()
    Bd[1:1 + hidden] = -1e6
    _, outd = O.learned_heads(segs, q_off, prm, X, Q, gamma, W, Wp, Bd, W2, 0.1, -0.2, hidden)
    assert all(o.alpha_mean == -0.2 for o in outd) and outd[0].beta == 0.5 == outd[1].beta
    # Eq. 7 single image, beta = 1: MAS = lambda_sp * rho
    assert abs(out[2].mas - 0.6 * out[2].rho_spatial) < 1e-15


# ---------------------------------------------------------------- NEXT-3: pooling, merged token, residual coding
def test_spatial_pool_against_uniform_filter_and_hand_counts():
    from scipy.ndimage import uniform_filter
    rng = np.random.default_rng(3)
    rows = [(0, 1, 1, 24 * 24, 1), (0, 2, 3, 6 * 5, 1), (1, 3, 7, 1, 1)]      # image 24 x 24, video 3 frames of 6 x 5, audio P = 1
    segs, n = O.make_segments(rows)
    gw = [24, 5, 1]
    s = rng.random(n)
    assert np.array_equal(O.spatial_pool(segs, gw, 1, s), s)                  # k = 1 is the identity
    for k in (2, 3, 5):
        out = O.spatial_pool(segs, gw, k, s)
        r0 = 0
        for (_, _, T, P, _), W in zip(rows, gw):
            H = P // W
            for t in range(T):
                g = s[r0:r0 + P].reshape(H, W)
                # library routine: zero-padded window sums of the map and of ones; origin shifts the even window like the oracle's
                org = 0 if k % 2 else -1
                num = uniform_filter(g, size=k, mode="constant", origin=org) * k * k
                den = uniform_filter(np.ones_like(g), size=k, mode="constant", origin=org) * k * k
                assert np.allclose(out[r0:r0 + P].reshape(H, W), num / den, rtol=1e-12, atol=1e-14), (k, W)
                r0 += P
    # hand counts on a 3 x 3 grid holding 1..9, k = 3: centre = 5, corner (0,0) = (1+2+4+5)/4 = 3, edge (0,1) = (1+2+3+4+5+6)/6 = 3.5
    seg9, _ = O.make_segments([(0, 1, 1, 9, 1)])
    out = O.spatial_pool(seg9, [3], 3, np.arange(1.0, 10.0))
    assert out[4] == 5.0 and out[0] == 3.0 and out[1] == 3.5 and out[8] == 7.0
    assert np.all(O.spatial_pool(seg9, [3], 3, np.full(9, 0.25)) == 0.25)     # a constant map stays constant


def test_merge_dropped_means():
    rng = np.random.default_rng(8)
    rows = [(0, 1, 1, 7, 1), (0, 2, 3, 5, 1)]
    segs, n = O.make_segments(rows)
    X = rng.integers(-8, 9, (n, 6)).astype(np.float32)
    mask = (rng.random(n) < 0.4).astype(np.uint8)
    mask[7:12] = 1                                   # frame 0 of the video: nothing dropped
    mask[12:17] = 0                                  # frame 1: everything dropped
    Y, nd = O.merge_dropped(segs, X, mask)
    assert Y.shape == (4, 6) and list(nd) == [int((mask[:7] == 0).sum()), 0, 5, int((mask[17:22] == 0).sum())]
    assert np.all(Y[1] == 0.0)
    assert np.array_equal(Y[2], X[12:17].astype(np.float64).mean(axis=0))
    for f, (a, b) in enumerate([(0, 7), (7, 12), (12, 17), (17, 22)]):
        kept_sum = X[a:b][mask[a:b] == 1].astype(np.float64).sum(axis=0)
        assert np.allclose(nd[f] * Y[f] + kept_sum, X[a:b].astype(np.float64).sum(axis=0), rtol=0, atol=1e-12)
    # bf16 storage decodes exactly
    Yb, _ = O.merge_dropped(segs, synth.f32_to_bf16_bits(X), mask)
    assert np.array_equal(Yb, Y)


def test_gather_residual_rules():
    rng = np.random.default_rng(9)
    rows = [(0, 1, 1, 4, 1), (0, 2, 3, 5, 1)]        # image rows 0..3, video rows 4..18 (3 frames of 5 patches)
    segs, n = O.make_segments(rows)
    X = rng.integers(-20, 21, (n, 8)).astype(np.float32)
    X[14:19] = X[9:14]                               # frame 2 identical to frame 1
    idx = np.array([1, 3, 4, 8, 9, 12, 14, 18], np.int32)
    for store in (lambda a: a, synth.f32_to_bf16_bits):
        Xs = store(X)
        Y = O.gather_residual(segs, Xs, idx)
        Yf = Y if Y.dtype == np.float32 else (Y.astype(np.uint32) << 16).view(np.float32)
        assert np.array_equal(Yf[:4], X[[1, 3, 4, 8]])               # image rows and key-frame rows are copies
        assert np.array_equal(Yf[4], X[9] - X[4]) and np.array_equal(Yf[5], X[12] - X[7])
        assert np.all(Yf[6:] == 0.0)                                 # static frame: zero residual
        assert np.array_equal(Yf[4] + X[4], X[9])                    # residual + previous = original (small integers: exact)
    # bf16 rounding of an inexact difference: nearest even
    Xb = np.zeros((2, 8), np.float32)
    Xb[1, 0], Xb[0, 0] = 1.0, 2.0 ** -9                              # 1 - 2^-9 needs 9 bits: ties to even -> 1.0
    Xb[1, 1], Xb[0, 1] = 1.0, 3 * 2.0 ** -10                         # 1 - 3*2^-10: nearest bf16 is 1 - 2^-8... = 0.99609375
    seg2, _ = O.make_segments([(0, 2, 2, 1, 1)])
    Yb = O.gather_residual(seg2, synth.f32_to_bf16_bits(Xb), np.array([1], np.int32))
    got = (Yb.astype(np.uint32) << 16).view(np.float32)[0]
    assert got[0] == 1.0 and got[1] == 0.99609375


# ---------------------------------------------------------------- the oracle under AddressSanitizer / UBSan
def test_oracle_selftest_under_asan_ubsan(tmp_path):
    """oracle/selftest.cpp (a few closed-form pins + a ragged whole pass in both selection modes) built with
    -fsanitize=address,undefined: an out-of-bounds access, misaligned load or signed overflow in oracle/mas_oracle.cpp aborts it."""
    import shutil
    import subprocess
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    odir = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "oracle")
    exe = str(tmp_path / "oracle_selftest")
    subprocess.check_call(["g++", "-O1", "-g", "-std=c++17", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-Wall", "-Wextra",
                           "-o", exe, os.path.join(odir, "selftest.cpp")])
    out = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert out.returncode == 0 and "oracle selftest ok" in out.stdout, out.stdout + out.stderr
