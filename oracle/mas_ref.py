"""ctypes front-end of the CPU oracle (oracle/mas_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from the CUDA package.  Arrays are numpy; bf16 tensors travel as uint16 bit patterns.
Definitions followed: SPEC.md S0-S5 (MSAO §4.1, Eq. 3-7).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mas_oracle.cpp")
_LIB = os.path.join(_HERE, "libmas_oracle.so")

F32, BF16 = 0, 1


def build(force=False):
    """g++ -O2, no fast-math, no OpenMP: the oracle stays plain and single-threaded."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", _LIB, _SRC])
    return _LIB


class Segment(C.Structure):
    _fields_ = [("request", C.c_int32), ("modality", C.c_int32), ("row0", C.c_int64), ("n_frames", C.c_int32),
                ("n_patches", C.c_int32), ("keep_k", C.c_int32), ("reserved_", C.c_int32)]


class Params(C.Structure):
    _fields_ = [("lambda_spatial", C.c_double), ("lambda_temp", C.c_double), ("tau_s", C.c_double), ("kappa", C.c_double),
                ("spatial_gain", C.c_double), ("spatial_bias", C.c_double), ("rel_gain", C.c_double), ("rel_bias", C.c_double),
                ("cut", C.c_double), ("select_mode", C.c_int32), ("pad_", C.c_int32)]


class SegmentOut(C.Structure):
    _fields_ = [("rho_spatial", C.c_double), ("gamma_avg", C.c_double), ("alpha_mean", C.c_double), ("beta", C.c_double),
                ("mas", C.c_double), ("mean_s", C.c_double), ("std_s", C.c_double), ("mean_r", C.c_double), ("std_r", C.c_double),
                ("n_tokens", C.c_int64), ("n_kept", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.mas_ref_keep_count.restype = C.c_int32
        _lib.mas_ref_keep_count.argtypes = [C.c_int64, C.c_double]
    return _lib


def default_params(**kw):
    p = Params()
    lib().mas_ref_params_default(C.byref(p))
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def keep_count(n, ratio):
    return int(lib().mas_ref_keep_count(int(n), float(ratio)))


def make_segments(rows):
    """rows: iterable of (request, modality, n_frames, n_patches, keep_k); row0 is the running sum."""
    rows = list(rows)
    arr = (Segment * len(rows))()
    r0 = 0
    for i, (req, mod, T, P, k) in enumerate(rows):
        arr[i] = Segment(req, mod, r0, T, P, k, 0)
        r0 += T * P
    return arr, r0


def _dtype_code(a):
    if a.dtype == np.float32:
        return F32
    if a.dtype == np.uint16:
        return BF16
    raise TypeError("X/Q must be float32 or uint16 (bf16 bits), got %s" % a.dtype)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc):
    if rc != 0:
        raise RuntimeError("oracle returned %d" % rc)


def rms(segs, X):
    X = np.ascontiguousarray(X)
    s = np.zeros(X.shape[0], np.float64)
    _check(lib().mas_ref_rms(segs, len(segs), C.c_int64(X.shape[1]), _dtype_code(X), _p(X), _p(s)))
    return s


def temporal(segs, X):
    X = np.ascontiguousarray(X)
    g = np.zeros(X.shape[0], np.float64)
    _check(lib().mas_ref_temporal(segs, len(segs), C.c_int64(X.shape[1]), _dtype_code(X), _p(X), _p(g)))
    return g


def draft_entropy(logits, theta_conf):
    """NEXT-4: Eq. 9-10 per row of logits[n_rows, V] (float32 or bf16 bits): (H float64, speculate uint8)."""
    L = np.ascontiguousarray(logits)
    H = np.zeros(L.shape[0], np.float64)
    flag = np.zeros(L.shape[0], np.uint8)
    _check(lib().mas_ref_draft_entropy(_p(L), C.c_int64(L.shape[0]), C.c_int64(L.shape[1]), C.c_int64(L.shape[1]), _dtype_code(L),
                                       C.c_double(theta_conf), _p(H), _p(flag)))
    return H, flag


def learned_heads(segs, q_off, params, X, Q, gamma, W, Wp, b1, w2, b_sp, b2, hidden):
    """NEXT-2: Eq. 3 / Eq. 6 with supplied weights.  W, Wp: [64, d] in X's dtype; b1, w2: [64].  -> (m_spatial, seg_out)."""
    X = np.ascontiguousarray(X)
    Q = np.ascontiguousarray(Q)
    W = np.ascontiguousarray(W)
    Wp = np.ascontiguousarray(Wp)
    assert W.shape == (64, X.shape[1]) == Wp.shape and W.dtype == X.dtype == Wp.dtype == Q.dtype
    q_off = np.ascontiguousarray(q_off, np.int64)
    g = np.ascontiguousarray(gamma, np.float64)
    b1 = np.ascontiguousarray(b1, np.float64)
    w2 = np.ascontiguousarray(w2, np.float64)
    assert b1.shape == (64,) == w2.shape and g.shape == (X.shape[0],)
    m = np.zeros(X.shape[0], np.float64)
    out = (SegmentOut * len(segs))()
    _check(lib().mas_ref_learned_heads(segs, len(segs), _p(q_off), C.c_int64(X.shape[1]), _dtype_code(X), C.byref(params), _p(X), _p(Q),
                                       _p(g), _p(W), _p(Wp), _p(b1), _p(w2), C.c_double(b_sp), C.c_double(b2), C.c_int32(hidden),
                                       _p(m), out))
    return m, out


def spatial_pool(segs, grid_w, k, s):
    """NEXT-3a: k x k count-valid window mean of the per-token scalar map on each frame's H x W grid (W per segment)."""
    s = np.ascontiguousarray(s, np.float64)
    gw = np.ascontiguousarray(grid_w, np.int32)
    out = np.zeros_like(s)
    _check(lib().mas_ref_spatial_pool(segs, len(segs), _p(gw), C.c_int32(k), _p(s), _p(out)))
    return out


def merge_dropped(segs, X, keep_mask):
    """NEXT-3b: one mean token per frame from the dropped rows -> (Ymerge float64 [F, d], n_dropped int64 [F])."""
    X = np.ascontiguousarray(X)
    m = np.ascontiguousarray(keep_mask, np.uint8)
    F = int(sum(sg.n_frames for sg in segs))
    Y = np.zeros((F, X.shape[1]), np.float64)
    nd = np.zeros(F, np.int64)
    _check(lib().mas_ref_merge_dropped(segs, len(segs), C.c_int64(X.shape[1]), _dtype_code(X), _p(X), _p(m), _p(Y), _p(nd)))
    return Y, nd


def gather_residual(segs, X, kept_idx):
    """NEXT-3c: kept rows, frames t >= 1 of temporal segments as x_t - x_{t-1}; Y has X's dtype."""
    X = np.ascontiguousarray(X)
    idx = np.ascontiguousarray(kept_idx, np.int32)
    Y = np.zeros((len(idx), X.shape[1]), X.dtype)
    _check(lib().mas_ref_gather_residual(segs, len(segs), C.c_int64(X.shape[1]), _dtype_code(X), _p(X), _p(idx), C.c_int64(len(idx)), _p(Y)))
    return Y


def temporal_lsh(segs, X, R, want_proj=False):
    """NEXT-1: literal LSH probe of Eq. 5 with K = 64 hashes from R[64, d] (same dtype as X)."""
    X = np.ascontiguousarray(X)
    R = np.ascontiguousarray(R)
    assert R.shape == (64, X.shape[1]) and R.dtype == X.dtype
    sig = np.zeros(X.shape[0], np.uint64)
    g = np.zeros(X.shape[0], np.float64)
    proj = np.zeros((X.shape[0], 64), np.float64) if want_proj else None
    _check(lib().mas_ref_temporal_lsh(segs, len(segs), C.c_int64(X.shape[1]), _dtype_code(X), _p(X), _p(R), _p(sig), _p(proj), _p(g)))
    return (sig, g, proj) if want_proj else (sig, g)


def crossmodal(segs, q_off, X, Q, want_S=False):
    X = np.ascontiguousarray(X)
    Q = np.ascontiguousarray(Q)
    q_off = np.ascontiguousarray(q_off, np.int64)
    rel = np.zeros(X.shape[0], np.float64)
    S = None
    stride = 0
    if want_S:
        stride = int(np.max(np.diff(q_off)))
        S = np.full((X.shape[0], stride), np.nan, np.float64)
    _check(lib().mas_ref_crossmodal(segs, len(segs), _p(q_off), len(q_off) - 1, C.c_int64(X.shape[1]), _dtype_code(X),
                                    _p(X), _p(Q), _p(rel), _p(S), C.c_int64(stride)))
    return (rel, S) if want_S else rel


def fuse(segs, params, s, gamma, rel):
    s = np.ascontiguousarray(s, np.float64)
    gamma = np.ascontiguousarray(gamma, np.float64)
    rel = np.ascontiguousarray(rel, np.float64)
    n = s.shape[0]
    m = np.zeros(n, np.float64)
    mas = np.zeros(n, np.float64)
    out = (SegmentOut * len(segs))()
    _check(lib().mas_ref_fuse(segs, len(segs), C.byref(params), _p(s), _p(gamma), _p(rel), _p(m), _p(mas), out))
    return m, mas, out


def select_compact(segs, params, X, mas_tok, cap_rows=None, want_Y=True, seg_mas=None):
    """seg_mas: per-segment MAS_s, needed by the adaptive mode (select_mode = 2) only."""
    X = np.ascontiguousarray(X)
    mas_tok = np.ascontiguousarray(mas_tok, np.float64)
    n, d = X.shape
    if cap_rows is None:
        cap_rows = n
    mask = np.zeros(n, np.uint8)
    idx = np.full(max(cap_rows, 1), -1, np.int32)
    off = np.zeros(len(segs) + 1, np.int64)
    Y = np.zeros((max(cap_rows, 1), d), X.dtype) if want_Y else None
    out = (SegmentOut * len(segs))()
    if seg_mas is not None:
        for k, v in enumerate(seg_mas):
            out[k].mas = float(v)
    _check(lib().mas_ref_select_compact(segs, len(segs), C.c_int64(d), _dtype_code(X), C.byref(params), _p(X), _p(mas_tok),
                                        _p(mask), _p(idx), _p(off), _p(Y), C.c_int64(cap_rows), out))
    return mask, idx, off, Y, out


def forward(segs, q_off, params, X, Q, cap_rows=None, want_Y=True):
    """Whole pass.  Returns a dict of numpy arrays (float64 scores) + the per-segment records."""
    X = np.ascontiguousarray(X)
    Q = np.ascontiguousarray(Q)
    q_off = np.ascontiguousarray(q_off, np.int64)
    n, d = X.shape
    if cap_rows is None:
        cap_rows = n
    r = dict(s=np.zeros(n), m_spatial=np.zeros(n), gamma=np.zeros(n), rel=np.zeros(n), mas_tok=np.zeros(n),
             keep_mask=np.zeros(n, np.uint8), kept_idx=np.full(max(cap_rows, 1), -1, np.int32),
             kept_off=np.zeros(len(segs) + 1, np.int64), Y=np.zeros((max(cap_rows, 1), d), X.dtype) if want_Y else None)
    out = (SegmentOut * len(segs))()
    _check(lib().mas_ref_forward(segs, len(segs), _p(q_off), len(q_off) - 1, C.c_int64(d), _dtype_code(X), C.byref(params),
                                 _p(X), _p(Q), _p(r["s"]), _p(r["m_spatial"]), _p(r["gamma"]), _p(r["rel"]), _p(r["mas_tok"]), out,
                                 _p(r["keep_mask"]), _p(r["kept_idx"]), _p(r["kept_off"]), _p(r["Y"]), C.c_int64(cap_rows)))
    r["seg_out"] = out
    return r


def seg_out_array(out, field):
    return np.array([getattr(o, field) for o in out])
