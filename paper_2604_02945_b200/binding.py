"""Thin ctypes binding over the C ABI of libmsas (include/msas.h).  Argument marshalling only: every step of the MAS
pass runs in the CUDA kernels behind the library.  PyTorch is used for device memory and streams, nothing else.

There is no CPU fallback: if libmsas.so has not been built (python -m paper_2604_02945_b200.build) this module raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmsas.so")

MAS_OK, MAS_ERR_INVALID_ARG, MAS_ERR_UNSUPPORTED, MAS_ERR_WORKSPACE, MAS_ERR_CUDA = 0, 1, 2, 3, 4
MAS_F32, MAS_BF16 = 0, 1
MAS_MOD_IMAGE, MAS_MOD_VIDEO, MAS_MOD_AUDIO = 1, 2, 3
MAS_SELECT_TOPK, MAS_SELECT_THRESHOLD, MAS_SELECT_ADAPTIVE = 0, 1, 2
MAS_MAX_QUERY_TOKENS = 128

EXPORTS = ["mas_version", "mas_last_cuda_error", "mas_status_string", "mas_params_default", "mas_keep_count",
           "mas_plan_workspace_bytes", "mas_plan_create", "mas_plan_destroy", "mas_plan_n_tokens", "mas_plan_n_queries",
           "mas_plan_kept_capacity", "mas_plan_forward_launches", "mas_plan_enable_profiling", "mas_plan_stage_times", "mas_spatial", "mas_temporal", "mas_crossmodal", "mas_fuse",
           "mas_select_compact", "mas_forward", "mas_forward_host", "mas_forward_host_async", "mas_score", "mas_score_schedule", "mas_plan_set_inline_query_norms", "mas_temporal_lsh", "mas_forward_lsh", "mas_draft_entropy_workspace_bytes", "mas_draft_entropy", "mas_draft_entropy_static", "mas_learned_heads", "mas_forward_heads", "mas_plan_n_frames", "mas_spatial_pool", "mas_merge_dropped",
           "mas_gather_residual"]


class mas_segment(C.Structure):
    _fields_ = [("request", C.c_int32), ("modality", C.c_int32), ("row0", C.c_int64), ("n_frames", C.c_int32),
                ("n_patches", C.c_int32), ("keep_k", C.c_int32), ("reserved_", C.c_int32)]


class mas_params(C.Structure):
    _fields_ = [("lambda_spatial", C.c_float), ("lambda_temp", C.c_float), ("tau_s", C.c_float), ("kappa", C.c_float),
                ("spatial_gain", C.c_float), ("spatial_bias", C.c_float), ("rel_gain", C.c_float), ("rel_bias", C.c_float),
                ("cut", C.c_float), ("select_mode", C.c_int32)]


class mas_segment_out(C.Structure):
    _fields_ = [("rho_spatial", C.c_float), ("gamma_avg", C.c_float), ("alpha_mean", C.c_float), ("beta", C.c_float),
                ("mas", C.c_float), ("mean_s", C.c_float), ("std_s", C.c_float), ("n_tokens", C.c_int32), ("n_kept", C.c_int32)]


SEG_OUT_DTYPE = np.dtype([("rho_spatial", "<f4"), ("gamma_avg", "<f4"), ("alpha_mean", "<f4"), ("beta", "<f4"), ("mas", "<f4"),
                          ("mean_s", "<f4"), ("std_s", "<f4"), ("n_tokens", "<i4"), ("n_kept", "<i4")])
assert SEG_OUT_DTYPE.itemsize == C.sizeof(mas_segment_out) == 36


class mas_outputs(C.Structure):
    _fields_ = [("m_spatial", C.c_void_p), ("gamma", C.c_void_p), ("rel", C.c_void_p), ("mas_tok", C.c_void_p),
                ("seg_out", C.c_void_p), ("keep_mask", C.c_void_p), ("kept_idx", C.c_void_p), ("kept_off", C.c_void_p),
                ("Y", C.c_void_p), ("cap_rows", C.c_int64)]


class mas_heads(C.Structure):
    _fields_ = [("W", C.c_void_p), ("Wp", C.c_void_p), ("b1", C.c_void_p), ("w2", C.c_void_p), ("b_spatial", C.c_float),
                ("b2", C.c_float), ("hidden", C.c_int32), ("reserved_", C.c_int32)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libmsas.so is not built (%s). Run: python -m paper_2604_02945_b200.build — there is no CPU fallback."
                          % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.mas_version.restype = C.c_int
    lib.mas_last_cuda_error.restype = C.c_int
    lib.mas_status_string.restype = C.c_char_p
    lib.mas_status_string.argtypes = [C.c_int]
    lib.mas_params_default.restype = None
    lib.mas_params_default.argtypes = [C.POINTER(mas_params)]
    lib.mas_keep_count.restype = i32
    lib.mas_keep_count.argtypes = [i64, C.c_double]
    lib.mas_plan_workspace_bytes.argtypes = [C.POINTER(mas_segment), i32, C.POINTER(i64), i32, i32, i32, C.POINTER(C.c_size_t)]
    lib.mas_plan_create.argtypes = [C.POINTER(vp), C.POINTER(mas_segment), i32, C.POINTER(i64), i32, i32, i32,
                                    C.POINTER(mas_params), vp, C.c_size_t, vp]
    lib.mas_plan_destroy.argtypes = [vp]
    for f in ("mas_plan_n_tokens", "mas_plan_n_queries", "mas_plan_kept_capacity"):
        getattr(lib, f).restype = i64
        getattr(lib, f).argtypes = [vp]
    lib.mas_plan_forward_launches.restype = i32
    lib.mas_plan_forward_launches.argtypes = [vp]
    lib.mas_plan_enable_profiling.argtypes = [vp, i32]
    lib.mas_plan_stage_times.argtypes = [vp, i32, C.POINTER(C.c_float)]
    lib.mas_spatial.argtypes = [vp, vp, vp, vp, vp]
    lib.mas_temporal.argtypes = [vp, vp, vp, vp]
    lib.mas_crossmodal.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.mas_temporal_lsh.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.mas_temporal_lsh.restype = C.c_int
    lib.mas_forward_lsh.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(mas_outputs), vp]
    lib.mas_forward_lsh.restype = C.c_int
    lib.mas_fuse.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.mas_select_compact.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, vp, vp]
    lib.mas_forward.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, vp]
    lib.mas_forward_host.argtypes = [vp, vp, vp, vp, vp, C.POINTER(mas_outputs), C.POINTER(mas_outputs), vp]
    lib.mas_forward_host_async.argtypes = [vp, vp, vp, vp, vp, C.POINTER(mas_outputs), C.POINTER(mas_outputs), vp]
    lib.mas_forward_host_async.restype = C.c_int
    lib.mas_score.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.mas_score.restype = C.c_int
    lib.mas_plan_set_inline_query_norms.restype = C.c_int
    lib.mas_plan_set_inline_query_norms.argtypes = [vp, i32]
    lib.mas_draft_entropy_workspace_bytes.argtypes = [i64, i64, C.POINTER(C.c_size_t)]
    lib.mas_draft_entropy_workspace_bytes.restype = C.c_int
    lib.mas_draft_entropy.argtypes = [vp, i64, i64, i64, i32, C.c_float, vp, vp, vp, C.c_size_t, vp]
    lib.mas_draft_entropy.restype = C.c_int
    lib.mas_draft_entropy_static.argtypes = [vp, i64, i64, i64, i32, C.c_float, vp, vp, vp]
    lib.mas_draft_entropy_static.restype = C.c_int
    lib.mas_learned_heads.argtypes = [vp, vp, vp, vp, C.POINTER(mas_heads), vp, vp, vp]
    lib.mas_learned_heads.restype = C.c_int
    lib.mas_forward_heads.argtypes = [vp, vp, vp, C.POINTER(mas_heads), vp, vp, C.POINTER(mas_outputs), vp]
    lib.mas_forward_heads.restype = C.c_int
    lib.mas_plan_n_frames.argtypes = [vp]
    lib.mas_plan_n_frames.restype = C.c_int64
    lib.mas_spatial_pool.argtypes = [vp, C.POINTER(C.c_int32), i32, vp, vp, vp]
    lib.mas_spatial_pool.restype = C.c_int
    lib.mas_merge_dropped.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.mas_merge_dropped.restype = C.c_int
    lib.mas_gather_residual.argtypes = [vp, vp, vp, vp, vp, i64, vp]
    lib.mas_gather_residual.restype = C.c_int
    lib.mas_score_schedule.restype = i32
    lib.mas_score_schedule.argtypes = [C.POINTER(mas_segment), i32, C.POINTER(i64), i32, i32, i32, i32, C.POINTER(i32), i32]
    for f in ("mas_plan_workspace_bytes", "mas_plan_create", "mas_plan_destroy", "mas_plan_enable_profiling", "mas_plan_stage_times", "mas_spatial", "mas_temporal", "mas_crossmodal",
              "mas_fuse", "mas_select_compact", "mas_forward", "mas_forward_host"):
        getattr(lib, f).restype = C.c_int
    return lib


lib = _load()


class MasError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = lib.mas_status_string(status).decode()
        if status == MAS_ERR_CUDA:
            msg += " [cudaError %d]" % lib.mas_last_cuda_error()
        super().__init__("%s: %s (status %d)" % (where, msg, status))


def _check(status, where):
    if status != MAS_OK:
        raise MasError(status, where)


def default_params(**kw):
    p = mas_params()
    lib.mas_params_default(C.byref(p))
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def keep_count(n, ratio):
    return int(lib.mas_keep_count(int(n), float(ratio)))


def make_segments(rows):
    """rows: iterable of (request, modality, n_frames, n_patches, keep_k) -> (ctypes array, N)."""
    rows = list(rows)
    arr = (mas_segment * max(len(rows), 1))()
    r0 = 0
    for i, (req, mod, T, P, k) in enumerate(rows):
        arr[i] = mas_segment(req, mod, r0, T, P, k, 0)
        r0 += T * P
    return arr, r0


def score_schedule(rows, q_off, d, dtype, sm_count=148):
    """Host-only: the tile schedule of the tcgen05 score kernel as an int32 array [n_tiles, 16]
    (cta, row0, n_rows, n_blocks, stride, mode, prev, halo, q_row0, L, seg, part0, k0, k1, n_wait, peer; see include/msas.h);
    empty if the shape takes the generic path."""
    segs, _ = make_segments(rows)
    q = np.ascontiguousarray(q_off, np.int64)
    qp = q.ctypes.data_as(C.POINTER(C.c_int64))
    n = lib.mas_score_schedule(segs, len(list(rows)), qp, len(q) - 1, d, dtype, sm_count, None, 0)
    if n < 0:
        raise MasError(-n, "mas_score_schedule")
    out = np.zeros((max(n, 1), 16), np.int32)
    lib.mas_score_schedule(segs, len(list(rows)), qp, len(q) - 1, d, dtype, sm_count, out.ctypes.data_as(C.POINTER(C.c_int32)), n)
    return out[:n]


def workspace_bytes(segs, n_segs, q_off, d, dtype):
    q = np.ascontiguousarray(q_off, np.int64)
    out = C.c_size_t(0)
    st = lib.mas_plan_workspace_bytes(segs, n_segs, q.ctypes.data_as(C.POINTER(C.c_int64)), len(q) - 1, d, dtype, C.byref(out))
    return st, out.value


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Plan:
    """Owns the device workspace (a torch uint8 tensor) and the opaque mas_plan."""

    def __init__(self, segments, q_off, d, dtype, params=None, device="cuda", stream=None):
        self.rows = list(segments)
        self.segs, self.N = make_segments(self.rows)
        self.n_segs = len(self.rows)
        self.q_off = np.ascontiguousarray(q_off, np.int64)
        self.d, self.dtype = int(d), int(dtype)
        self.params = params if params is not None else default_params()
        self.device = torch.device(device)
        st, nbytes = workspace_bytes(self.segs, self.n_segs, self.q_off, self.d, self.dtype)
        _check(st, "mas_plan_workspace_bytes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._h = C.c_void_p()
        _check(lib.mas_plan_create(C.byref(self._h), self.segs, self.n_segs, self.q_off.ctypes.data_as(C.POINTER(C.c_int64)),
                                   len(self.q_off) - 1, self.d, self.dtype, C.byref(self.params), C.c_void_p(base), nbytes,
                                   _stream_ptr(stream)), "mas_plan_create")
        self.kept_capacity = int(lib.mas_plan_kept_capacity(self._h))
        self.n_queries = int(lib.mas_plan_n_queries(self._h))
        self.forward_launches = int(lib.mas_plan_forward_launches(self._h))
        self.torch_dtype = torch.bfloat16 if self.dtype == MAS_BF16 else torch.float32

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib.mas_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_inline_query_norms(self, on):
        _check(lib.mas_plan_set_inline_query_norms(self._h, 1 if on else 0), "mas_plan_set_inline_query_norms")
        self.forward_launches = int(lib.mas_plan_forward_launches(self._h))

    def enable_profiling(self, max_calls):
        _check(lib.mas_plan_enable_profiling(self._h, int(max_calls)), "mas_plan_enable_profiling")

    def stage_times(self, call):
        ms = (C.c_float * 3)()
        _check(lib.mas_plan_stage_times(self._h, int(call), ms), "mas_plan_stage_times")
        return [float(v) for v in ms]

    # ---- allocation helpers (device memory only)
    def _f32(self, n=None):
        return torch.empty(self.N if n is None else n, dtype=torch.float32, device=self.device)

    def alloc_outputs(self, cap_rows=None, want_Y=True):
        cap = self.kept_capacity if cap_rows is None else int(cap_rows)
        return dict(m_spatial=self._f32(), gamma=self._f32(), rel=self._f32(), mas_tok=self._f32(),
                    seg_out=torch.zeros(self.n_segs * 36, dtype=torch.uint8, device=self.device),
                    keep_mask=torch.empty(self.N, dtype=torch.uint8, device=self.device),
                    kept_idx=torch.full((max(cap, 1),), -1, dtype=torch.int32, device=self.device),
                    kept_off=torch.zeros(self.n_segs + 1, dtype=torch.int64, device=self.device),
                    Y=torch.zeros((max(cap, 1), self.d), dtype=self.torch_dtype, device=self.device) if want_Y else None,
                    cap_rows=cap)

    # ---- staged entry points
    def spatial(self, X, stream=None):
        s, m = self._f32(), self._f32()
        _check(lib.mas_spatial(self._h, _ptr(X), _ptr(s), _ptr(m), _stream_ptr(stream)), "mas_spatial")
        return s, m

    def temporal(self, X, stream=None):
        g = self._f32()
        _check(lib.mas_temporal(self._h, _ptr(X), _ptr(g), _stream_ptr(stream)), "mas_temporal")
        return g

    def temporal_lsh(self, X, Rm, stream=None):
        """NEXT-1: signatures (int64 view of the uint64 bits) and gamma of the literal LSH probe; Rm = [64, d] like X."""
        sig = torch.zeros(self.N, dtype=torch.int64, device=self.device)
        g = self._f32()
        _check(lib.mas_temporal_lsh(self._h, _ptr(X), _ptr(Rm), _ptr(sig), _ptr(g), _stream_ptr(stream)), "mas_temporal_lsh")
        return sig, g

    def learned_heads(self, X, Q, gamma, W, Wp, b1, w2, b_spatial, b2, hidden, stream=None):
        """NEXT-2: Eq. 3 / Eq. 6 with supplied weights (W, Wp: [64, d] like X; b1, w2: fp32 [64]) -> (m_spatial, seg_out)."""
        hd = mas_heads(_ptr(W), _ptr(Wp), _ptr(b1), _ptr(w2), float(b_spatial), float(b2), int(hidden), 0)
        m = self._f32()
        so = torch.zeros(self.n_segs * 36, dtype=torch.uint8, device=self.device)
        _check(lib.mas_learned_heads(self._h, _ptr(X), _ptr(Q), _ptr(gamma), C.byref(hd), _ptr(m), _ptr(so), _stream_ptr(stream)),
               "mas_learned_heads")
        return m, so

    def forward_heads(self, X, Q, W, Wp, b1, w2, b_spatial, b2, hidden, out=None, stream=None):
        """mas_forward + the learned heads in one pass: returns (outputs, learned m_spatial, learned seg_out)."""
        o = out if out is not None else self.alloc_outputs()
        hd = mas_heads(_ptr(W), _ptr(Wp), _ptr(b1), _ptr(w2), float(b_spatial), float(b2), int(hidden), 0)
        m = self._f32()
        so = torch.zeros(self.n_segs * 36, dtype=torch.uint8, device=self.device)
        _check(lib.mas_forward_heads(self._h, _ptr(X), _ptr(Q), C.byref(hd), _ptr(m), _ptr(so), C.byref(self._bundle(o)), _stream_ptr(stream)),
               "mas_forward_heads")
        return o, m, so

    # ---- NEXT-3: pooling, merged token, residual coding
    def spatial_pool(self, s, grid_w, k, stream=None):
        gw = (C.c_int32 * self.n_segs)(*[int(v) for v in grid_w])
        out = self._f32()
        _check(lib.mas_spatial_pool(self._h, gw, int(k), _ptr(s), _ptr(out), _stream_ptr(stream)), "mas_spatial_pool")
        return out

    def merge_dropped(self, X, keep_mask, stream=None):
        F = int(lib.mas_plan_n_frames(self._h))
        Y = torch.zeros((F, self.d), dtype=torch.float32, device=self.device)
        nd = torch.zeros(F, dtype=torch.int32, device=self.device)
        _check(lib.mas_merge_dropped(self._h, _ptr(X), _ptr(keep_mask), _ptr(Y), _ptr(nd), _stream_ptr(stream)), "mas_merge_dropped")
        return Y, nd

    def gather_residual(self, X, kept_idx, kept_off, cap_rows=None, stream=None):
        cap = self.kept_capacity if cap_rows is None else int(cap_rows)
        Y = torch.zeros((max(cap, 1), self.d), dtype=X.dtype, device=self.device)
        _check(lib.mas_gather_residual(self._h, _ptr(X), _ptr(kept_idx), _ptr(kept_off), _ptr(Y), cap, _stream_ptr(stream)), "mas_gather_residual")
        return Y

    def score(self, X, Q, want_gamma=True, out=None, stream=None):
        """a0-a3 in one pass: (s, gamma or None, rel).  `out` = (s, gamma, rel) buffers to reuse."""
        s, g, r = out if out is not None else (self._f32(), self._f32() if want_gamma else None, self._f32())
        _check(lib.mas_score(self._h, _ptr(X), _ptr(Q), _ptr(s), _ptr(g) if want_gamma else None, _ptr(r), _stream_ptr(stream)), "mas_score")
        return s, (g if want_gamma else None), r

    def crossmodal(self, X, Q, want_S=False, stream=None):
        rel = self._f32()
        S = torch.full((self.N, MAS_MAX_QUERY_TOKENS), float("nan"), dtype=torch.float32, device=self.device) if want_S else None
        _check(lib.mas_crossmodal(self._h, _ptr(X), _ptr(Q), _ptr(rel), _ptr(S), _stream_ptr(stream)), "mas_crossmodal")
        return (rel, S) if want_S else rel

    def fuse(self, s, gamma, rel, stream=None):
        m, mas = self._f32(), self._f32()
        so = torch.zeros(self.n_segs * 36, dtype=torch.uint8, device=self.device)
        _check(lib.mas_fuse(self._h, _ptr(s), _ptr(gamma), _ptr(rel), _ptr(m), _ptr(mas), _ptr(so), _stream_ptr(stream)), "mas_fuse")
        return m, mas, so

    def select_compact(self, X, mas_tok, cap_rows=None, want_Y=True, stream=None, seg_out=None):
        """seg_out: the fuse step's segment records (adaptive mode reads their MAS_s); a fresh zeroed table otherwise."""
        o = self.alloc_outputs(cap_rows, want_Y)
        if seg_out is not None:
            o["seg_out"] = seg_out
        _check(lib.mas_select_compact(self._h, _ptr(X), _ptr(mas_tok), _ptr(o["keep_mask"]), _ptr(o["kept_idx"]), _ptr(o["kept_off"]),
                                      _ptr(o["Y"]), o["cap_rows"], _ptr(o["seg_out"]), _stream_ptr(stream)), "mas_select_compact")
        return o

    # ---- fused entry point
    def forward(self, X, Q, out=None, stream=None):
        o = out if out is not None else self.alloc_outputs()
        _check(lib.mas_forward(self._h, _ptr(X), _ptr(Q), _ptr(o.get("m_spatial")), _ptr(o.get("gamma")), _ptr(o.get("rel")),
                               _ptr(o.get("mas_tok")), _ptr(o.get("seg_out")), _ptr(o.get("keep_mask")), _ptr(o.get("kept_idx")),
                               _ptr(o.get("kept_off")), _ptr(o.get("Y")), o["cap_rows"], _stream_ptr(stream)), "mas_forward")
        return o

    def forward_lsh(self, X, Q, Rm, out=None, stream=None):
        """mas_forward + the literal LSH probe in one pass: returns (outputs, sig int64 view, gamma_lsh)."""
        o = out if out is not None else self.alloc_outputs()
        sig = torch.zeros(self.N, dtype=torch.int64, device=self.device)
        g = self._f32()
        _check(lib.mas_forward_lsh(self._h, _ptr(X), _ptr(Q), _ptr(Rm), _ptr(sig), _ptr(g), C.byref(self._bundle(o)), _stream_ptr(stream)),
               "mas_forward_lsh")
        return o, sig, g

    @staticmethod
    def _bundle(o):
        b = mas_outputs()
        for k in ("m_spatial", "gamma", "rel", "mas_tok", "seg_out", "keep_mask", "kept_idx", "kept_off", "Y"):
            t = o.get(k)
            setattr(b, k, None if t is None else t.data_ptr())
        b.cap_rows = int(o["cap_rows"])
        return b

    def forward_host(self, h_X, h_Q, d_X, d_Q, d_out, h_out, stream=None):
        """HOST tensors in (pinned recommended), HOST tensors out; blocks until the results are on the host."""
        _check(lib.mas_forward_host(self._h, _ptr(h_X), _ptr(h_Q), _ptr(d_X), _ptr(d_Q), C.byref(self._bundle(d_out)),
                                    C.byref(self._bundle(h_out)) if h_out is not None else None, _stream_ptr(stream)),
               "mas_forward_host")


    def forward_host_async(self, h_X, h_Q, d_X, d_Q, d_out, h_out, stream=None):
        """As forward_host, without the final synchronisation (results valid once the stream is synchronised)."""
        _check(lib.mas_forward_host_async(self._h, _ptr(h_X), _ptr(h_Q), _ptr(d_X), _ptr(d_Q), C.byref(self._bundle(d_out)),
                                          C.byref(self._bundle(h_out)) if h_out is not None else None, _stream_ptr(stream)),
               "mas_forward_host_async")


def draft_entropy(logits, theta_conf, workspace=None, H=None, speculate=None, stream=None):
    """NEXT-4: Eq. 9-10 per row of a device tensor logits[n_rows, V] (float32 or bfloat16): (H float32, speculate uint8)."""
    n, V = logits.shape
    dt = MAS_BF16 if logits.dtype == torch.bfloat16 else MAS_F32
    nb = C.c_size_t(0)
    _check(lib.mas_draft_entropy_workspace_bytes(n, V, C.byref(nb)), "mas_draft_entropy_workspace_bytes")
    ws = workspace if workspace is not None else torch.empty(nb.value, dtype=torch.uint8, device=logits.device)
    H = H if H is not None else torch.empty(n, dtype=torch.float32, device=logits.device)
    sp = speculate if speculate is not None else torch.empty(n, dtype=torch.uint8, device=logits.device)
    _check(lib.mas_draft_entropy(_ptr(logits), n, V, logits.stride(0), dt, float(theta_conf), _ptr(H), _ptr(sp), _ptr(ws), ws.numel(),
                                 _stream_ptr(stream)), "mas_draft_entropy")
    return H, sp


DRAFT_ENTROPY_STATIC_MAX_PARTIALS = 16384   # include/msas.h, MAS_DRAFT_ENTROPY_STATIC_MAX_PARTIALS


def draft_entropy_static(logits, theta_conf, H, speculate, stream=None):
    """As draft_entropy, through the entry point that allocates nothing: the caller passes the outputs (H float32 [n_rows],
    speculate uint8 [n_rows]; either may be None), the partial sums live in the library's static device array."""
    n, V = logits.shape
    dt = MAS_BF16 if logits.dtype == torch.bfloat16 else MAS_F32
    _check(lib.mas_draft_entropy_static(_ptr(logits), n, V, logits.stride(0), dt, float(theta_conf), _ptr(H), _ptr(speculate),
                                        _stream_ptr(stream)), "mas_draft_entropy_static")
    return H, speculate


def seg_out_numpy(t):
    """uint8 torch tensor holding mas_segment_out records -> numpy structured array (host)."""
    return np.frombuffer(t.detach().cpu().numpy().tobytes(), dtype=SEG_OUT_DTYPE)


def to_device(arr, device="cuda"):
    """numpy array (uint16 = bf16 bits, or float32) -> device tensor of the matching torch dtype."""
    t = torch.from_numpy(np.ascontiguousarray(arr))
    if arr.dtype == np.uint16:
        t = t.view(torch.bfloat16)
    return t.to(device)
