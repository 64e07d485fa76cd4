"""Shared helpers of the GPU parity tests: run the CUDA path through the C-ABI binding and the oracle on the same seeded
host arrays and compare under SPEC.md "Parity rules"."""
import numpy as np

RTOL, ATOL = 1e-3, 1e-6          # north_star: relative error 1e-3 (bf16 inputs, fp32 accumulation)
SEL_BAND = 1e-3                  # selection must agree wherever the oracle score is further than this from the cut


def assert_close(gpu, ref, name):
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    assert gpu.shape == ref.shape, (name, gpu.shape, ref.shape)
    err = np.abs(gpu - ref)
    tol = RTOL * np.abs(ref) + ATOL
    bad = np.nonzero(err > tol)[0]
    assert bad.size == 0, "%s: %d/%d outside tolerance; worst idx %d gpu=%r ref=%r" % (
        name, bad.size, ref.size, bad[np.argmax(err[bad] - tol[bad])], gpu[bad[0]], ref[bad[0]])


def adaptive_keep(seg_mas, n):
    """NEXT-3 rule restated: the smallest retention Eq. 11's constraint beta >= 1 - MAS_s admits."""
    return int(min(n, max(1, np.ceil((1.0 - float(seg_mas)) * n - 1e-9))))


def check_selection(rows, select_mode, cut, ref_mas, gpu_mask, gpu_idx, gpu_off, row_base=0, gpu_seg_mas=None, ref_so=None, ref_m=None):
    """rows: (request, modality, T, P, keep_k) of the compared segments; arrays cover exactly these segments
    (gpu_idx holds global ids: subtract row_base).  SPEC.md parity rules for selection.
    Adaptive mode (2): the keep count is an integer decided by a float, so it is checked (a) exactly against the rule
    applied to the GPU's own fp32 MAS_s and (b) against the oracle's count within what the MAS_s tolerance can move it;
    the selection itself is then the top-k comparison at the GPU's count."""
    gpu_mask = np.asarray(gpu_mask).astype(bool)
    r0 = 0
    for k, (_, _, T, P, kk) in enumerate(rows):
        n = T * P
        mas = np.asarray(ref_mas[r0:r0 + n], np.float64)
        if select_mode == 2:
            kk = int(gpu_off[k + 1] - gpu_off[k])
            assert kk == adaptive_keep(np.float32(gpu_seg_mas[k]), n), (k, kk, float(gpu_seg_mas[k]), n)
            near = np.count_nonzero(np.abs(np.asarray(ref_m[r0:r0 + n]) - 0.3) <= 1e-3 * 0.3) if ref_m is not None else 0
            tol = RTOL * abs(ref_so[k].mas) + ATOL + 0.6 * near / n
            assert abs(kk - ref_so[k].n_kept) <= 1 + int(np.ceil(tol * n)), (k, kk, ref_so[k].n_kept, tol * n)
        if select_mode in (0, 2):
            order = np.sort(mas)
            c = order[kk - 1] if kk >= n else 0.5 * (order[kk - 1] + order[kk])
            ref_keep = np.zeros(n, bool)
            ref_keep[np.lexsort((np.arange(n), mas))[:kk]] = True       # (MAS, index) order
            assert gpu_off[k + 1] - gpu_off[k] == kk, "segment %d: n_kept %d != keep_k %d" % (k, gpu_off[k + 1] - gpu_off[k], kk)
        else:
            c = cut
            ref_keep = mas <= cut
        decided = np.abs(mas - c) > SEL_BAND
        gm = gpu_mask[r0:r0 + n]
        diff = np.nonzero(decided & (gm != ref_keep))[0]
        assert diff.size == 0, "segment %d: %d decided tokens with a different mask bit (first %d, mas %r, cut %r)" % (
            k, diff.size, diff[0], mas[diff[0]], c)
        idx = np.asarray(gpu_idx[gpu_off[k]:gpu_off[k + 1]], np.int64) - row_base - r0
        assert np.all(np.diff(idx) > 0), "segment %d: kept_idx not strictly ascending" % k
        assert idx.size == 0 or (idx.min() >= 0 and idx.max() < n), "segment %d: kept_idx outside the segment" % k
        assert np.array_equal(np.nonzero(gm)[0], idx), "segment %d: mask and kept_idx disagree" % k
        assert np.array_equal(idx[decided[idx]], np.nonzero(ref_keep & decided)[0]), "segment %d: decided kept lists differ" % k
        r0 += n


def check_seg_out(rows, gpu_so, ref_so, ref_m, tau_s=0.3, lambda_spatial=0.6):
    """Per-segment records.  rho may differ by the tokens whose M_i sits within 1e-3*tau_s of tau_s (SPEC)."""
    r0 = 0
    for k, (_, _, T, P, _) in enumerate(rows):
        n = T * P
        g, r = gpu_so[k], ref_so[k]
        for f in ("gamma_avg", "alpha_mean", "beta", "mean_s", "std_s"):
            assert abs(float(g[f]) - getattr(r, f)) <= RTOL * abs(getattr(r, f)) + ATOL, (k, f, float(g[f]), getattr(r, f))
        near = np.count_nonzero(np.abs(np.asarray(ref_m[r0:r0 + n]) - tau_s) <= 1e-3 * tau_s)
        assert abs(float(g["rho_spatial"]) - r.rho_spatial) <= near / n + 1e-6, (k, "rho", float(g["rho_spatial"]), r.rho_spatial, near)
        slack = lambda_spatial * near / n
        assert abs(float(g["mas"]) - r.mas) <= RTOL * abs(r.mas) + ATOL + slack, (k, "mas", float(g["mas"]), r.mas)
        assert int(g["n_tokens"]) == n
        r0 += n


# ---------------------------------------------------------------- the oracle over every request of a workload, on all host cores
_POOL_JOB = None   # (workload, oracle params kwargs): inherited by the forked workers, never pickled


def request_slices(w):
    """[(segment indices, first row, end row)] per request."""
    seg_req = np.array([s[0] for s in w.segments])
    seg_rows = np.array([s[2] * s[3] for s in w.segments])
    seg_row0 = np.concatenate([[0], np.cumsum(seg_rows)])
    out = []
    for r in range(w.n_requests):
        ks = np.nonzero(seg_req == r)[0]
        out.append((ks, int(seg_row0[ks[0]]), int(seg_row0[ks[-1] + 1])))
    return out


def oracle_request(r):
    """The oracle's whole pass on request r alone (requests are independent: SURVEY.md 8(e))."""
    from oracle import mas_ref as O
    w, prm_kw = _POOL_JOB
    ks, lo, hi = request_slices(w)[r]
    rows = [(0,) + tuple(w.segments[k][1:]) for k in ks]
    segs, _ = O.make_segments(rows)
    prm = O.default_params(select_mode=w.select_mode, cut=w.cut, **prm_kw)
    ref = O.forward(segs, [0, int(w.q_off[r + 1] - w.q_off[r])], prm, w.X[lo:hi], w.Q[w.q_off[r]:w.q_off[r + 1]], want_Y=False)
    so = [(o.rho_spatial, o.gamma_avg, o.alpha_mean, o.beta, o.mas, o.mean_s, o.std_s, o.n_tokens, o.n_kept) for o in ref["seg_out"]]
    return r, {k: ref[k] for k in ("m_spatial", "gamma", "rel", "mas_tok")}, so


class SegOut:
    __slots__ = ("rho_spatial", "gamma_avg", "alpha_mean", "beta", "mas", "mean_s", "std_s", "n_tokens", "n_kept")

    def __init__(self, t):
        for k, v in zip(self.__slots__, t):
            setattr(self, k, v)


def oracle_all_requests(w, requests=None, procs=None, **prm_kw):
    """{request: (scores dict, [SegOut])} for the given requests (default: all), the single-threaded oracle run as one process per
    host core over disjoint requests (fork: the workers inherit the inputs and never touch CUDA)."""
    import multiprocessing as mp
    import os
    global _POOL_JOB
    reqs = list(range(w.n_requests)) if requests is None else list(requests)
    _POOL_JOB = (w, prm_kw)
    n = min(len(reqs), procs or os.cpu_count() or 1)
    out = {}
    # longest requests first: the tail of the pool is then short
    sl = request_slices(w)
    reqs.sort(key=lambda r: -(sl[r][2] - sl[r][1]) * int(w.q_off[r + 1] - w.q_off[r]))
    if n <= 1:
        results = map(oracle_request, reqs)
    else:
        pool = mp.get_context("fork").Pool(n)
        results = pool.imap_unordered(oracle_request, reqs, chunksize=1)
    for r, scores, so in results:
        out[r] = (scores, [SegOut(t) for t in so])
    if n > 1:
        pool.close(); pool.join()
    _POOL_JOB = None
    return out
