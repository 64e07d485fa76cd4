"""Seeded synthetic workloads with the token shapes of the paper's inputs (image-text, video-text-audio; MSAO §5.2
V1-V7).  The paper's VQAv2 / MMBench data and Qwen encoders are not available; these stand in for them
(recipe: SURVEY.md §8(d), restated in DESIGN.md §"Input recipe").

This module only DRAWS inputs.  It contains none of the method's arithmetic and is the one module that serves both
the CUDA path and the oracle (tests feed the same host arrays to each).  numpy only; bf16 tensors are uint16 bit
patterns.  Every request is generated from its own Philox stream keyed by (seed, request), so requests can be
generated, sharded and sampled independently.
"""
from dataclasses import dataclass, field

import numpy as np

MOD_IMAGE, MOD_VIDEO, MOD_AUDIO = 1, 2, 3
SELECT_TOPK, SELECT_THRESHOLD, SELECT_ADAPTIVE = 0, 1, 2
GRID = 24  # 24 x 24 = 576 patch tokens per image / frame


def f32_to_bf16_bits(x):
    """Round-to-nearest-even fp32 -> bf16 bit pattern (uint16).  Inputs are finite."""
    u = np.ascontiguousarray(x, np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b):
    return (np.ascontiguousarray(b, np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def keep_count(n, ratio):
    """SPEC S5/G16 (host-side integer rule; the library exports the same rule as mas_keep_count)."""
    import math
    return int(min(n, max(1, math.ceil(ratio * n - 1e-9))))


@dataclass
class Workload:
    name: str
    d: int
    dtype: str                      # "bf16" | "f32"
    segments: list                  # (request, modality, n_frames, n_patches, keep_k)
    q_off: np.ndarray               # int64 [R+1]
    X: np.ndarray                   # [N, d] uint16 (bf16 bits) or float32
    Q: np.ndarray                   # [sum L, d]
    select_mode: int = SELECT_TOPK
    cut: float = 0.5
    salient: np.ndarray = None      # bool [N]: planted salient rows (sanity metric only)
    meta: dict = field(default_factory=dict)

    @property
    def n_tokens(self):
        return int(self.X.shape[0])

    @property
    def n_requests(self):
        return len(self.q_off) - 1

    def kept_capacity(self):
        if self.select_mode != SELECT_TOPK:
            return self.n_tokens
        return int(sum(s[4] for s in self.segments))


def _rng(seed, request):
    return np.random.Generator(np.random.Philox(np.random.SeedSequence([int(seed), int(request)])))


def _store(x, dtype):
    return f32_to_bf16_bits(x) if dtype == "bf16" else np.ascontiguousarray(x, np.float32)


def _unit(rng, d):
    v = rng.standard_normal(d, dtype=np.float32)
    return v / np.linalg.norm(v)


def _ordinary(rng, n, d):
    norms = np.exp(0.5 * rng.standard_normal(n, dtype=np.float32))          # LogNormal(0, 0.5)
    return norms[:, None] * rng.standard_normal((n, d), dtype=np.float32), norms


def _salient(rng, n, d, u_b, a=0.5):
    norms = np.exp(0.5 * rng.standard_normal(n, dtype=np.float32))
    g = rng.standard_normal((n, d), dtype=np.float32)
    return 4.0 * norms[:, None] * (np.float32(np.sqrt(1 - a * a)) * g + np.float32(a * np.sqrt(d)) * u_b[None, :])


def _aligned_query(rng, d, mean_vec):
    m = mean_vec / np.linalg.norm(mean_vec)
    w = rng.standard_normal(d, dtype=np.float32)
    w = w - np.dot(w, m) * m
    w = w / np.linalg.norm(w)
    return np.float32(np.sqrt(d)) * (np.float32(0.8) * m + np.float32(0.6) * w)


def _block_patches(r0, c0, h, w, limit=GRID * GRID):
    idx = [((r0 + i) % GRID) * GRID + ((c0 + j) % GRID) for i in range(h) for j in range(w)]
    return np.array([p for p in idx if p < limit], np.int64)


def _image_rows(rng, P, d, n_blocks, size_lo, size_hi):
    """One image segment: ordinary rows + planted salient blocks on the first 576 patches.  Returns fp32 rows,
    salient mask, list of block mean vectors."""
    x, _ = _ordinary(rng, P, d)
    sal = np.zeros(P, bool)
    means = []
    for _ in range(n_blocks):
        h = int(rng.integers(size_lo, size_hi + 1))
        w = int(rng.integers(size_lo, size_hi + 1))
        r0 = int(rng.integers(0, GRID - h + 1))
        c0 = int(rng.integers(0, GRID - w + 1))
        pp = _block_patches(r0, c0, h, w, limit=min(P, GRID * GRID))
        if len(pp) == 0:
            continue
        u_b = _unit(rng, d)
        x[pp] = _salient(rng, len(pp), d, u_b)
        sal[pp] = True
        means.append(x[pp].mean(axis=0))
    return x, sal, means


def _queries(rng, L, d, aligned_means):
    q = rng.standard_normal((L, d), dtype=np.float32)
    for j, m in enumerate(aligned_means[:L]):
        q[j] = _aligned_query(rng, d, m)
    return q


def _finish(name, d, dtype, segs, Ls, Xs, Qs, sal, **kw):
    q_off = np.zeros(len(Ls) + 1, np.int64)
    q_off[1:] = np.cumsum(Ls)
    return Workload(name=name, d=d, dtype=dtype, segments=segs, q_off=q_off, X=np.concatenate(Xs, axis=0),
                    Q=np.concatenate(Qs, axis=0), salient=np.concatenate(sal), **kw)


def single_image(seed=0, d=1024, dtype="f32", L=32, keep_ratio=0.25):
    """Config 1: one 24x24 image, one 6x6 salient block, two aligned queries."""
    rng = _rng(seed, 0)
    P = GRID * GRID
    x, sal, means = _image_rows(rng, P, d, 1, 6, 6)
    q = _queries(rng, L, d, [means[0], means[0]])
    return _finish("single_image", d, dtype, [(0, MOD_IMAGE, 1, P, keep_count(P, keep_ratio))], [L], [_store(x, dtype)],
                   [_store(q, dtype)], [sal])


def batched_images(seed=1, R=64, d=4096, dtype="bf16", L_lo=16, L_hi=64, keep_ratio=0.25, P=GRID * GRID):
    """Config 2: R single-image requests, 1-4 salient blocks of 3..8 x 3..8, 1-3 aligned queries."""
    segs, Ls, Xs, Qs, sals = [], [], [], [], []
    for r in range(R):
        rng = _rng(seed, r)
        nb = int(rng.integers(1, 5))
        x, sal, means = _image_rows(rng, P, d, nb, 3, 8)
        L = int(rng.integers(L_lo, L_hi + 1))
        na = int(rng.integers(1, 4))
        al = [means[int(rng.integers(0, len(means)))] for _ in range(na)] if means else []
        q = _queries(rng, L, d, al)
        segs.append((r, MOD_IMAGE, 1, P, keep_count(P, keep_ratio)))
        Ls.append(L); Xs.append(_store(x, dtype)); Qs.append(_store(q, dtype)); sals.append(sal)
    return _finish("batched_images", d, dtype, segs, Ls, Xs, Qs, sals)


def _video_rows(rng, T, P, d, dtype, static_frac, moving_block, n_static_blocks=0):
    """AR(1) patches x_t = 0.95 x_{t-1} + 0.31 n_p N(0,I) kept as an fp32 state and rounded on store.  Static patches
    freeze their state (stored rows are bit-identical frame to frame).  Salient rows override the stored row only,
    never the state (reading recorded in DESIGN.md)."""
    state, norms = _ordinary(rng, P, d)
    static = rng.random(P) < static_frac if static_frac > 0 else np.zeros(P, bool)
    u_b = _unit(rng, d)
    if moving_block:
        r0 = int(rng.integers(0, GRID - 8 + 1))
        c0 = int(rng.integers(0, GRID))
    fixed_pp = []
    for _ in range(n_static_blocks):
        h = int(rng.integers(3, 9)); w = int(rng.integers(3, 9))
        fixed_pp.append(_block_patches(int(rng.integers(0, GRID - h + 1)), int(rng.integers(0, GRID - w + 1)), h, w,
                                       limit=min(P, GRID * GRID)))
    out = np.empty((T * P, d), np.uint16 if dtype == "bf16" else np.float32)
    sal = np.zeros(T * P, bool)
    block_mean = None
    for t in range(T):
        if t > 0:
            dyn = ~static
            state[dyn] = np.float32(0.95) * state[dyn] + np.float32(0.31) * norms[dyn, None] * rng.standard_normal(
                (int(dyn.sum()), d), dtype=np.float32)
        frame = state
        pps = []
        if moving_block:
            pps.append(_block_patches(r0, c0 + t, 8, 8, limit=min(P, GRID * GRID)))
        pps += fixed_pp
        pps = [pp for pp in pps if len(pp)]
        if pps:
            frame = state.copy()
            for pp in pps:
                frame[pp] = _salient(rng, len(pp), d, u_b)
                sal[t * P + pp] = True
            if block_mean is None:
                block_mean = frame[pps[0]].mean(axis=0)
        out[t * P:(t + 1) * P] = _store(frame, dtype)
    return out, sal, block_mean, static


def video(seed=2, R=8, T=32, P=GRID * GRID, d=4096, dtype="bf16", L=48, keep_ratio=0.15, static_frac=0.6):
    """Config 3: R videos of T frames; 60 % static background patches (bit-copies), moving 8x8 salient block."""
    segs, Ls, Xs, Qs, sals, statics = [], [], [], [], [], []
    for r in range(R):
        rng = _rng(seed, r)
        x, sal, bm, static = _video_rows(rng, T, P, d, dtype, static_frac, moving_block=True)
        q = _queries(rng, L, d, [bm, bm] if bm is not None else [])
        segs.append((r, MOD_VIDEO, T, P, keep_count(T * P, keep_ratio)))
        Ls.append(L); Xs.append(x); Qs.append(_store(q, dtype)); sals.append(sal); statics.append(static)
    w = _finish("video", d, dtype, segs, Ls, Xs, Qs, sals)
    w.meta["static"] = statics
    return w


def audio_vision(seed=3, R=16, d=4096, dtype="bf16", L=64, P_img=GRID * GRID, T_aud=1500, img_ratio=0.25, aud_ratio=0.40):
    """Config 4: per request one image segment and one audio segment (AR(1) rho 0.9, 20 % near-silent frames)."""
    segs, Ls, Xs, Qs, sals = [], [], [], [], []
    for r in range(R):
        rng = _rng(seed, r)
        xi, sal_i, means = _image_rows(rng, P_img, d, 1, 3, 8)
        a = np.empty((T_aud, d), np.float32)
        a[0] = rng.standard_normal(d, dtype=np.float32)
        noise = rng.standard_normal((T_aud, d), dtype=np.float32)
        for t in range(1, T_aud):
            a[t] = np.float32(0.9) * a[t - 1] + np.float32(np.sqrt(0.19)) * noise[t]
        silent = rng.random(T_aud) < 0.2
        a[silent] *= np.float32(0.05)
        span = int(rng.integers(0, max(1, T_aud - 50)))
        am = a[span:span + 50].mean(axis=0)
        q = _queries(rng, L, d, [means[0], means[0], am, am] if means else [am, am])
        segs.append((r, MOD_IMAGE, 1, P_img, keep_count(P_img, img_ratio)))
        segs.append((r, MOD_AUDIO, T_aud, 1, keep_count(T_aud, aud_ratio)))
        Ls.append(L); Xs += [_store(xi, dtype), _store(a, dtype)]; Qs.append(_store(q, dtype))
        sals += [sal_i, np.zeros(T_aud, bool)]
    return _finish("audio_vision", d, dtype, segs, Ls, Xs, Qs, sals)


def ragged(seed=4, R=256, d=4096, dtype="bf16", n_lo=144, n_hi=2880, L_lo=8, L_hi=128, cut=0.5):
    """Config 5: ragged serving batch, image-type (T=1) or video-type (T=5) requests, threshold selection."""
    segs, Ls, Xs, Qs, sals = [], [], [], [], []
    for r in range(R):
        rng = _rng(seed, r)
        n = int(rng.integers(n_lo, n_hi + 1))
        L = int(rng.integers(L_lo, L_hi + 1))
        if rng.random() < 0.5:
            nb = int(rng.integers(1, 5))
            x, sal, means = _image_rows(rng, n, d, nb, 3, 8)
            x = _store(x, dtype)
            segs.append((r, MOD_IMAGE, 1, n, n))
            bm = means[0] if means else None
        else:
            P = max(1, n // 5)
            x, sal, bm, _ = _video_rows(rng, 5, P, d, dtype, 0.0, moving_block=False, n_static_blocks=int(rng.integers(1, 5)))
            segs.append((r, MOD_VIDEO, 5, P, 5 * P))
        q = _queries(rng, L, d, [bm] * int(rng.integers(1, 4)) if bm is not None else [])
        Ls.append(L); Xs.append(x); Qs.append(_store(q, dtype)); sals.append(sal)
    return _finish("ragged", d, dtype, segs, Ls, Xs, Qs, sals, select_mode=SELECT_THRESHOLD, cut=cut)


# The five BASELINE.json configs, full size, in order.
CONFIGS = {
    "single_image": single_image,
    "batched_images": batched_images,
    "video": video,
    "audio_vision": audio_vision,
    "ragged": ragged,
}


def draft_logits(seed=7, n_rows=256, V=151936, dtype="bf16"):
    """NEXT-4 input: draft-model logits for `n_rows` decode steps over a Qwen-sized vocabulary (PAPER.md:141-149 reads
    them from Qwen2-VL-2B, which is not available): Gaussian logits whose per-row scale is log-uniform in [0.3, 8]
    (flat to peaked distributions) plus a handful of boosted tokens.  Returns [n_rows, V] float32 or bf16 bits."""
    rng = _rng(seed, 0)
    scale = np.exp(rng.uniform(np.log(0.3), np.log(8.0), n_rows)).astype(np.float32)
    L = rng.standard_normal((n_rows, V), dtype=np.float32) * scale[:, None]
    for r in range(n_rows):
        hot = rng.integers(0, V, size=int(rng.integers(1, 6)))
        L[r, hot] += rng.uniform(2.0, 12.0, size=hot.size).astype(np.float32)
    return _store(L, dtype)


def make(name, **kw):
    return CONFIGS[name](**kw)


def shard_requests(costs, world_size):
    """Contiguous request ranges balanced by cost: returns world_size (lo, hi) pairs."""
    costs = np.asarray(costs, np.float64)
    total = costs.sum()
    csum = np.concatenate([[0.0], np.cumsum(costs)])
    bounds = [0]
    for k in range(1, world_size):
        target = total * k / world_size
        j = int(np.searchsorted(csum, target, side="left"))
        j = min(max(j, bounds[-1]), len(costs))
        if j > 0 and j <= len(costs) and abs(csum[j - 1] - target) < abs(csum[min(j, len(costs))] - target):
            j = max(j - 1, bounds[-1])
        bounds.append(j)
    bounds.append(len(costs))
    return [(bounds[k], bounds[k + 1]) for k in range(world_size)]
