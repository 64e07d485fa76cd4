"""GPU parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances: SPEC.md "Parity rules" (north_star: 1e-3 relative for scores, bit-exact masks / indices
wherever the oracle score is more than 1e-3 from the cut, bit-exact compacted rows)."""
import numpy as np
import pytest
import torch

from oracle import mas_ref as O
from paper_2604_02945_b200 import synth
from tests import parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2604_02945_b200 import binding
    return binding


def _dt(B, w):
    return B.MAS_BF16 if w.dtype == "bf16" else B.MAS_F32


def _plan(B, w, **prm):
    return B.Plan(w.segments, w.q_off, w.d, _dt(B, w), B.default_params(select_mode=w.select_mode, cut=w.cut, **prm))


def _oracle_params(w, **prm):
    return O.default_params(select_mode=w.select_mode, cut=w.cut, **prm)


def small_workloads():
    """Shrunken versions of the five BASELINE.json configs: several 128-row tiles plus ragged tails."""
    return [
        synth.single_image(seed=0, d=1024, dtype="f32"),                                    # config 1 at full size
        synth.single_image(seed=5, d=200, dtype="f32", L=7),                                # fp32, d % 8 != 0
        synth.batched_images(seed=1, R=5, d=512, L_lo=3, L_hi=70, P=333),                   # ragged tile tails, mixed L
        synth.video(seed=2, R=2, T=4, P=576, d=256, L=48),
        synth.video(seed=6, R=2, T=7, P=50, d=264, L=17, static_frac=0.5),                  # P < tile rows, d % 64 != 0
        synth.audio_vision(seed=3, R=2, d=256, L=64, P_img=576, T_aud=300),
        synth.ragged(seed=4, R=9, d=128, n_lo=20, n_hi=700, L_lo=1, L_hi=128),
    ]


IDS = ["cfg1_image_f32", "image_f32_d200", "batched_images", "video", "video_smallP", "audio_vision", "ragged_threshold"]


@pytest.mark.parametrize("w", small_workloads(), ids=IDS)
def test_staged_scores(B, w):
    segs, n = O.make_segments(w.segments)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    s, m = plan.spatial(X)
    gam = plan.temporal(X)
    rel, S = plan.crossmodal(X, Q, want_S=True)
    torch.cuda.synchronize()
    ref_s = O.rms(segs, w.X)
    ref_g = O.temporal(segs, w.X)
    ref_rel, ref_S = O.crossmodal(segs, w.q_off, w.X, w.Q, want_S=True)
    P.assert_close(s.cpu().numpy(), ref_s, "s")
    P.assert_close(gam.cpu().numpy(), ref_g, "gamma")
    assert np.array_equal(gam.cpu().numpy() == 0.0, ref_g == 0.0)          # bit-identical rows give exactly 0.0f
    P.assert_close(rel.cpu().numpy(), ref_rel, "rel")
    rel_only = plan.crossmodal(X, Q, want_S=False)                         # no S: bf16 / d % 64 == 0 plans take the tcgen05 score kernel
    torch.cuda.synchronize()
    P.assert_close(rel_only.cpu().numpy(), ref_rel, "rel (without S)")
    # raw dot products: error relative to |x||q| (the scale of the accumulation), not to a possibly tiny S_ij
    Sg = S.cpu().numpy()
    r0 = 0
    xn = ref_s * np.sqrt(w.d)
    for (req, _, T, Pn, _) in w.segments:
        L = int(w.q_off[req + 1] - w.q_off[req])
        qseg = O.make_segments([(0, 1, 1, L, 1)])[0]
        qn = O.rms(qseg, w.Q[w.q_off[req]:w.q_off[req + 1]]) * np.sqrt(w.d)
        sl = slice(r0, r0 + T * Pn)
        err = np.abs(Sg[sl, :L] - ref_S[sl, :L])
        assert np.all(err <= 1e-4 * xn[sl, None] * qn[None, :] + 1e-6), "S"
        assert np.all(np.isnan(Sg[sl, L:]))                                  # columns >= L untouched
        r0 += T * Pn
    m_ref, _, _ = O.fuse(segs, _oracle_params(w), ref_s, ref_g, ref_rel)
    P.assert_close(m.cpu().numpy(), m_ref, "m_spatial")
    plan.close()


@pytest.mark.parametrize("w", small_workloads(), ids=IDS)
def test_score_one_pass(B, w):
    """mas_score = the score stage of mas_forward on its own: gamma and rel identical to the fused call's, s against the oracle."""
    segs, n = O.make_segments(w.segments)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    s, g, r = plan.score(X, Q)
    s2, g2, r2 = plan.score(X, Q, want_gamma=False)
    o = plan.forward(X, Q)
    torch.cuda.synchronize()
    assert g2 is None and torch.equal(s, s2) and torch.equal(r, r2)
    assert torch.equal(g, o["gamma"]) and torch.equal(r, o["rel"])
    P.assert_close(s.cpu().numpy(), O.rms(segs, w.X), "s")
    plan.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_staged_fuse_and_select_on_shared_scalars(B, mode):
    """mas_fuse / mas_select_compact in isolation: both sides get the same fp32 scalars, selection must be bit-exact."""
    rng = np.random.default_rng(40 + mode)
    rows = [(0, 1, 1, 576, 144), (0, 3, 1500, 1, 600), (1, 2, 5, 300, 225), (2, 1, 1, 1, 1), (3, 2, 33, 555, 2000), (3, 1, 1, 130, 130)]
    segs, n = O.make_segments(rows)
    s = (np.abs(rng.standard_normal(n)) + 0.3).astype(np.float32)
    gam = rng.random(n).astype(np.float32)
    rel = (0.05 * rng.standard_normal(n)).astype(np.float32)
    w_d = 64
    X = rng.standard_normal((n, w_d)).astype(np.float32)
    plan = B.Plan(rows, [0, 4, 8, 12, 16], w_d, B.MAS_F32, B.default_params(select_mode=mode, cut=0.45))
    prm = O.default_params(select_mode=mode, cut=0.45)
    m, mas, so = plan.fuse(torch.from_numpy(s).cuda(), torch.from_numpy(gam).cuda(), torch.from_numpy(rel).cuda())
    m_ref, mas_ref_, so_ref = O.fuse(segs, prm, s, gam, rel)
    P.assert_close(m.cpu().numpy(), m_ref, "m_spatial")
    P.assert_close(mas.cpu().numpy(), mas_ref_, "mas_tok")
    P.check_seg_out(rows, B.seg_out_numpy(so), so_ref, m_ref)
    # selection on scores with heavy ties, quantised so that both sides see identical fp32 values
    vals = (rng.integers(0, 64, n) / 64.0).astype(np.float32)
    o = plan.select_compact(torch.from_numpy(X).cuda(), torch.from_numpy(vals).cuda())
    mask_r, idx_r, off_r, Y_r, so_r = O.select_compact(segs, prm, X, vals)
    off = o["kept_off"].cpu().numpy()
    assert np.array_equal(off, off_r)
    assert np.array_equal(o["keep_mask"].cpu().numpy(), mask_r)
    tot = int(off[-1])
    assert np.array_equal(o["kept_idx"].cpu().numpy()[:tot], idx_r[:tot])
    assert np.array_equal(o["Y"].cpu().numpy()[:tot], Y_r[:tot])
    assert [int(v) for v in B.seg_out_numpy(o["seg_out"])["n_kept"]] == [x.n_kept for x in so_r]
    plan.close()


def _forward_and_compare(B, w, sample_requests=None, **prm):
    """Run mas_forward on the whole workload; compare the sampled requests (default: all) against the oracle."""
    plan = _plan(B, w, **prm)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    o = plan.forward(X, Q)
    torch.cuda.synchronize()
    host = {k: (v.cpu().numpy() if isinstance(v, torch.Tensor) and k not in ("Y", "seg_out") else v) for k, v in o.items()}
    so = B.seg_out_numpy(o["seg_out"])
    seg_req = np.array([s[0] for s in w.segments])
    seg_rows = np.array([s[2] * s[3] for s in w.segments])
    seg_row0 = np.concatenate([[0], np.cumsum(seg_rows)])
    reqs = range(w.n_requests) if sample_requests is None else sample_requests
    refs = P.oracle_all_requests(w, reqs, **prm)          # one oracle process per host core over disjoint requests
    for r in reqs:
        ks = np.nonzero(seg_req == r)[0]
        rows = [(0,) + tuple(w.segments[k][1:]) for k in ks]
        lo, hi = int(seg_row0[ks[0]]), int(seg_row0[ks[-1] + 1])
        ref, ref_so = refs[r]
        ref = dict(ref, seg_out=ref_so)
        for name in ("m_spatial", "gamma", "rel", "mas_tok"):
            P.assert_close(host[name][lo:hi], ref[name], "%s[req %d]" % (name, r))
        assert np.array_equal(host["gamma"][lo:hi] == 0.0, ref["gamma"] == 0.0)
        P.check_seg_out(rows, so[ks[0]:ks[-1] + 1], ref["seg_out"], ref["m_spatial"])
        off = host["kept_off"][ks[0]:ks[-1] + 2]
        P.check_selection(rows, w.select_mode, w.cut, ref["mas_tok"], host["keep_mask"][lo:hi], host["kept_idx"], off, row_base=lo,
                          gpu_seg_mas=so["mas"][ks[0]:ks[-1] + 1], ref_so=ref["seg_out"], ref_m=ref["m_spatial"])
    # whole-batch structural properties (hold at any size)
    total = int(host["kept_off"][-1])
    assert host["keep_mask"].sum() == total
    assert np.array_equal(np.nonzero(host["keep_mask"])[0], host["kept_idx"][:total])
    assert [int(v) for v in so["n_kept"]] == list(np.diff(host["kept_off"]))
    idx = o["kept_idx"][:total].long()
    assert torch.equal(o["Y"][:total].view(torch.uint8), X[idx].view(torch.uint8))       # bit-exact compacted rows
    g = host["gamma"]
    assert np.all((g >= 0) & (g <= 1 + 1e-6)) and np.all((host["mas_tok"] >= -1e-6) & (host["mas_tok"] <= 1 + 1e-6))
    plan.close()
    return host, so


@pytest.mark.parametrize("w", small_workloads(), ids=IDS)
def test_forward_small(B, w):
    _forward_and_compare(B, w)


def test_forward_nondefault_params(B):
    w = synth.video(seed=8, R=2, T=3, P=200, d=128, L=9)
    _forward_and_compare(B, w, lambda_spatial=0.3, lambda_temp=0.5, tau_s=0.45, kappa=3.0, spatial_gain=2.0, spatial_bias=-0.5,
                         rel_gain=0.5, rel_bias=0.25)


def test_edge_cases(B):
    rng = np.random.default_rng(77)
    d = 64
    # zero rows, identical rows, a one-token segment, L = 1 and L = 128, minimum d
    rows = [(0, 2, 3, 4, 5), (1, 1, 1, 1, 1), (2, 3, 6, 1, 2)]
    n = 12 + 1 + 6
    X = rng.standard_normal((n, d)).astype(np.float32)
    X[5] = X[1]            # frame 1 patch 1 identical to frame 0
    X[6] = 0               # zero row against non-zero previous -> gamma 1
    X[10] = 0              # zero row, previous (6) also zero -> gamma 0
    X[14] = X[13]
    Xb = synth.f32_to_bf16_bits(X)
    Q = synth.f32_to_bf16_bits(rng.standard_normal((1 + 128 + 2, d)).astype(np.float32))
    Q[129] = 0             # zero query
    w = synth.Workload("edge", d, "bf16", rows, np.array([0, 1, 129, 131]), Xb, Q, salient=np.zeros(n, bool))
    host, so = _forward_and_compare(B, w)
    assert host["gamma"][5] == 0.0 and host["gamma"][6] == 1.0 and host["gamma"][10] == 0.0 and host["gamma"][14] == 0.0
    assert host["rel"][6] == 0.0
    # minimum width d = 8 (bf16) and d = 4... the documented floor is 8
    w8 = synth.batched_images(seed=12, R=2, d=8, L_lo=2, L_hi=5, P=40)
    _forward_and_compare(B, w8)


def test_threshold_cap_overflow_and_empty_segments(B):
    w = synth.ragged(seed=14, R=4, d=64, n_lo=100, n_hi=300, L_lo=4, L_hi=9, cut=0.2)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    full = plan.forward(X, Q)
    total = int(full["kept_off"][-1].item())
    assert 0 < total < w.n_tokens
    cap = max(1, total // 2)
    o = plan.alloc_outputs(cap_rows=cap + 3)
    o["kept_idx"][cap:] = -7
    o["Y"][cap:] = 123.0
    o["cap_rows"] = cap
    plan.forward(X, Q, out=o)
    torch.cuda.synchronize()
    assert int(o["kept_off"][-1].item()) == total                                     # true total still reported
    assert torch.equal(o["kept_idx"][:cap], full["kept_idx"][:cap])
    assert torch.all(o["kept_idx"][cap:] == -7) and torch.all(o["Y"][cap:] == 123.0)   # nothing written past the cap
    plan.close()
    # a cut below every score keeps nothing anywhere
    w0 = synth.ragged(seed=14, R=3, d=64, n_lo=100, n_hi=300, L_lo=4, L_hi=9, cut=-1.0)
    plan = _plan(B, w0)
    o = plan.forward(B.to_device(w0.X), B.to_device(w0.Q))
    assert int(o["kept_off"][-1].item()) == 0 and int(o["keep_mask"].sum().item()) == 0
    plan.close()


def test_invariances_on_gpu(B):
    w = synth.video(seed=31, R=2, T=4, P=150, d=128, L=12)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    a = plan.forward(X, Q)
    b = plan.forward(X, Q)                                                            # bit-reproducible
    for k in ("m_spatial", "gamma", "rel", "mas_tok", "keep_mask", "kept_idx", "kept_off", "seg_out", "Y"):
        assert torch.equal(a[k].view(torch.uint8), b[k].view(torch.uint8)), k
    c = plan.forward(X * 4.0, Q * 0.25)                                               # power-of-two scaling
    for k in ("m_spatial", "gamma", "rel", "mas_tok"):
        P.assert_close(c[k].cpu().numpy(), a[k].cpu().numpy(), k)
    assert torch.equal(a["keep_mask"], c["keep_mask"])
    perm = torch.cat([torch.randperm(12), 12 + torch.randperm(12)]).cuda()            # query order is irrelevant
    e = plan.forward(X, Q[perm])
    P.assert_close(e["rel"].cpu().numpy(), a["rel"].cpu().numpy(), "rel under query permutation")
    plan.close()


def test_forward_host_matches_device_path(B):
    w = synth.batched_images(seed=33, R=3, d=256, L_lo=5, L_hi=20)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    dev = plan.forward(X, Q)
    hX = torch.from_numpy(w.X).view(torch.bfloat16).pin_memory()
    hQ = torch.from_numpy(w.Q).view(torch.bfloat16).pin_memory()
    dX, dQ = torch.empty_like(X), torch.empty_like(Q)
    d_out = plan.alloc_outputs()
    h_out = {k: (torch.zeros_like(v, device="cpu").pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in d_out.items()}
    plan.forward_host(hX, hQ, dX, dQ, d_out, h_out)
    for k in ("m_spatial", "gamma", "rel", "mas_tok", "keep_mask", "kept_idx", "kept_off", "seg_out", "Y"):
        assert torch.equal(h_out[k].view(torch.uint8), dev[k].cpu().view(torch.uint8)), k
    plan.close()


@pytest.mark.parametrize("mode", [0, 1], ids=["topk", "threshold"])
def test_forward_host_async_two_plans_two_streams(B, mode):
    """The pipelined end-to-end pattern of bench.py: two plans on two streams called alternately, results valid after the
    streams are synchronised, identical to the blocking call."""
    ws = [synth.video(seed=91 + i, R=2, T=3, P=200, d=256, L=12) for i in range(2)]
    for w in ws:
        w.select_mode, w.cut = mode, 0.45
    plans = [_plan(B, w) for w in ws]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    hXs = [torch.from_numpy(w.X).view(torch.bfloat16).pin_memory() for w in ws]
    hQs = [torch.from_numpy(w.Q).view(torch.bfloat16).pin_memory() for w in ws]
    dXs = [torch.empty(w.X.shape, dtype=torch.bfloat16, device="cuda") for w in ws]
    dQs = [torch.empty(w.Q.shape, dtype=torch.bfloat16, device="cuda") for w in ws]
    d_outs = [p.alloc_outputs() for p in plans]
    h_outs = [{k: (torch.zeros_like(v, device="cpu").pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in d.items()} for d in d_outs]
    torch.cuda.synchronize()
    for rep in range(3):
        for i in range(2):
            plans[i].forward_host_async(hXs[i], hQs[i], dXs[i], dQs[i], d_outs[i], h_outs[i], stream=streams[i])
    for st in streams:
        st.synchronize()
    for i in range(2):
        ref = plans[i].forward(B.to_device(ws[i].X), B.to_device(ws[i].Q))
        torch.cuda.synchronize()
        tot = int(ref["kept_off"][-1].item())
        for k in ("mas_tok", "keep_mask", "kept_off", "seg_out"):
            assert torch.equal(h_outs[i][k].view(torch.uint8), ref[k].cpu().view(torch.uint8)), k
        assert torch.equal(h_outs[i]["kept_idx"][:tot], ref["kept_idx"][:tot].cpu())
        assert torch.equal(h_outs[i]["Y"][:tot].view(torch.uint8), ref["Y"][:tot].cpu().view(torch.uint8))
    for p in plans:
        p.close()


def test_unsupported_inputs_fail_loudly(B):
    w = synth.batched_images(seed=34, R=1, d=64, L_lo=4, L_hi=4, P=32)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    Xmis = torch.empty(w.n_tokens * 64 + 8, dtype=torch.bfloat16, device="cuda")[1:1 + w.n_tokens * 64].view(w.n_tokens, 64)
    with pytest.raises(B.MasError) as ei:
        plan.forward(Xmis, Q)
    assert ei.value.status == B.MAS_ERR_UNSUPPORTED
    o = plan.alloc_outputs()
    o["kept_idx"] = None
    with pytest.raises(B.MasError):
        plan.forward(X, Q, out=o)                                                     # Y without kept_idx
    plan.close()


# ---------------------------------------------------------------- full BASELINE.json sizes, bench launch configuration
import os

FULL = [("batched_images", {}, [0, 31, 63]), ("video", {}, [5]), ("audio_vision", {}, [7]), ("ragged", {}, [3, 100, 255])]


@pytest.mark.parametrize("name,kw,sample", FULL, ids=[f[0] for f in FULL])
def test_forward_full_size(B, name, kw, sample):
    """BASELINE.json configs 2-5 at full size, in the launch configuration bench.py times: EVERY request against the oracle (the
    oracle sharded over the host cores, one request per process at a time).  MSAS_PARITY_QUICK=1 compares the sampled requests only."""
    w = synth.make(name, **kw)
    _forward_and_compare(B, w, sample_requests=sample if os.environ.get("MSAS_PARITY_QUICK") else None)


@pytest.mark.parametrize("name", ["batched_images", "video", "ragged"])
def test_forward_full_size_is_bit_reproducible(B, name):
    """Two runs of the full-size pass on the same inputs give the same bits in every output: the K-split parts of a row block are
    added in exchange-slot order and every reduction of the segment kernel is fixed-order (no floating-point atomics anywhere)."""
    w = synth.make(name)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    a = plan.forward(X, Q)
    b = plan.forward(X, Q)
    torch.cuda.synchronize()
    for k in ("m_spatial", "gamma", "rel", "mas_tok", "keep_mask", "kept_off"):
        assert torch.equal(a[k], b[k]), k
    total = min(int(a["kept_off"][-1].item()), int(a["cap_rows"]))          # rows past the kept count are never written
    assert torch.equal(a["kept_idx"][:total], b["kept_idx"][:total]) and torch.equal(a["Y"][:total], b["Y"][:total])
    plan.close()


# ---------------------------------------------------------------- segment sizes around every internal boundary
def _random_workload(seed, seg_shapes, d, L_list, select_mode=0, cut=0.5, keep_ratio=0.3):
    """seg_shapes: list of (request, modality, T, P); plain random rows (no planted structure needed here)."""
    rng = np.random.default_rng(seed)
    rows, n = [], 0
    for (req, mod, T, P) in seg_shapes:
        rows.append((req, mod, T, P, synth.keep_count(T * P, keep_ratio)))
        n += T * P
    X = rng.standard_normal((n, d)).astype(np.float32) * np.exp(0.5 * rng.standard_normal((n, 1))).astype(np.float32)
    r0 = 0
    for (req, mod, T, P) in seg_shapes:            # make temporal segments correlated, with some bit-identical rows
        for t in range(1, T):
            cur, prev = slice(r0 + t * P, r0 + (t + 1) * P), slice(r0 + (t - 1) * P, r0 + t * P)
            X[cur] = 0.9 * X[prev] + 0.4 * X[cur]
            same = np.nonzero(rng.random(P) < 0.3)[0]
            X[r0 + t * P + same] = X[r0 + (t - 1) * P + same]      # copied in fp32: still bit-identical after rounding
        r0 += T * P
    q_off = np.concatenate([[0], np.cumsum(L_list)]).astype(np.int64)
    Q = rng.standard_normal((int(q_off[-1]), d)).astype(np.float32)
    Xb = synth.f32_to_bf16_bits(X)
    return synth.Workload("sweep", d, "bf16", rows, q_off, Xb, synth.f32_to_bf16_bits(Q), select_mode=select_mode, cut=cut,
                          salient=np.zeros(n, bool))


SWEEPS = {
    # double-tile boundaries of the score kernel (128 / 256 rows) and single-box heights, images and short videos
    "tile_heights": ([(0, 1, 1, 1), (0, 1, 1, 15), (1, 1, 1, 129), (1, 2, 3, 90), (2, 1, 1, 200), (3, 1, 1, 256), (4, 1, 1, 257), (5, 1, 1, 600),
                      (6, 2, 2, 130), (7, 3, 40, 1)], 128, [5, 33, 64, 1, 128, 17, 48, 9]),
    # segment kernel: 2 CTAs per segment, 512 threads
    "cluster2": ([(0, 1, 1, 2100), (0, 2, 3, 400), (1, 1, 1, 7)], 64, [12, 3]),
    # 4 CTAs per segment
    "cluster4": ([(0, 2, 5, 1000), (1, 1, 1, 300)], 64, [20, 6]),
    # 8 CTAs per segment
    "cluster8": ([(0, 1, 1, 9000), (1, 2, 2, 33)], 64, [7, 2]),
}


@pytest.mark.parametrize("name", list(SWEEPS), ids=list(SWEEPS))
@pytest.mark.parametrize("mode", [0, 1], ids=["topk", "threshold"])
def test_forward_segment_size_sweep(B, name, mode):
    shapes, d, L = SWEEPS[name]
    w = _random_workload(101 + mode, shapes, d, L, select_mode=mode, cut=0.45)
    _forward_and_compare(B, w)


# ---------------------------------------------------------------- NEXT-3: adaptive retention (beta >= 1 - MAS_s)
@pytest.mark.parametrize("name", ["images", "video", "audio_vision", "cluster8", "tile_heights"])
def test_forward_adaptive_retention(B, name):
    if name in SWEEPS:
        shapes, d, L = SWEEPS[name]
        w = _random_workload(300, shapes, d, L, select_mode=2, cut=0.45)
    else:
        w = {"images": synth.batched_images(seed=41, R=5, d=512, L_lo=3, L_hi=70, P=333),
             "video": synth.video(seed=42, R=2, T=4, P=576, d=256, L=48),
             "audio_vision": synth.audio_vision(seed=43, R=2, d=256, L=64, P_img=576, T_aud=300)}[name]
        w.select_mode = 2
    plan = _plan(B, w)
    assert plan.kept_capacity == w.n_tokens
    host, so = _forward_and_compare(B, w)
    nk = np.array([int(v) for v in so["n_kept"]])
    nt = np.array([s[2] * s[3] for s in w.segments])
    assert np.all(nk >= 1) and np.all(nk <= nt)
    assert np.all(nk >= (1.0 - so["mas"].astype(np.float64)) * nt - 1e-6)         # the constraint itself
    plan.close()


def test_staged_adaptive_select_on_shared_scalars(B):
    """mas_select_compact in adaptive mode reads MAS_s from the fuse step's records: bit-exact against the oracle given the
    same fp32 MAS_s and token scores; NULL records are refused."""
    rng = np.random.default_rng(47)
    rows = [(0, 1, 1, 576, 1), (0, 3, 1500, 1, 1), (1, 2, 5, 300, 1), (2, 1, 1, 1, 1), (3, 2, 33, 555, 1), (3, 1, 1, 130, 1)]
    segs, n = O.make_segments(rows)
    X = rng.standard_normal((n, 64)).astype(np.float32)
    plan = B.Plan(rows, [0, 4, 8, 12, 16], 64, B.MAS_F32, B.default_params(select_mode=2))
    prm = O.default_params(select_mode=2)
    vals = (rng.integers(0, 64, n) / 64.0).astype(np.float32)
    seg_mas = np.array([0.3, 0.999, 0.0, 0.5, 0.123456, 1.0], np.float32)
    so_in = torch.zeros(len(rows) * 36, dtype=torch.uint8, device="cuda")
    so_np = B.seg_out_numpy(so_in.cpu()).copy()
    so_np["mas"] = seg_mas
    so_in.copy_(torch.from_numpy(so_np.view(np.uint8).reshape(-1)))
    o = plan.select_compact(torch.from_numpy(X).cuda(), torch.from_numpy(vals).cuda(), seg_out=so_in)
    mask_r, idx_r, off_r, Y_r, so_r = O.select_compact(segs, prm, X, vals, seg_mas=seg_mas)
    off = o["kept_off"].cpu().numpy()
    assert np.array_equal(off, off_r)
    assert list(np.diff(off)) == [P.adaptive_keep(m, r[2] * r[3]) for m, r in zip(seg_mas, rows)]
    assert np.array_equal(o["keep_mask"].cpu().numpy(), mask_r)
    tot = int(off[-1])
    assert np.array_equal(o["kept_idx"].cpu().numpy()[:tot], idx_r[:tot])
    assert np.array_equal(o["Y"].cpu().numpy()[:tot], Y_r[:tot])
    from paper_2604_02945_b200.binding import lib, _ptr
    rc = lib.mas_select_compact(plan._h, None, _ptr(torch.from_numpy(vals).cuda()), None, None, None, None, 0, None, None)
    assert rc == B.MAS_ERR_INVALID_ARG
    plan.close()


def test_separate_query_norm_launch_gives_identical_results(B):
    """The fallback for devices where the score kernel cannot be launched cooperatively: same bits."""
    w = synth.video(seed=21, R=2, T=3, P=300, d=256, L=33)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    a = plan.forward(X, Q)
    torch.cuda.synchronize()
    n_inline = plan.forward_launches
    plan.set_inline_query_norms(False)
    assert plan.forward_launches == n_inline + 1
    b = plan.forward(X, Q)
    torch.cuda.synchronize()
    for k in ("m_spatial", "gamma", "rel", "mas_tok", "keep_mask", "kept_idx", "kept_off", "Y"):
        assert torch.equal(a[k], b[k]), k
    plan.close()


# ---------------------------------------------------------------- NEXT-1: literal LSH temporal probe (Eq. 5)
def _popcount64(a):
    a = a.astype(np.uint64)
    return np.array([bin(int(v)).count("1") for v in a], np.int64)


@pytest.mark.parametrize("w", [synth.video(seed=31, R=2, T=4, P=300, d=256, L=8), synth.video(seed=32, R=1, T=3, P=70, d=200, L=4, dtype="f32"),
                               synth.audio_vision(seed=33, R=2, d=128, L=5, P_img=130, T_aud=260)],
                         ids=["video_bf16", "video_f32_d200", "audio_vision"])
def test_temporal_lsh_matches_oracle(B, w):
    rng = np.random.default_rng(1234)
    Rf = rng.standard_normal((64, w.d)).astype(np.float32)
    Rm = synth.f32_to_bf16_bits(Rf) if w.dtype == "bf16" else Rf
    segs, n = O.make_segments(w.segments)
    sig_r, g_r, proj = O.temporal_lsh(segs, w.X, Rm, want_proj=True)
    plan = _plan(B, w)
    sig_t, g_t = plan.temporal_lsh(B.to_device(w.X), B.to_device(Rm))
    torch.cuda.synchronize()
    sig_g = sig_t.cpu().numpy().view(np.uint64)
    g_g = g_t.cpu().numpy()
    # a hash bit is decided by the sign of a projection: both sides must agree wherever the oracle's projection is not
    # within rounding distance of zero (fp32 accumulation of exact bf16 products: ~1e-5 |x||r|; fp32 inputs go through a
    # hi/lo bf16 split: ~1e-4)
    Xf = synth.bf16_bits_to_f32(w.X) if w.dtype == "bf16" else w.X
    Rff = synth.bf16_bits_to_f32(Rm) if w.dtype == "bf16" else Rm
    bound = 2e-4 * np.linalg.norm(Xf.astype(np.float64), axis=1)[:, None] * np.linalg.norm(Rff.astype(np.float64), axis=1)[None, :]
    decided = np.abs(proj) > bound
    bits_r = ((sig_r[:, None] >> np.arange(64, dtype=np.uint64)[None, :]) & np.uint64(1)).astype(bool)
    bits_g = ((sig_g[:, None] >> np.arange(64, dtype=np.uint64)[None, :]) & np.uint64(1)).astype(bool)
    assert decided.mean() > 0.99
    assert np.array_equal(bits_r[decided], bits_g[decided])
    # gamma: exact function of the GPU's own signatures ...
    row = 0
    for (req, mod, T, P, k) in w.segments:
        sl = slice(row, row + T * P)
        if T == 1:
            assert np.all(g_g[sl] == 0.0)
        else:
            assert np.all(g_g[row:row + P] == 1.0)
            want = _popcount64(sig_g[row + P:row + T * P] ^ sig_g[row:row + (T - 1) * P]) / 64.0
            assert np.array_equal(g_g[row + P:row + T * P], want.astype(np.float32))
        row += T * P
    # ... and within the undecided bits of the two rows of the oracle's gamma
    und = (~decided).sum(1)
    row = 0
    for (req, mod, T, P, k) in w.segments:
        if T > 1:
            i = np.arange(row + P, row + T * P)
            assert np.all(np.abs(g_g[i] - g_r[i]) <= (und[i] + und[i - P]) / 64.0 + 1e-7)
        row += T * P
    # bit-identical rows (the static patches of the video recipe) collide on every hash
    same = np.zeros(n, bool)
    row = 0
    for (req, mod, T, P, k) in w.segments:
        if T > 1:
            i = np.arange(row + P, row + T * P)
            same[i] = np.all(w.X[i] == w.X[i - P], axis=1)
        row += T * P
    assert np.all(g_g[same] == 0.0)
    plan.close()


@pytest.mark.parametrize("w", [synth.video(seed=41, R=2, T=4, P=300, d=256, L=48), synth.batched_images(seed=42, R=3, d=512, L_lo=5, L_hi=64, P=600),
                               synth.ragged(seed=43, R=6, d=128, n_lo=50, n_hi=500, L_lo=60, L_hi=128)],
                         ids=["video_fused", "images_fused_double_tiles", "ragged_L128_staged_fallback"])
def test_forward_lsh_one_pass(B, w):
    """mas_forward_lsh = mas_forward (same outputs up to the summation grouping of the row statistics, which follows the
    chunk geometry) + signatures that match the oracle on every decided bit."""
    rng = np.random.default_rng(4321)
    Rm = synth.f32_to_bf16_bits(rng.standard_normal((64, w.d)).astype(np.float32))
    segs, n = O.make_segments(w.segments)
    sig_r, g_r, proj = O.temporal_lsh(segs, w.X, Rm, want_proj=True)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    base = plan.forward(X, Q)
    o, sig_t, g_t = plan.forward_lsh(X, Q, B.to_device(Rm))
    torch.cuda.synchronize()
    for k in ("m_spatial", "gamma", "rel", "mas_tok"):
        assert torch.allclose(base[k], o[k], rtol=2e-5, atol=1e-6), k
    assert torch.equal(base["kept_off"], o["kept_off"])
    assert (base["keep_mask"] != o["keep_mask"]).float().mean().item() < 1e-3          # only exact near-ties may flip
    tot = int(o["kept_off"][-1].item())
    assert torch.equal(o["Y"][:tot].view(torch.uint8), X[o["kept_idx"][:tot].long()].view(torch.uint8))
    sig_g = sig_t.cpu().numpy().view(np.uint64)
    Xf, Rf = synth.bf16_bits_to_f32(w.X).astype(np.float64), synth.bf16_bits_to_f32(Rm).astype(np.float64)
    decided = np.abs(proj) > 2e-4 * np.linalg.norm(Xf, axis=1)[:, None] * np.linalg.norm(Rf, axis=1)[None, :]
    sh = np.arange(64, dtype=np.uint64)[None, :]
    bits_r = ((sig_r[:, None] >> sh) & np.uint64(1)).astype(bool)
    bits_g = ((sig_g[:, None] >> sh) & np.uint64(1)).astype(bool)
    assert decided.mean() > 0.99 and np.array_equal(bits_r[decided], bits_g[decided])
    g_g = g_t.cpu().numpy()
    row = 0
    for (req, mod, T, P, k) in w.segments:
        if T == 1:
            assert np.all(g_g[row:row + P] == 0.0)
        else:
            assert np.all(g_g[row:row + P] == 1.0)
            want = _popcount64(sig_g[row + P:row + T * P] ^ sig_g[row:row + (T - 1) * P]) / 64.0
            assert np.array_equal(g_g[row + P:row + T * P], want.astype(np.float32))
        row += T * P
    plan.close()


# ---------------------------------------------------------------- NEXT-4: draft-confidence entropy (Eq. 9-10)
@pytest.mark.parametrize("n,V,dtype", [(5, 1000, "f32"), (7, 4100, "bf16"), (64, 151936, "bf16"), (3, 151936, "f32"), (300, 8, "bf16")],
                         ids=["small_f32", "ragged_bf16", "qwen_vocab_bf16", "qwen_vocab_f32_few_rows", "tiny_vocab_many_rows"])
def test_draft_entropy_matches_oracle(B, n, V, dtype):
    L = synth.draft_logits(seed=11, n_rows=n, V=V, dtype=dtype)
    theta = 2.5
    H_r, f_r = O.draft_entropy(L, theta)
    Vp = (V + 7) // 8 * 8 + 8                                        # padded row stride (16-byte multiple), not V
    dev = torch.zeros((n, Vp), dtype=torch.bfloat16 if dtype == "bf16" else torch.float32, device="cuda")
    dev[:, :V] = B.to_device(L)
    dev[:, V:] = 50.0                                                # poison the padding: it must not be read
    H, sp = B.draft_entropy(dev[:, :V], theta)
    torch.cuda.synchronize()
    H = H.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(H - H_r) <= 2e-4 * np.abs(H_r) + 2e-4), np.abs(H - H_r).max()
    decided = np.abs(H_r - theta) > 1e-3
    assert np.array_equal(sp.cpu().numpy()[decided], f_r[decided])
    assert H.min() >= -1e-4 and H.max() <= np.log(V) + 1e-3


def test_draft_entropy_with_masked_logits(B):
    """Logits of -inf (top-k / top-p filtered drafts) contribute nothing (0 ln 0 = 0, SPEC NEXT-4); a row with one finite logit has H = 0."""
    rng = np.random.default_rng(77)
    n, V = 6, 5000
    L = (3.0 * rng.standard_normal((n, V))).astype(np.float32)
    L[0, 50:] = -np.inf                                   # 50 candidates survive
    L[1, :] = -np.inf; L[1, 4321] = 2.5                   # one survivor: H = 0
    L[2, ::2] = -np.inf                                   # every other logit masked (whole 16-byte groups stay mixed)
    L[3, :4096] = -np.inf                                 # the leading groups are entirely masked
    L[4, 8:16] = -np.inf                                  # one whole 16-byte group of a bf16 row
    for dtype in ("f32", "bf16"):
        Lh = L if dtype == "f32" else synth.f32_to_bf16_bits(L)
        H, sp = B.draft_entropy(B.to_device(Lh), 2.0)
        torch.cuda.synchronize()
        H_r, f_r = O.draft_entropy(Lh, 2.0)
        Hg = H.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(Hg)) and abs(Hg[1]) < 1e-6
        assert np.all(np.abs(Hg - H_r) <= 2e-4 * H_r + 2e-4), (dtype, Hg, H_r)
        decided = np.abs(H_r - 2.0) > 1e-3
        assert np.array_equal(sp.cpu().numpy()[decided], f_r[decided])


# ---------------------------------------------------------------- NEXT-2: learned heads (Eq. 3, Eq. 6 with supplied weights)
def _head_weights(rng, d, hidden, dtype):
    W = np.zeros((64, d), np.float32)
    Wp = np.zeros((64, d), np.float32)
    W[0] = rng.standard_normal(d) * (1.5 / np.sqrt(d))               # logits of O(1): M spreads around tau_s
    W[1:1 + hidden] = rng.standard_normal((hidden, d)) / np.sqrt(d)
    Wp[1:1 + hidden] = rng.standard_normal((hidden, d)) / np.sqrt(d)
    W[1 + hidden:] = 3.0                                             # ignored rows
    b1 = np.zeros(64, np.float32)
    w2 = np.zeros(64, np.float32)
    b1[1:1 + hidden] = 0.3 * rng.standard_normal(hidden)
    w2[1:1 + hidden] = rng.standard_normal(hidden)
    b1[0] = w2[0] = 9.0                                              # ignored entries
    if dtype == "bf16":
        return synth.f32_to_bf16_bits(W), synth.f32_to_bf16_bits(Wp), b1, w2
    return W, Wp, b1, w2


@pytest.mark.parametrize("w", [synth.batched_images(seed=51, R=5, d=512, L_lo=3, L_hi=70, P=333), synth.video(seed=52, R=2, T=4, P=576, d=256, L=48),
                               synth.video(seed=53, R=2, T=5, P=50, d=200, L=9, dtype="f32"), synth.audio_vision(seed=54, R=3, d=256, L=64, P_img=576, T_aud=300),
                               synth.single_image(seed=55, d=1024, dtype="f32")],
                         ids=["images", "video", "video_f32_d200", "audio_vision", "single_image_f32"])
@pytest.mark.parametrize("hidden", [1, 16, 63])
def test_learned_heads(B, w, hidden):
    rng = np.random.default_rng(500 + hidden)
    W, Wp, b1, w2 = _head_weights(rng, w.d, hidden, w.dtype)
    b_sp, b2 = -0.8, 0.15
    segs, n = O.make_segments(w.segments)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    gam = plan.temporal(X)
    m, so = plan.learned_heads(X, Q, gam, B.to_device(W), B.to_device(Wp), torch.from_numpy(b1).cuda(), torch.from_numpy(w2).cuda(), b_sp, b2, hidden)
    torch.cuda.synchronize()
    g = B.seg_out_numpy(so)
    ref_m, ref = O.learned_heads(segs, w.q_off, _oracle_params(w), w.X, w.Q, gam.cpu().numpy().astype(np.float64), W, Wp, b1, w2, b_sp, b2, hidden)
    P.assert_close(m.cpu().numpy(), ref_m, "m_spatial (learned)")
    r0 = 0
    for k, (_, _, T, Pn, _) in enumerate(w.segments):
        nk = T * Pn
        near = np.count_nonzero(np.abs(ref_m[r0:r0 + nk] - 0.3) <= 1e-3 * 0.3)
        assert abs(float(g["rho_spatial"][k]) - ref[k].rho_spatial) <= near / nk + 1e-6
        # alpha = w2 . relu(pre) + b2 may cancel to any small value: the absolute term is the pre-activations' error (fp32 tensor-core
        # column sums, ~1e-6 of their O(1) scale; hidden layer and softmax in double) times sum |w2|
        assert abs(float(g["alpha_mean"][k]) - ref[k].alpha_mean) <= P.RTOL * abs(ref[k].alpha_mean) + 1e-5 * np.sum(np.abs(w2)), (k, float(g["alpha_mean"][k]), ref[k].alpha_mean)
        assert abs(float(g["gamma_avg"][k]) - ref[k].gamma_avg) <= 1e-5
        assert abs(float(g["beta"][k]) - ref[k].beta) <= P.RTOL * abs(ref[k].beta) + P.ATOL, (k, float(g["beta"][k]), ref[k].beta)
        assert abs(float(g["mas"][k]) - ref[k].mas) <= P.RTOL * abs(ref[k].mas) + P.ATOL + 0.6 * near / nk
        assert int(g["n_tokens"][k]) == nk
        r0 += nk
    # softmax identity per request on the GPU's own numbers
    req = np.array([s[0] for s in w.segments])
    for r in range(w.n_requests):
        assert abs(float(g["beta"][req == r].sum()) - 1.0) < 1e-5
    plan.close()


def _check_learned(B, w, m, so, gamma_np, W, Wp, b1, w2, b_sp, b2, hidden):
    segs, n = O.make_segments(w.segments)
    g = B.seg_out_numpy(so)
    ref_m, ref = O.learned_heads(segs, w.q_off, _oracle_params(w), w.X, w.Q, gamma_np.astype(np.float64), W, Wp, b1, w2, b_sp, b2, hidden)
    P.assert_close(m.cpu().numpy(), ref_m, "m_spatial (learned)")
    r0 = 0
    for k, (_, _, T, Pn, _) in enumerate(w.segments):
        nk = T * Pn
        near = np.count_nonzero(np.abs(ref_m[r0:r0 + nk] - 0.3) <= 1e-3 * 0.3)
        assert abs(float(g["rho_spatial"][k]) - ref[k].rho_spatial) <= near / nk + 1e-6
        assert abs(float(g["alpha_mean"][k]) - ref[k].alpha_mean) <= P.RTOL * abs(ref[k].alpha_mean) + 1e-5 * np.sum(np.abs(w2)), (k, float(g["alpha_mean"][k]), ref[k].alpha_mean)
        assert abs(float(g["gamma_avg"][k]) - ref[k].gamma_avg) <= 1e-5
        assert abs(float(g["beta"][k]) - ref[k].beta) <= P.RTOL * abs(ref[k].beta) + P.ATOL, (k, float(g["beta"][k]), ref[k].beta)
        assert abs(float(g["mas"][k]) - ref[k].mas) <= P.RTOL * abs(ref[k].mas) + P.ATOL + 0.6 * near / nk
        assert int(g["n_tokens"][k]) == nk
        r0 += nk


@pytest.mark.parametrize("name", ["images", "video", "audio_vision_L64", "tile_heights", "cluster8", "images_L70_fallback", "video_f32_fallback"])
def test_forward_heads_one_pass(B, name):
    """mas_forward_heads = mas_forward (same outputs up to the summation grouping of the row statistics) + the learned
    descriptors, with the weight rows riding the score kernel's MMA where the fast path applies (else the staged fallback)."""
    if name in SWEEPS:
        shapes, d, L = SWEEPS[name]
        w = _random_workload(400, shapes, d, [min(l, 64) for l in L])
    else:
        w = {"images": lambda: synth.batched_images(seed=61, R=6, d=512, L_lo=3, L_hi=64, P=333),
             "video": lambda: synth.video(seed=62, R=2, T=4, P=576, d=256, L=48),
             "audio_vision_L64": lambda: synth.audio_vision(seed=63, R=2, d=256, L=64, P_img=576, T_aud=300),
             "images_L70_fallback": lambda: synth.batched_images(seed=64, R=4, d=512, L_lo=60, L_hi=70, P=200),
             "video_f32_fallback": lambda: synth.video(seed=65, R=1, T=3, P=70, d=200, L=4, dtype="f32")}[name]()
    hidden = 24
    rng = np.random.default_rng(77)
    W, Wp, b1, w2 = _head_weights(rng, w.d, hidden, w.dtype)
    b_sp, b2 = -0.8, 0.15
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    base = plan.forward(X, Q)
    o, m, so = plan.forward_heads(X, Q, B.to_device(W), B.to_device(Wp), torch.from_numpy(b1).cuda(), torch.from_numpy(w2).cuda(), b_sp, b2, hidden)
    torch.cuda.synchronize()
    for k in ("m_spatial", "gamma", "rel", "mas_tok"):
        assert torch.allclose(base[k], o[k], rtol=2e-5, atol=1e-6), k
    assert torch.equal(base["kept_off"], o["kept_off"])
    assert (base["keep_mask"] != o["keep_mask"]).float().mean().item() < 1e-3          # only exact near-ties may flip
    tot = int(o["kept_off"][-1].item())
    assert torch.equal(o["Y"][:tot].view(torch.uint8), X[o["kept_idx"][:tot].long()].view(torch.uint8))
    _check_learned(B, w, m, so, o["gamma"].cpu().numpy(), W, Wp, b1, w2, b_sp, b2, hidden)
    # twice in a row on the same plan: the scratch partials and counters are re-armed
    o2, m2, so2 = plan.forward_heads(X, Q, B.to_device(W), B.to_device(Wp), torch.from_numpy(b1).cuda(), torch.from_numpy(w2).cuda(), b_sp, b2, hidden)
    torch.cuda.synchronize()
    assert torch.equal(m, m2) and torch.equal(so, so2)
    plan.close()


def test_learned_heads_argument_checks(B):
    w = synth.video(seed=56, R=1, T=3, P=40, d=64, L=4)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    W, Wp, b1, w2 = _head_weights(np.random.default_rng(1), w.d, 4, "bf16")
    args = (B.to_device(W), B.to_device(Wp), torch.from_numpy(b1).cuda(), torch.from_numpy(w2).cuda(), 0.0, 0.0)
    for hidden in (0, 64):
        with pytest.raises(Exception):
            plan.learned_heads(X, Q, plan.temporal(X), *args, hidden)
    with pytest.raises(Exception):
        plan.learned_heads(X, Q, None, *args, 4)             # temporal segment without gamma
    plan.close()


# ---------------------------------------------------------------- NEXT-3: pooling, merged token, residual coding
def _grid_w(w):
    """A grid width per segment: the largest divisor of P not above sqrt(P) (24 for 576; 1 for audio frames)."""
    out = []
    for (_, _, T, P, _) in w.segments:
        W = max(v for v in range(1, int(P ** 0.5) + 1) if P % v == 0)
        out.append(P // W if P // W <= 64 else W)
    return out


@pytest.mark.parametrize("w", [synth.batched_images(seed=71, R=4, d=128, L_lo=3, L_hi=9, P=576), synth.video(seed=72, R=2, T=4, P=300, d=128, L=8),
                               synth.audio_vision(seed=73, R=2, d=64, L=5, P_img=130, T_aud=260)], ids=["images", "video", "audio_vision"])
@pytest.mark.parametrize("k", [1, 2, 3, 5])
def test_spatial_pool(B, w, k):
    segs, n = O.make_segments(w.segments)
    gw = _grid_w(w)
    plan = _plan(B, w)
    s, _ = plan.spatial(B.to_device(w.X))
    out = plan.spatial_pool(s, gw, k)
    torch.cuda.synchronize()
    ref = O.spatial_pool(segs, gw, k, s.cpu().numpy().astype(np.float64))        # both sides pool the same fp32 map
    assert np.allclose(out.cpu().numpy(), ref, rtol=2e-6, atol=0)
    if k == 1:
        assert torch.equal(out, s)
    with pytest.raises(Exception):
        plan.spatial_pool(s, [7] * len(gw), k)                                   # 7 divides none of these P
    plan.close()


@pytest.mark.parametrize("w", [synth.batched_images(seed=74, R=5, d=512, L_lo=3, L_hi=9, P=333), synth.video(seed=75, R=2, T=4, P=300, d=2304, L=8),
                               synth.video(seed=76, R=1, T=3, P=70, d=200, L=4, dtype="f32"), synth.audio_vision(seed=77, R=2, d=256, L=5, P_img=130, T_aud=260),
                               synth.video(seed=78, R=1, T=3, P=70, d=6144, L=4),      # 12 KB rows: four vectors per lane in the bulk-copy merge
                               synth.video(seed=79, R=1, T=2, P=40, d=9216, L=4)],     # 18 KB rows: beyond the bulk-copy merge, the LSU kernel
                         ids=["images", "video_d2304", "video_f32_d200", "audio_vision", "video_d6144", "video_d9216"])
def test_merge_dropped_and_residual_gather(B, w):
    segs, n = O.make_segments(w.segments)
    plan = _plan(B, w)
    X, Q = B.to_device(w.X), B.to_device(w.Q)
    o = plan.forward(X, Q)
    torch.cuda.synchronize()
    mask = o["keep_mask"].cpu().numpy()
    # merged token: fp32 sums of up to P rows against the oracle's double mean
    Y, nd = plan.merge_dropped(X, o["keep_mask"])
    torch.cuda.synchronize()
    Yr, ndr = O.merge_dropped(segs, w.X, mask)
    assert np.array_equal(nd.cpu().numpy(), ndr)
    Xf = (synth.bf16_bits_to_f32(w.X) if w.dtype == "bf16" else w.X).astype(np.float64)
    scale = np.sqrt((Xf ** 2).mean())
    assert np.allclose(Y.cpu().numpy(), Yr, rtol=1e-4, atol=1e-5 * scale)
    # residual gather: bit-exact against the oracle on the GPU's own kept list
    tot = int(o["kept_off"][-1].item())
    idx = o["kept_idx"][:tot].cpu().numpy()
    Yres = plan.gather_residual(X, o["kept_idx"], o["kept_off"])
    torch.cuda.synchronize()
    ref = O.gather_residual(segs, w.X, idx)
    got = Yres[:tot].cpu()
    got = got.view(torch.int16).numpy().view(np.uint16) if w.dtype == "bf16" else got.numpy()
    assert np.array_equal(got, ref)
    # key-frame and image rows are plain copies: identical to the plain gather there
    seg_of = np.concatenate([np.full(s[2] * s[3], k) for k, s in enumerate(w.segments)])
    row0 = np.concatenate([[0], np.cumsum([s[2] * s[3] for s in w.segments])])
    is_res = np.array([w.segments[seg_of[r]][2] > 1 and r - row0[seg_of[r]] >= w.segments[seg_of[r]][3] for r in idx])
    plain = o["Y"][:tot].cpu()
    plain = plain.view(torch.int16).numpy().view(np.uint16) if w.dtype == "bf16" else plain.numpy()
    assert np.array_equal(got[~is_res], plain[~is_res])
    # capacity: nothing past cap_rows
    cap = max(1, tot // 3)
    Yc = plan.gather_residual(X, o["kept_idx"], o["kept_off"], cap_rows=cap)
    torch.cuda.synchronize()
    gc = Yc[:cap].cpu()
    gc = gc.view(torch.int16).numpy().view(np.uint16) if w.dtype == "bf16" else gc.numpy()
    assert np.array_equal(gc, ref[:cap])
    plan.close()


# ---------------------------------------------------------------- CUDA graph capture and replay of mas_forward
@pytest.mark.parametrize("w", [synth.batched_images(seed=81, R=6, d=512, L_lo=3, L_hi=64, P=333), synth.video(seed=82, R=2, T=4, P=300, d=256, L=33)],
                         ids=["images", "video"])
def test_forward_in_a_cuda_graph(B, w):
    """The launch-bound inner loop of a server is one graph launch: cooperative score kernel + PDL-chained segment and
    gather kernels are captured once and replayed on new inputs; the grid-wide counters re-arm themselves."""
    plan = _plan(B, w)
    Xs, Qs = B.to_device(w.X).clone(), B.to_device(w.Q).clone()           # static buffers of the graph
    out = plan.alloc_outputs()
    eager = plan.forward(Xs, Qs)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        plan.forward(Xs, Qs, out=out)                                    # warm-up on the capture stream
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        plan.forward(Xs, Qs, out=out)
    for rep in range(3):
        g.replay()
    torch.cuda.synchronize()
    for k in ("m_spatial", "gamma", "rel", "mas_tok", "keep_mask", "kept_idx", "kept_off", "Y"):
        assert torch.equal(eager[k], out[k]), k
    # new inputs through the same graph: rows reversed inside the static buffer
    w2 = synth.batched_images(seed=83, R=6, d=512, L_lo=3, L_hi=64, P=333) if w.name.startswith("batched") else synth.video(seed=84, R=2, T=4, P=300, d=256, L=33)
    if w2.X.shape == w.X.shape and w2.Q.shape == w.Q.shape and np.array_equal(w2.q_off, w.q_off):
        Xs.copy_(B.to_device(w2.X)); Qs.copy_(B.to_device(w2.Q))
        g.replay()
        torch.cuda.synchronize()
        fresh = plan.forward(B.to_device(w2.X), B.to_device(w2.Q))
        torch.cuda.synchronize()
        for k in ("mas_tok", "keep_mask", "kept_idx", "Y"):
            assert torch.equal(fresh[k], out[k]), k
    plan.close()
