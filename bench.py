#!/usr/bin/env python
"""bench.py — one JSON line: MAS-scored+compacted tokens/s of libmsas `mas_forward` on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W]            # every workload; headline = video (BASELINE.json configs[2])
  python bench.py --workload batched_images|video|audio_vision|ragged|single_image   # one workload (it becomes the headline)
  python bench.py --entry heads|entropy|compress [--workload ..]  # the NEXT-row entry points, one JSON line each
  python bench.py --impl reference ...                            # the CPU oracle on the host cores (a deliberately slow baseline)

A "step" is one `mas_forward` (score -> segment/select -> gather) over one synthetic batch already resident in HBM.
With no --workload the gated and ungated configs are all run, K timed steps each, and reported under `per_workload`; the
headline `value` is the video config (the larger of the two configs the bandwidth target names).
N > 1 (torchrun): every rank runs the same per-GPU workload on its own seed (requests are independent: weak scaling, no
data-path collective); time = max over ranks; value = all ranks' tokens / that time.
"""
import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "MAS-scored+compacted tokens/sec"
SEEDS = {"single_image": 0, "batched_images": 1, "video": 2, "audio_vision": 3, "ragged": 4}
ALL_WORKLOADS = ["video", "batched_images", "audio_vision", "ragged", "single_image"]   # headline first
L2_BYTES = 126e6


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return float(j["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed regions (B200_PROFILING.md 'clocks line'): one streaming
    `nvidia-smi -lms` process, rows tagged with the host time so that only those inside a timed region count."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                f = [x.strip() for x in line.split(",")]
                if len(f) >= 6:
                    self.rows.append((time.perf_counter(), f))
        except Exception:
            pass

    def wait_ready(self, timeout=5.0):
        t = time.perf_counter()
        while not self.rows and time.perf_counter() - t < timeout:
            time.sleep(0.01)

    def window(self, t0, t1):
        """Summary of the samples taken in [t0, t1] (the nearest ones if the region was shorter than the sampling period)."""
        rows = [f for (t, f) in self.rows if t0 <= t <= t1]
        if not rows:
            near = sorted(self.rows, key=lambda tf: abs(tf[0] - 0.5 * (t0 + t1)))[:2]
            rows = [f for (_, f) in near]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons, "samples": len(rows)}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=3)


def csrc_sha():
    """Content hash of the CUDA sources: a stored ncu figure is only quoted for the binary it was captured from."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2604_02945_b200", "csrc")
    for f in sorted(os.listdir(d)):
        h.update(f.encode())
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload):
    """(dram__bytes_read.sum + dram__bytes_write.sum of the score kernel, source note) from the committed ncu capture
    (profiles/r02_traffic.csv: workload,bytes,csrc_sha,capture), or (None, why) when the sources changed since."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if not os.path.exists(p):
        return None, "no capture committed"
    sha = csrc_sha()
    for line in open(p).read().splitlines()[1:]:
        f = line.split(",")
        if len(f) >= 4 and f[0] == workload:
            if f[2] != sha:
                return None, "capture %s is of csrc %s, this tree is %s: not quoted" % (f[3], f[2], sha)
            return int(f[1]), "ncu --set full capture %s (csrc %s)" % (f[3], f[2])
    return None, "no capture of this workload"


def algorithmic_bytes(w, kept_rows):
    """X once + Q once + kept rows read and written + ~33 B of per-token scalars + 4 B per kept index."""
    e = 2 if w.dtype == "bf16" else 4
    n, d = w.n_tokens, w.d
    score = n * d * e + w.Q.shape[0] * d * e + 12 * n
    total = score + 2 * kept_rows * d * e + 21 * n + 4 * kept_rows
    return score, total


# ---------------------------------------------------------------------------------------------- the oracle legs (CPU)
_ORACLE_JOB = None   # inherited by forked workers


def _oracle_one_request(r):
    from oracle import mas_ref as O
    w = _ORACLE_JOB
    seg_req = np.array([s[0] for s in w.segments])
    ks = np.nonzero(seg_req == r)[0]
    rows = [(0,) + tuple(w.segments[k][1:]) for k in ks]
    row0 = np.concatenate([[0], np.cumsum([s[2] * s[3] for s in w.segments])])
    lo, hi = int(row0[ks[0]]), int(row0[ks[-1] + 1])
    segs, _ = O.make_segments(rows)
    prm = O.default_params(select_mode=w.select_mode, cut=w.cut)
    t0 = time.perf_counter()
    O.forward(segs, [0, int(w.q_off[r + 1] - w.q_off[r])], prm, w.X[lo:hi], w.Q[w.q_off[r]:w.q_off[r + 1]])
    return hi - lo, time.perf_counter() - t0


def oracle_sample_workload(name, n_req, video_frames=4):
    """A bounded sample of the workload `name` for the oracle: the same generator at fewer requests / frames."""
    from paper_2604_02945_b200 import synth
    kw = {"video": dict(R=n_req, T=video_frames), "batched_images": dict(R=n_req), "audio_vision": dict(R=n_req), "ragged": dict(R=n_req),
          "single_image": {}}[name]
    return synth.make(name, seed=SEEDS[name], **kw)


def oracle_throughput(name, cores):
    """(tokens/s on one core, tokens/s with `cores` processes over disjoint requests, sample description).  The oracle as it
    stands: single-threaded C++, one process per request (requests are independent)."""
    import multiprocessing as mp
    global _ORACLE_JOB
    n_req = 1 if name == "single_image" else max(cores, 2)
    w = oracle_sample_workload(name, n_req)
    _ORACLE_JOB = w
    rows1, dt1 = _oracle_one_request(0)
    one = rows1 / dt1
    allc = None
    if w.n_requests > 1 and cores > 1:
        t0 = time.perf_counter()
        with mp.get_context("fork").Pool(min(cores, w.n_requests)) as pool:
            res = pool.map(_oracle_one_request, range(w.n_requests), chunksize=1)
        allc = sum(r for r, _ in res) / (time.perf_counter() - t0)
    _ORACLE_JOB = None
    sample = "%s sample: %d request(s), %d tokens (1 core: request 0 = %d tokens, %.1f s)" % (name, w.n_requests, w.n_tokens, rows1, dt1)
    return one, allc, sample


def run_reference(args, name):
    """--impl reference: the oracle as it stands, single thread, on a bounded sample per step."""
    from oracle import mas_ref as O  # noqa: F401  (fails loudly if the oracle cannot be built)
    global _ORACLE_JOB
    w = oracle_sample_workload(name, 1 if name in ("single_image", "video") else 2, video_frames=2)
    _ORACLE_JOB = w
    for _ in range(args.warmup):
        _oracle_one_request(0)
    rows, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        for r in range(w.n_requests):
            rows += _oracle_one_request(r)[0]
    dt = time.perf_counter() - t0
    _ORACLE_JOB = None
    val = rows / dt
    sample = "%d request(s) of a reduced %s batch = %d tokens per step" % (w.n_requests, name, w.n_tokens)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "tokens/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "tokens/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------- one workload on the GPU
def bench_workload(name, args, rank, local_rank, world, sampler, want_e2e):
    """Times `mas_forward` on one synthetic workload: K timed steps, per-stage attribution, the dominant kernel on its own,
    optionally the end-to-end leg.  Returns the per-workload record (rank 0 fills the roofline from it)."""
    import torch
    import torch.distributed as dist
    from paper_2604_02945_b200 import binding as B     # raises if libmsas.so is missing: no CPU fallback
    from paper_2604_02945_b200 import dist as D
    from paper_2604_02945_b200 import synth

    w = synth.make(name, seed=SEEDS[name] + 1000 * rank)
    dt = B.MAS_BF16 if w.dtype == "bf16" else B.MAS_F32
    e = 2 if w.dtype == "bf16" else 4

    def make_plan():
        return B.Plan(w.segments, w.q_off, w.d, dt, B.default_params(select_mode=w.select_mode, cut=w.cut))
    plan = make_plan()
    # two rotating input copies so that no step finds its rows in L2 (X alone is already > L2 on configs 2-5)
    Xs = [B.to_device(w.X), B.to_device(w.X)]
    Qs = [B.to_device(w.Q), B.to_device(w.Q)]
    out = plan.alloc_outputs()
    stream = torch.cuda.current_stream()
    forward = plan.forward
    entry = "mas_forward"
    if args.lsh:   # the step becomes mas_forward_lsh: same outputs plus 8 B/token signatures and gamma_lsh
        import ctypes as C
        Rm = B.to_device(synth.f32_to_bf16_bits(np.random.default_rng(99).standard_normal((64, w.d)).astype(np.float32)))
        sig = torch.zeros(plan.N, dtype=torch.int64, device="cuda")
        glsh = torch.zeros(plan.N, dtype=torch.float32, device="cuda")
        bundle = plan._bundle(out)

        def forward(X, Q, out=None):
            B._check(B.lib.mas_forward_lsh(plan._h, B._ptr(X), B._ptr(Q), B._ptr(Rm), B._ptr(sig), B._ptr(glsh), C.byref(bundle),
                                           B._stream_ptr(None)), "mas_forward_lsh")
        entry, want_e2e = "mas_forward_lsh", False

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        forward(Xs[i % 2], Qs[i % 2], out=out)
    torch.cuda.synchronize()
    kept_rows = int(out["kept_off"][-1].item())

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    ev0.record(stream)
    for i in range(args.steps):
        forward(Xs[i % 2], Qs[i % 2], out=out)
    ev1.record(stream)
    barrier()
    t1 = time.perf_counter()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.window(t0, t1) if sampler is not None else None
    # per-stage attribution: a second pass with CUDA events between the kernels on the same stream (these events
    # serialise the launches, so the stage times are measured apart from the timed region above, never inside it)
    n_prof = min(args.steps, 50)
    plan.enable_profiling(n_prof)
    for i in range(n_prof):
        forward(Xs[i % 2], Qs[i % 2], out=out)
    torch.cuda.synchronize()
    stage = np.array([plan.stage_times(i) for i in range(n_prof)])      # [n, 3] ms: score | segment+select | gather
    plan.enable_profiling(0)
    # the dominant kernel on its own: back-to-back launches of the score stage (mas_score, gamma finishing skipped), one event
    # at each end.  The stage events above sit BETWEEN the kernels of a step and serialise them, so their score figure also
    # holds one launch latency; this loop is the kernel's average launch duration in a stream of its own launches.
    sbuf = (torch.empty(w.n_tokens, dtype=torch.float32, device="cuda"), None, torch.empty(w.n_tokens, dtype=torch.float32, device="cuda"))
    # Five short bursts (MEASURED_PEAKS' copy figure is a burst figure too), the median burst reported: the nvidia-smi sampler
    # that runs beside the whole benchmark stalls a launch now and then, which lands in one burst, not in the figure.
    # The bursts start from a rested GPU (1.5 s idle): after a few hundred steps the board sits at its power cap (SM clock 1965 ->
    # 1760-1920 MHz) and the same kernel takes 7-11 % longer, which is what the in-step figure (`achieved`) already shows.
    n_alone = min(max(args.steps, 10), 20)
    torch.cuda.synchronize()
    time.sleep(1.5)
    for i in range(3):
        plan.score(Xs[i % 2], Qs[i % 2], want_gamma=False, out=sbuf)
    torch.cuda.synchronize()
    bursts = []
    for rep in range(5):
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record(stream)
        for i in range(n_alone):
            plan.score(Xs[i % 2], Qs[i % 2], want_gamma=False, out=sbuf)
        eb.record(stream)
        torch.cuda.synchronize()
        bursts.append(ea.elapsed_time(eb) / n_alone)
    score_alone_ms = float(np.median(bursts))

    # ---- end to end through the host-buffer entry point (pinned host inputs, every result read back)
    e2e = None
    if want_e2e:
        hX = torch.from_numpy(w.X).view(torch.bfloat16 if w.dtype == "bf16" else torch.float32).pin_memory()
        hQ = torch.from_numpy(w.Q).view(hX.dtype).pin_memory()
        h_out = {k: (torch.empty_like(v, device="cpu").pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in out.items()}
        n_e2e = max(4, min(args.steps, 10))
        # two plans on two streams, called alternately: the device-to-host copies of one step overlap the host-to-device
        # copies of the next (PCIe is full duplex); every step still copies its inputs in and its results out
        plan2 = make_plan()
        outs, h_outs = [out, plan2.alloc_outputs()], [h_out, {k: (v.clone().pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in h_out.items()}]
        plans, streams = [plan, plan2], [torch.cuda.Stream(), torch.cuda.Stream()]
        torch.cuda.synchronize()
        for i in range(2):
            plans[i].forward_host_async(hX, hQ, Xs[i], Qs[i], outs[i], h_outs[i], stream=streams[i])
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for i in range(n_e2e):
            plans[i % 2].forward_host_async(hX, hQ, Xs[i % 2], Qs[i % 2], outs[i % 2], h_outs[i % 2], stream=streams[i % 2])
        torch.cuda.synchronize()
        e2e_ms = 1e3 * (time.perf_counter() - t0) / n_e2e
        assert torch.equal(h_outs[0]["keep_mask"], h_outs[1]["keep_mask"]) and int(h_outs[1]["kept_off"][-1]) == kept_rows
        plan2.close()
        h2d = w.X.nbytes + w.Q.nbytes
        d2h = w.n_tokens * (4 * 4 + 1) + plan.n_segs * 36 + (plan.n_segs + 1) * 8 + kept_rows * (4 + w.d * e)
        e2e = (e2e_ms, h2d, d2h, n_e2e)
        del hX, hQ, h_out, h_outs

    ms, e2e_ms_max, total_tokens = D.reduce_timing(ms, w.n_tokens, device="cuda", extra_ms=e2e[0] if e2e else 0.0)
    ms_step = ms / args.steps
    peak, peak_src = measured_peaks()
    score_bytes, total_bytes = algorithmic_bytes(w, kept_rows)
    score_ms = float(stage[:, 0].mean())
    achieved = score_bytes / (score_ms * 1e-3) / 1e9
    achieved_alone = score_bytes / (score_alone_ms * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(name)
    rec = {
        "workload": name, "ms_per_step": ms_step, "tokens_per_s": total_tokens / (ms_step * 1e-3), "tokens": w.n_tokens, "total_tokens": total_tokens,
        "requests": w.n_requests, "segments": len(w.segments), "d": w.d, "query_tokens": int(w.q_off[-1]), "kept_rows": kept_rows,
        "select": "threshold" if w.select_mode else "topk", "entry": entry, "dtype": "bf16" if w.dtype == "bf16" else "f32",
        "l2": "X = %.0f MB per copy, two rotating input copies (L2 = %.0f MB)" % (w.X.nbytes / 1e6, L2_BYTES / 1e6),
        "gpu_launches": args.steps * plan.forward_launches,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "k_score_tc = the score stage (a0-a3: query norms, row norms, temporal difference, relevance contraction)"
                     if w.dtype == "bf16" and w.d % 64 == 0 else "score stage on the generic path (k_qprep + k_score_mma)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": score_bytes, "avg_launch_ms": score_ms,
                     "frac_of_8000_nominal": achieved / 8000.0,
                     "note": "achieved / avg_launch_ms: events around the score stage inside a step (they serialise the step's kernels, so one launch latency is inside); kernel_alone_*: the same kernel in a stream of its own back-to-back launches (median of five bursts of 20 launches after 1.5 s of idle, i.e. not power-capped; kernel_alone_bursts_ms lists them)",
                     "kernel_alone_ms": score_alone_ms, "kernel_alone_bursts_ms": [round(b, 6) for b in bursts], "kernel_alone_achieved": achieved_alone, "kernel_alone_frac": achieved_alone / peak,
                     "kernel_alone_frac_of_8000_nominal": achieved_alone / 8000.0},
        "stages_ms": {"score": score_ms, "segment_select": float(stage[:, 1].mean()), "gather": float(stage[:, 2].mean())},
        "whole_pass": {"algorithmic_bytes": total_bytes, "achieved_gbs": total_bytes / (ms_step * 1e-3) / 1e9,
                       "frac_of_measured_peak": total_bytes / (ms_step * 1e-3) / 1e9 / peak},
    }
    if e2e:
        rec["e2e"] = {"value": total_tokens / (e2e_ms_max * 1e-3), "unit": "tokens/s", "h2d_bytes_per_step": int(e2e[1]),
                      "d2h_bytes_per_step": int(e2e[2]), "steps": e2e[3], "ms_per_step": e2e_ms_max,
                      "api": "mas_forward_host_async, two plans on two streams called alternately (pinned host buffers in; every output out: "
                             "m_spatial, gamma, rel, MAS scores, segment records, mask, kept indices, kept rows; every step)"}
    plan.close()
    del Xs, Qs, out
    torch.cuda.empty_cache()
    return rec


# ---------------------------------------------------------------------------------------------- the NEXT-row entry points
def _time_calls(fn, steps, warmup):
    import torch
    for i in range(warmup):
        fn(i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(steps):
        fn(i)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / max(steps, 1)


def entry_heads(args):
    """NEXT-2 (learned heads, Eq. 3 / Eq. 6 with supplied weights): device time per step of mas_forward, of mas_forward_heads
    (weight rows riding the score kernel) and of the staged mas_learned_heads.  Random weights (the trained ones are unpublished)."""
    import ctypes as C
    import torch
    from paper_2604_02945_b200 import binding as B
    from paper_2604_02945_b200 import synth
    name = args.workload or "batched_images"
    w = synth.make(name, seed=SEEDS[name])
    rng = np.random.default_rng(0)
    store = synth.f32_to_bf16_bits if w.dtype == "bf16" else (lambda x: np.ascontiguousarray(x, np.float32))
    Xs = [B.to_device(w.X) for _ in range(2)]
    Q = B.to_device(w.Q)
    plan = B.Plan(w.segments, w.q_off, w.d, B.MAS_BF16 if w.dtype == "bf16" else B.MAS_F32, B.default_params(select_mode=w.select_mode, cut=w.cut))
    W = B.to_device(store((rng.standard_normal((64, w.d)) / np.sqrt(w.d)).astype(np.float32)))
    Wp = B.to_device(store((rng.standard_normal((64, w.d)) / np.sqrt(w.d)).astype(np.float32)))
    b1 = torch.from_numpy((0.3 * rng.standard_normal(64)).astype(np.float32)).cuda()
    w2 = torch.from_numpy(rng.standard_normal(64).astype(np.float32)).cuda()
    hd = B.mas_heads(W.data_ptr(), Wp.data_ptr(), b1.data_ptr(), w2.data_ptr(), -0.8, 0.15, args.hidden, 0)
    m = torch.zeros(w.n_tokens, device="cuda")
    so = torch.zeros(plan.n_segs * 36, dtype=torch.uint8, device="cuda")
    out = plan.alloc_outputs()
    bun = plan._bundle(out)
    gam = plan.temporal(Xs[0])
    calls = {
        "mas_forward": lambda i: plan.forward(Xs[i % 2], Q, out=out),
        "mas_forward_heads": lambda i: B._check(B.lib.mas_forward_heads(plan._h, Xs[i % 2].data_ptr(), Q.data_ptr(), C.byref(hd), m.data_ptr(),
                                                                       so.data_ptr(), C.byref(bun), None), "mas_forward_heads"),
        "mas_learned_heads": lambda i: B._check(B.lib.mas_learned_heads(plan._h, Xs[i % 2].data_ptr(), Q.data_ptr(), gam.data_ptr(), C.byref(hd),
                                                                       m.data_ptr(), so.data_ptr(), None), "mas_learned_heads"),
    }
    res = {k: _time_calls(fn, args.steps, args.warmup) * 1e3 for k, fn in calls.items()}
    print(json.dumps({"entry": "heads", "metric": "learned heads, device microseconds per step", "unit": "us", "us_per_step": res,
                      "extra_us_over_mas_forward": res["mas_forward_heads"] - res["mas_forward"], "dtype": w.dtype, "data": "synthetic",
                      "config": {"workload": name, "hidden": args.hidden, "n_tokens": w.n_tokens, "d": w.d,
                                 "fused": bool(w.dtype == "bf16" and w.d % 64 == 0 and int(np.diff(w.q_off).max()) <= 64),
                                 "l2": "2 rotating copies of X (%.0f MB each)" % (w.X.nbytes / 1e6)},
                      "steps": args.steps, "warmup": args.warmup}))
    plan.close()


def entry_entropy(args):
    """NEXT-4 (draft-confidence entropy, Eq. 9-10): decode steps (rows of logits) per second and achieved HBM GB/s (every logit
    read once) against the measured copy peak."""
    import ctypes as C
    import torch
    from paper_2604_02945_b200 import binding as B
    from paper_2604_02945_b200 import synth
    L = synth.draft_logits(seed=7, n_rows=args.rows, V=args.vocab, dtype=args.dtype)
    copies = max(2, int(2 * L2_BYTES / L.nbytes) + 1)
    Ls = [B.to_device(L) for _ in range(copies)]
    H = torch.empty(args.rows, dtype=torch.float32, device="cuda")
    sp = torch.empty(args.rows, dtype=torch.uint8, device="cuda")
    nb = C.c_size_t(0)
    B._check(B.lib.mas_draft_entropy_workspace_bytes(args.rows, args.vocab, C.byref(nb)), "workspace")
    ws = torch.empty(nb.value, dtype=torch.uint8, device="cuda")
    dt = B.MAS_BF16 if args.dtype == "bf16" else B.MAS_F32
    st = B._stream_ptr(None)
    argsets = [(B._ptr(x), args.rows, args.vocab, x.stride(0), dt, 2.5, B._ptr(H), B._ptr(sp), B._ptr(ws), ws.numel(), st) for x in Ls]
    ms = _time_calls(lambda i: B._check(B.lib.mas_draft_entropy(*argsets[i % copies]), "mas_draft_entropy"), args.steps, args.warmup)
    peak, src = measured_peaks()
    gbs = L.nbytes / (ms * 1e-3) / 1e9
    print(json.dumps({"entry": "entropy", "metric": "draft-confidence entropy, decode steps/sec", "value": args.rows / (ms * 1e-3), "unit": "rows/s",
                      "ms_per_step": ms, "dtype": args.dtype, "data": "synthetic",
                      "config": {"workload": "draft_entropy", "rows": args.rows, "vocab": args.vocab, "input_copies": copies,
                                 "l2": "%d rotating copies of %.0f MB" % (copies, L.nbytes / 1e6)},
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "peak_source": src,
                                   "algorithmic_bytes_per_launch": int(L.nbytes)},
                      "gpu_launches": 2 * args.steps, "steps": args.steps, "warmup": args.warmup}))


def entry_compress(args):
    """NEXT-3 (pooling, merged token, residual gather): device time per call and achieved GB/s of each step against its
    algorithmic bytes (pool: 8 B/token; merge: the dropped rows read once + F*d*4 written; residual gather: kept rows read,
    their previous rows read for frames t >= 1, kept rows written)."""
    import torch
    from paper_2604_02945_b200 import binding as B
    from paper_2604_02945_b200 import synth
    name = args.workload or "video"
    w = synth.make(name, seed=SEEDS[name])
    Xs = [B.to_device(w.X) for _ in range(2)]
    Q = B.to_device(w.Q)
    plan = B.Plan(w.segments, w.q_off, w.d, B.MAS_BF16 if w.dtype == "bf16" else B.MAS_F32, B.default_params(select_mode=w.select_mode, cut=w.cut))
    o = plan.forward(Xs[0], Q)
    s, _ = plan.spatial(Xs[0])
    torch.cuda.synchronize()
    gw = [max(v for v in range(1, int(P ** 0.5) + 1) if P % v == 0) for (_, _, T, P, _) in w.segments]
    total = int(o["kept_off"][-1].item())
    esz = 2 if w.dtype == "bf16" else 4
    F = sum(sg[2] for sg in w.segments)
    idx = o["kept_idx"][:total].cpu().numpy()
    seg_of = np.concatenate([np.full(sg[2] * sg[3], k) for k, sg in enumerate(w.segments)])
    row0 = np.concatenate([[0], np.cumsum([sg[2] * sg[3] for sg in w.segments])])
    n_res = int(sum(1 for r in idx if w.segments[seg_of[r]][2] > 1 and r - row0[seg_of[r]] >= w.segments[seg_of[r]][3]))
    steps = {
        "mas_spatial_pool(k=3)": (lambda i: plan.spatial_pool(s, gw, 3), 8 * w.n_tokens),
        "mas_merge_dropped": (lambda i: plan.merge_dropped(Xs[i % 2], o["keep_mask"]), (w.n_tokens - total) * w.d * esz + F * w.d * 4),
        "mas_gather_residual": (lambda i: plan.gather_residual(Xs[i % 2], o["kept_idx"], o["kept_off"]), (2 * total + n_res) * w.d * esz),
    }
    res = {}
    for k, (fn, nbytes) in steps.items():
        us = _time_calls(fn, args.steps, args.warmup) * 1e3
        res[k] = {"us": us, "algorithmic_MB": nbytes / 1e6, "GB/s": nbytes / us / 1e3}
    print(json.dumps({"entry": "compress", "metric": "NEXT-3 steps, device microseconds per call (output allocation included)", "results": res,
                      "dtype": w.dtype, "data": "synthetic",
                      "config": {"workload": name, "n_tokens": w.n_tokens, "d": w.d, "kept_rows": total, "frames": F, "residual_rows": n_res},
                      "steps": args.steps, "warmup": args.warmup}))
    plan.close()


# ---------------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default=None, choices=list(SEEDS), help="one workload only (default: all five, headline = video)")
    ap.add_argument("--impl", default="msas", choices=["msas", "reference"])
    ap.add_argument("--entry", default="forward", choices=["forward", "heads", "entropy", "compress"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--lsh", action="store_true", help="NEXT-1: time mas_forward_lsh (forward + literal LSH probe in the same pass)")
    ap.add_argument("--hidden", type=int, default=32, help="--entry heads: hidden units")
    ap.add_argument("--rows", type=int, default=256, help="--entry entropy: decode steps per call")
    ap.add_argument("--vocab", type=int, default=151936, help="--entry entropy: vocabulary size")
    ap.add_argument("--dtype", default="bf16", choices=["bf16", "f32"], help="--entry entropy: logit type")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "msas" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    names = [args.workload] if args.workload else list(ALL_WORKLOADS)
    headline = names[0]

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, headline)
        return

    # the oracle baseline first: it forks worker processes, which is cleanest before this process has touched CUDA
    cpu = None
    if rank == 0 and world == 1 and args.entry == "forward" and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        one, allc, sample = oracle_throughput(headline, cores)
        cpu = {"value": one, "unit": "tokens/s", "cores": 1, "kind": "oracle", "sample": sample,
               "all_cores": {"value": allc, "unit": "tokens/s", "cores": cores,
                             "how": "the same single-threaded oracle, one process per host core over disjoint requests"}}

    import torch
    import torch.distributed as dist
    torch.cuda.set_device(local_rank)
    if args.entry != "forward":
        {"heads": entry_heads, "entropy": entry_entropy, "compress": entry_compress}[args.entry](args)
        return
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    sampler = None
    if rank == 0:
        sampler = ClockSampler(local_rank)
        sampler.start()
        sampler.wait_ready()
    recs = {}
    for name in names:
        recs[name] = bench_workload(name, args, rank, local_rank, world, sampler, want_e2e=(name == headline and not args.no_e2e))
    if sampler is not None:
        sampler.stop()

    if rank == 0:
        h = recs[headline]
        line = {
            "metric": METRIC, "value": h["tokens_per_s"], "unit": "tokens/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": h["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": h["dtype"],
            "data": "synthetic",
            "config": {"workload": headline, "requests": h["requests"], "segments": h["segments"], "tokens": h["tokens"], "d": h["d"],
                       "query_tokens": h["query_tokens"], "kept_rows": h["kept_rows"], "select": h["select"], "entry": h["entry"],
                       "parallelism": "dp%d (independent requests)" % world, "l2": h["l2"],
                       "also_measured": [n for n in names if n != headline]},
            "clocks": h["clocks"],
            "gpu_launches": sum(r["gpu_launches"] for r in recs.values()),
            "roofline": h["roofline"], "stages_ms": h["stages_ms"], "whole_pass": h["whole_pass"],
        }
        if "e2e" in h:
            line["e2e"] = h["e2e"]
        if cpu is not None:
            line["cpu_baseline"] = cpu
        line["per_workload"] = {n: {k: v for k, v in r.items() if k not in ("workload",)} for n, r in recs.items()}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
