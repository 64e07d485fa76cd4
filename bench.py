#!/usr/bin/env python
"""bench.py — one JSON line: MAS-scored+compacted tokens/s of libmsas `mas_forward` on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload batched_images|video|audio_vision|ragged|single_image]
  python bench.py --impl reference ...        # the CPU oracle on the host cores (a deliberately slow baseline)

A "step" is one `mas_forward` (score -> segment/select -> gather) over one synthetic batch already resident in HBM.
N > 1 (torchrun): every rank runs the same per-GPU workload on its own seed (requests are independent: weak scaling, no
data-path collective); time = max over ranks; value = all ranks' tokens / that time.
"""
import argparse
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
L2_BYTES = 126e6


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return float(j["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md 'clocks line'): one streaming
    `nvidia-smi -lms` process, rows tagged with the host time so that only those inside the timed region count."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc, self.t0, self.t1 = index, [], None, None, None

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

    def summary(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=3)
        rows = [f for (t, f) in self.rows if self.t0 is not None and self.t0 <= t <= self.t1] or [f for (_, f) in self.rows[-3:]]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons, "samples": len(rows)}


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of the score kernel from the committed ncu capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    if os.path.exists(p):
        for line in open(p).read().splitlines()[1:]:
            k, v = line.split(",")
            if k == workload:
                return int(v)
    return None


def algorithmic_bytes(w, kept_rows):
    """X once + Q once + kept rows read and written + ~33 B of per-token scalars + 4 B per kept index."""
    e = 2 if w.dtype == "bf16" else 4
    n, d = w.n_tokens, w.d
    score = n * d * e + w.Q.shape[0] * d * e + 12 * n
    total = score + 2 * kept_rows * d * e + 21 * n + 4 * kept_rows
    return score, total


def oracle_sample(w, n_req):
    """The first n_req requests of the workload as oracle inputs."""
    from oracle import mas_ref as O
    seg_req = np.array([s[0] for s in w.segments])
    ks = np.nonzero(seg_req < n_req)[0]
    rows = [w.segments[k] for k in ks]
    n_rows = sum(r[2] * r[3] for r in rows)
    segs, n = O.make_segments(rows)
    prm = O.default_params(select_mode=w.select_mode, cut=w.cut)
    X, Q, q_off = w.X[:n_rows], w.Q[:w.q_off[n_req]], w.q_off[:n_req + 1]
    return lambda: O.forward(segs, q_off, prm, X, Q), n_rows


def run_reference(args, w):
    """--impl reference: the oracle as it stands, single thread, on a bounded sample per step."""
    per_step_req = {"single_image": 1, "batched_images": 4, "video": 1, "audio_vision": 1, "ragged": 2}[args.workload]
    if args.workload == "video":   # one full video request is ~70 s in the oracle: shrink the sample to 2 frames' worth of rows
        from paper_2604_02945_b200 import synth
        w = synth.video(seed=SEEDS["video"], R=1, T=2)
    fn, n_rows = oracle_sample(w, min(per_step_req, w.n_requests))
    for _ in range(args.warmup):
        fn()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        fn()
    dt = time.perf_counter() - t0
    val = n_rows * args.steps / dt
    sample = "first %d request(s) of the workload = %d tokens per step" % (per_step_req, n_rows)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "tokens/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "tokens/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="batched_images", choices=list(SEEDS))
    ap.add_argument("--impl", default="msas", choices=["msas", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--lsh", action="store_true", help="NEXT-1: time mas_forward_lsh (forward + literal LSH probe in the same pass)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "msas" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    from paper_2604_02945_b200 import synth

    if args.impl == "reference":
        if rank != 0:
            return
        run_reference(args, synth.make(args.workload, seed=SEEDS[args.workload]) if args.workload != "video" else None)
        return

    import torch
    import torch.distributed as dist
    from paper_2604_02945_b200 import binding as B     # raises if libmsas.so is missing: no CPU fallback

    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w = synth.make(args.workload, seed=SEEDS[args.workload] + 1000 * rank)
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
    if args.lsh:   # the step becomes mas_forward_lsh: same outputs plus 8 B/token signatures and gamma_lsh
        import ctypes as C
        Rm = B.to_device(synth.f32_to_bf16_bits(np.random.default_rng(99).standard_normal((64, w.d)).astype(np.float32)))
        sig = torch.zeros(plan.N, dtype=torch.int64, device="cuda")
        glsh = torch.zeros(plan.N, dtype=torch.float32, device="cuda")
        bundle = plan._bundle(out)

        def forward(X, Q, out=None):
            B._check(B.lib.mas_forward_lsh(plan._h, B._ptr(X), B._ptr(Q), B._ptr(Rm), B._ptr(sig), B._ptr(glsh), C.byref(bundle),
                                           B._stream_ptr(None)), "mas_forward_lsh")
        plan.forward = forward
        args.no_e2e = True

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        plan.forward(Xs[i % 2], Qs[i % 2], out=out)
    torch.cuda.synchronize()
    kept_rows = int(out["kept_off"][-1].item())

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        sampler.wait_ready()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.t0 = time.perf_counter()
    ev0.record(stream)
    for i in range(args.steps):
        plan.forward(Xs[i % 2], Qs[i % 2], out=out)
    ev1.record(stream)
    barrier()
    sampler.t1 = time.perf_counter()
    ms = ev0.elapsed_time(ev1)
    # per-stage attribution: a second pass with CUDA events between the kernels on the same stream (these events
    # serialise the launches, so the stage times are measured apart from the timed region above, never inside it)
    n_prof = min(args.steps, 50)
    plan.enable_profiling(n_prof)
    for i in range(n_prof):
        plan.forward(Xs[i % 2], Qs[i % 2], out=out)
    torch.cuda.synchronize()
    clocks = sampler.summary() if rank == 0 else None
    stage = np.array([plan.stage_times(i) for i in range(n_prof)])      # [n, 3] ms: score | segment+select | gather
    plan.enable_profiling(0)
    # the dominant kernel on its own: back-to-back launches of the score stage (mas_score, gamma finishing skipped), one event
    # at each end.  The stage events above sit BETWEEN the kernels of a step and serialise them, so their score figure also
    # holds one launch latency; this loop is the kernel's average launch duration in a stream of its own launches.
    sbuf = (torch.empty(w.n_tokens, dtype=torch.float32, device="cuda"), None, torch.empty(w.n_tokens, dtype=torch.float32, device="cuda"))
    n_alone = min(args.steps, 200)
    for i in range(3):
        plan.score(Xs[i % 2], Qs[i % 2], want_gamma=False, out=sbuf)
    torch.cuda.synchronize()
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ea.record(stream)
    for i in range(n_alone):
        plan.score(Xs[i % 2], Qs[i % 2], want_gamma=False, out=sbuf)
    eb.record(stream)
    torch.cuda.synchronize()
    score_alone_ms = ea.elapsed_time(eb) / n_alone

    # ---- end to end through the host-buffer entry point (pinned host inputs, results read back)
    e2e = None
    if not args.no_e2e:
        hX = torch.from_numpy(w.X).view(torch.bfloat16 if w.dtype == "bf16" else torch.float32).pin_memory()
        hQ = torch.from_numpy(w.Q).view(hX.dtype).pin_memory()
        h_out = {k: (torch.empty_like(v, device="cpu").pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in out.items()}
        h_out["gamma"] = h_out["rel"] = h_out["m_spatial"] = None          # the user-facing result: MAS scores, mask, kept rows
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
        d2h = w.n_tokens * (4 + 1) + plan.n_segs * 36 + (plan.n_segs + 1) * 8 + kept_rows * (4 + w.d * e)
        e2e = (e2e_ms, h2d, d2h, n_e2e)

    from paper_2604_02945_b200 import dist as D
    ms, e2e_ms_max, total_tokens = D.reduce_timing(ms, w.n_tokens, device="cuda", extra_ms=e2e[0] if e2e else 0.0)
    if e2e:
        e2e = (e2e_ms_max,) + e2e[1:]

    if rank == 0:
        ms_step = ms / args.steps
        peak, peak_src = measured_peaks()
        score_bytes, total_bytes = algorithmic_bytes(w, kept_rows)
        score_ms = float(stage[:, 0].mean())
        achieved = score_bytes / (score_ms * 1e-3) / 1e9
        achieved_alone = score_bytes / (score_alone_ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": total_tokens / (ms_step * 1e-3), "unit": "tokens/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic",
            "config": {"workload": args.workload, "requests": w.n_requests, "segments": len(w.segments), "tokens": w.n_tokens,
                       "d": w.d, "query_tokens": int(w.q_off[-1]), "kept_rows": kept_rows,
                       "select": "threshold" if w.select_mode else "topk", "entry": "mas_forward_lsh" if args.lsh else "mas_forward", "parallelism": "dp%d (independent requests)" % world,
                       "l2": "X = %.0f MB per copy, two rotating input copies (> %.0f MB L2 on configs 2-5)" % (w.X.nbytes / 1e6, L2_BYTES / 1e6)},
            "clocks": clocks,
            "gpu_launches": args.steps * plan.forward_launches,
            "roofline": {"bound": "hbm", "kernel": "score stage (a0-a3: norms, temporal difference, relevance contraction)",
                         "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic(args.workload),
                         "peak_source": peak_src, "algorithmic_bytes_per_launch": score_bytes, "avg_launch_ms": score_ms,
                         "frac_of_8000_nominal": achieved / 8000.0,
                         "note": "achieved / avg_launch_ms: events around the score stage inside a step (they serialise the step's kernels, so one launch latency is inside); kernel_alone_*: the same kernel in a stream of its own back-to-back launches",
                         "kernel_alone_ms": score_alone_ms, "kernel_alone_achieved": achieved_alone, "kernel_alone_frac": achieved_alone / peak},
            "stages_ms": {"score": score_ms, "segment_select": float(stage[:, 1].mean()), "gather": float(stage[:, 2].mean())},
            "whole_pass": {"algorithmic_bytes": total_bytes, "achieved_gbs": total_bytes / (ms_step * 1e-3) / 1e9,
                           "frac_of_measured_peak": total_bytes / (ms_step * 1e-3) / 1e9 / peak},
        }
        if e2e:
            line["e2e"] = {"value": total_tokens / (e2e[0] * 1e-3), "unit": "tokens/s", "h2d_bytes_per_step": int(e2e[1]),
                           "d2h_bytes_per_step": int(e2e[2]), "steps": e2e[3], "ms_per_step": e2e[0],
                           "api": "mas_forward_host_async, two plans on two streams called alternately (pinned host buffers in, MAS scores + mask + kept rows out, every step)"}
        if world == 1 and not args.no_cpu_baseline:
            n_req = {"single_image": 1, "batched_images": 64, "video": 1, "audio_vision": 3, "ragged": 12}[args.workload]
            wb = w if args.workload != "video" else synth.video(seed=SEEDS["video"], R=1, T=8)
            fn, n_rows = oracle_sample(wb, min(n_req, wb.n_requests))
            t0 = time.perf_counter()
            runs = 0
            while runs == 0 or (time.perf_counter() - t0 < 10.0 and runs < 8):
                fn()
                runs += 1
            dt_o = time.perf_counter() - t0
            line["cpu_baseline"] = {"value": runs * n_rows / dt_o, "unit": "tokens/s", "cores": 1, "kind": "oracle",
                                    "host_cores_available": os.cpu_count(),
                                    "sample": "first %d request(s) = %d tokens, %d run(s), %.1f s" % (min(n_req, wb.n_requests), n_rows, runs, dt_o)}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
