"""Cost of the NEXT-3 steps (pooling, merged token, residual gather) on one B200:
`python -m paper_2604_02945_b200.compress_bench [--workload video]`.

Prints one JSON line with the device time per call and the achieved GB/s of each step against its algorithmic bytes
(pool: 8 B/token; merge: the dropped rows read once + F*d*4 written; residual gather: kept rows read, their previous
rows read for frames t >= 1, kept rows written).  Synthetic inputs, two rotating copies of X.  Not part of bench.py."""
import argparse
import json

import torch

from . import binding as B
from . import synth

SEEDS = {"single_image": 0, "batched_images": 1, "video": 2, "audio_vision": 3, "ragged": 4}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="video", choices=sorted(SEEDS))
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    a = ap.parse_args()
    w = synth.make(a.workload, seed=SEEDS[a.workload])
    Xs = [B.to_device(w.X) for _ in range(2)]
    Q = B.to_device(w.Q)
    dt = B.MAS_BF16 if w.dtype == "bf16" else B.MAS_F32
    plan = B.Plan(w.segments, w.q_off, w.d, dt, B.default_params(select_mode=w.select_mode, cut=w.cut))
    o = plan.forward(Xs[0], Q)
    s, _ = plan.spatial(Xs[0])
    torch.cuda.synchronize()
    gw = []
    for (_, _, T, P, _) in w.segments:
        W = max(v for v in range(1, int(P ** 0.5) + 1) if P % v == 0)
        gw.append(W)
    total = int(o["kept_off"][-1].item())
    esz = 2 if w.dtype == "bf16" else 4
    n_drop = w.n_tokens - total
    F = sum(sg[2] for sg in w.segments)
    idx = o["kept_idx"][:total].cpu().numpy()
    import numpy as np
    seg_of = np.concatenate([np.full(sg[2] * sg[3], k) for k, sg in enumerate(w.segments)])
    row0 = np.concatenate([[0], np.cumsum([sg[2] * sg[3] for sg in w.segments])])
    n_res = int(sum(1 for r in idx if w.segments[seg_of[r]][2] > 1 and r - row0[seg_of[r]] >= w.segments[seg_of[r]][3]))
    steps = {
        "mas_spatial_pool(k=3)": (lambda i: plan.spatial_pool(s, gw, 3), 8 * w.n_tokens),
        "mas_merge_dropped": (lambda i: plan.merge_dropped(Xs[i % 2], o["keep_mask"]), n_drop * w.d * esz + F * w.d * 4),
        "mas_gather_residual": (lambda i: plan.gather_residual(Xs[i % 2], o["kept_idx"], o["kept_off"]), (2 * total + n_res) * w.d * esz),
    }
    res = {}
    for name, (fn, nbytes) in steps.items():
        for i in range(a.warmup):
            fn(i)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(a.steps):
            fn(i)
        e1.record()
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) / a.steps * 1e3
        res[name] = {"us": us, "algorithmic_MB": nbytes / 1e6, "GB/s": nbytes / us / 1e3}
    print(json.dumps({"metric": "NEXT-3 steps, device microseconds per call (output allocation included)", "results": res, "dtype": w.dtype,
                      "data": "synthetic", "config": {"workload": a.workload, "n_tokens": w.n_tokens, "d": w.d, "kept_rows": total,
                                                      "frames": F, "residual_rows": n_res}, "steps": a.steps, "warmup": a.warmup}))
    plan.close()


if __name__ == "__main__":
    main()
