"""Cost of the learned heads (NEXT-2, Eq. 3 / Eq. 6 with supplied weights) on one B200:
`python -m paper_2604_02945_b200.heads_bench [--workload batched_images|video] [--hidden 32]`.

Prints one JSON line with the device time per step of mas_forward, of mas_forward_heads (weight rows riding the score
kernel) and of the staged mas_learned_heads, on the synthetic workload of that name, two copies of X rotated so that no
step finds its rows in L2.  Weights are random (the paper's trained ones are unpublished).  Not part of bench.py's
contract (that one measures the MAS pass)."""
import argparse
import ctypes as C
import json

import numpy as np
import torch

from . import binding as B
from . import synth

SEEDS = {"single_image": 0, "batched_images": 1, "video": 2, "audio_vision": 3, "ragged": 4}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="batched_images", choices=sorted(SEEDS))
    ap.add_argument("--hidden", type=int, default=32)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    a = ap.parse_args()
    w = synth.make(a.workload, seed=SEEDS[a.workload])
    rng = np.random.default_rng(0)
    store = synth.f32_to_bf16_bits if w.dtype == "bf16" else (lambda x: np.ascontiguousarray(x, np.float32))
    Xs = [B.to_device(w.X) for _ in range(2)]
    Q = B.to_device(w.Q)
    dt = B.MAS_BF16 if w.dtype == "bf16" else B.MAS_F32
    plan = B.Plan(w.segments, w.q_off, w.d, dt, B.default_params(select_mode=w.select_mode, cut=w.cut))
    W = B.to_device(store((rng.standard_normal((64, w.d)) / np.sqrt(w.d)).astype(np.float32)))
    Wp = B.to_device(store((rng.standard_normal((64, w.d)) / np.sqrt(w.d)).astype(np.float32)))
    b1 = torch.from_numpy((0.3 * rng.standard_normal(64)).astype(np.float32)).cuda()
    w2 = torch.from_numpy(rng.standard_normal(64).astype(np.float32)).cuda()
    hd = B.mas_heads(W.data_ptr(), Wp.data_ptr(), b1.data_ptr(), w2.data_ptr(), -0.8, 0.15, a.hidden, 0)
    m = torch.zeros(w.n_tokens, device="cuda")
    so = torch.zeros(plan.n_segs * 36, dtype=torch.uint8, device="cuda")
    out = plan.alloc_outputs()
    bun = plan._bundle(out)
    gam = plan.temporal(Xs[0])

    def forward(i):
        plan.forward(Xs[i % 2], Q, out=out)

    def forward_heads(i):   # the C calls themselves: no per-step allocation
        B._check(B.lib.mas_forward_heads(plan._h, Xs[i % 2].data_ptr(), Q.data_ptr(), C.byref(hd), m.data_ptr(), so.data_ptr(),
                                         C.byref(bun), None), "mas_forward_heads")

    def learned_heads(i):
        B._check(B.lib.mas_learned_heads(plan._h, Xs[i % 2].data_ptr(), Q.data_ptr(), gam.data_ptr(), C.byref(hd), m.data_ptr(),
                                         so.data_ptr(), None), "mas_learned_heads")

    res = {}
    for name, fn in (("mas_forward", forward), ("mas_forward_heads", forward_heads), ("mas_learned_heads", learned_heads)):
        for i in range(a.warmup):
            fn(i)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(a.steps):
            fn(i)
        e1.record()
        torch.cuda.synchronize()
        res[name] = e0.elapsed_time(e1) / max(a.steps, 1) * 1e3
    print(json.dumps({"metric": "learned heads, device microseconds per step", "unit": "us", "us_per_step": res,
                      "extra_us_over_mas_forward": res["mas_forward_heads"] - res["mas_forward"], "dtype": w.dtype, "data": "synthetic",
                      "config": {"workload": a.workload, "hidden": a.hidden, "n_tokens": w.n_tokens, "d": w.d,
                                 "fused": bool(w.dtype == "bf16" and w.d % 64 == 0 and int(np.diff(w.q_off).max()) <= 64),
                                 "l2": "2 rotating copies of X (%.0f MB each)" % (w.X.nbytes / 1e6)},
                      "steps": a.steps, "warmup": a.warmup}))
    plan.close()


if __name__ == "__main__":
    main()
