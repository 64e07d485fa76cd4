"""Throughput of mas_draft_entropy (NEXT-4, Eq. 9-10) on one B200: `python -m paper_2604_02945_b200.entropy_bench`.

Prints one JSON line: decode steps (rows of logits) per second, achieved HBM GB/s (algorithmic bytes = every logit read
once) against the measured copy peak in MEASURED_PEAKS.json.  Inputs are synthetic (synth.draft_logits), two copies
rotated so that no step finds its rows in L2.  Not part of bench.py's contract (that one measures the MAS pass)."""
import argparse
import json
import os

import torch

from . import binding as B
from . import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rows", type=int, default=256)
    ap.add_argument("--vocab", type=int, default=151936)
    ap.add_argument("--dtype", default="bf16", choices=["bf16", "f32"])
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    a = ap.parse_args()
    L = synth.draft_logits(seed=7, n_rows=a.rows, V=a.vocab, dtype=a.dtype)
    copies = max(2, int(2 * 126e6 / L.nbytes) + 1)
    Ls = [B.to_device(L) for _ in range(copies)]
    H = torch.empty(a.rows, dtype=torch.float32, device="cuda")
    sp = torch.empty(a.rows, dtype=torch.uint8, device="cuda")
    import ctypes as C
    nb = C.c_size_t(0)
    B._check(B.lib.mas_draft_entropy_workspace_bytes(a.rows, a.vocab, C.byref(nb)), "workspace")
    ws = torch.empty(nb.value, dtype=torch.uint8, device="cuda")
    dt = B.MAS_BF16 if a.dtype == "bf16" else B.MAS_F32
    st = B._stream_ptr(None)
    argsets = [(B._ptr(x), a.rows, a.vocab, x.stride(0), dt, 2.5, B._ptr(H), B._ptr(sp), B._ptr(ws), ws.numel(), st) for x in Ls]

    def step(i):   # the C call itself: the Python convenience wrapper costs more host time than the kernels take
        B._check(B.lib.mas_draft_entropy(*argsets[i % copies]), "mas_draft_entropy")
    for i in range(a.warmup):
        step(i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(a.steps):
        step(i)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / a.steps
    peak, src = 6650.0, "fallback (B200_PROFILING.md)"
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        peak, src = float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    gbs = L.nbytes / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "draft-confidence entropy, decode steps/sec", "value": a.rows / (ms * 1e-3), "unit": "rows/s",
                      "ms_per_step": ms, "dtype": a.dtype, "data": "synthetic",
                      "config": {"workload": "draft_entropy", "rows": a.rows, "vocab": a.vocab, "input_copies": copies,
                                 "l2": "%d rotating copies of %.0f MB" % (copies, L.nbytes / 1e6)},
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "peak_source": src,
                                   "algorithmic_bytes_per_launch": int(L.nbytes)},
                      "gpu_launches": 2 * a.steps}))


if __name__ == "__main__":
    main()
