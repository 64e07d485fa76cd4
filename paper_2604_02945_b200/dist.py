"""Host-side multi-GPU plumbing: requests are independent, so ranks take disjoint request ranges and
never exchange data on the hot path.  The only collectives are the two small reductions a benchmark needs (max of the
per-rank device time, sum of the per-rank token counts), both outside any timed region.  Works on any backend
(`nccl` on GPUs, `gloo` in the CPU tests)."""
import numpy as np
import torch
import torch.distributed as dist

from . import synth


def request_costs(workload):
    """Bytes each request pulls through the score pass: its token rows plus its query rows."""
    e = 2 if workload.dtype == "bf16" else 4
    cost = np.zeros(workload.n_requests, np.float64)
    for (req, _mod, T, P, _k) in workload.segments:
        cost[req] += float(T) * P * workload.d * e
    cost += np.diff(workload.q_off).astype(np.float64) * workload.d * e
    return cost


def shard_for_rank(workload, rank, world_size):
    """(first request, one past the last request) of `rank`: contiguous ranges balanced by request_costs()."""
    return synth.shard_requests(request_costs(workload), world_size)[rank]


def reduce_timing(ms, tokens, device="cpu", extra_ms=0.0):
    """Whole-job timing: (max over ranks of ms, max over ranks of extra_ms, sum over ranks of tokens)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), float(extra_ms), float(tokens)
    t = torch.tensor([ms, extra_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([tokens], dtype=torch.float64, device=device)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(n[0])
