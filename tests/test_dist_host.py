"""N > 1 host logic on CPU: two gloo ranks shard the requests of one workload, each runs the pass on its shard (the
oracle stands in for the device here: this test is about the sharding and the reductions, not the kernels) and the
union must equal the single-process result; the timing reduction must be max / sum."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import mas_ref as O
    from paper_2604_02945_b200 import dist as D
    from paper_2604_02945_b200 import synth
    w = synth.batched_images(seed=1, R=5, d=64, P=40)
    lo, hi = D.shard_for_rank(w, rank, world)
    rows = [s for s in w.segments if lo <= s[0] < hi]
    row0 = sum(s[2] * s[3] for s in w.segments if s[0] < lo)
    n_rows = sum(s[2] * s[3] for s in rows)
    rows_local = [(s[0] - lo,) + tuple(s[1:]) for s in rows]
    segs, n = O.make_segments(rows_local)
    assert n == n_rows
    q0, q1 = int(w.q_off[lo]), int(w.q_off[hi])
    ref = O.forward(segs, w.q_off[lo:hi + 1] - w.q_off[lo], O.default_params(), w.X[row0:row0 + n_rows], w.Q[q0:q1], want_Y=False)
    np.save(os.path.join(out_dir, "mas_%d.npy" % rank), ref["mas_tok"])
    np.save(os.path.join(out_dir, "range_%d.npy" % rank), np.array([lo, hi, row0, n_rows]))
    ms, extra, tok = D.reduce_timing(10.0 + rank, n_rows, extra_ms=5.0 - rank)
    np.save(os.path.join(out_dir, "red_%d.npy" % rank), np.array([ms, extra, tok]))
    dist.destroy_process_group()


def test_two_rank_sharding_and_reduction(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from oracle import mas_ref as O
    from paper_2604_02945_b200 import synth
    w = synth.batched_images(seed=1, R=5, d=64, P=40)
    segs, n = O.make_segments(w.segments)
    whole = O.forward(segs, w.q_off, O.default_params(), w.X, w.Q, want_Y=False)["mas_tok"]
    ranges = [np.load(tmp_path / ("range_%d.npy" % r)) for r in range(world)]
    assert ranges[0][0] == 0 and ranges[0][1] == ranges[1][0] and ranges[1][1] == w.n_requests   # a partition of the requests
    assert 0 < ranges[0][1] < w.n_requests                                                      # both ranks have work
    got = np.concatenate([np.load(tmp_path / ("mas_%d.npy" % r)) for r in range(world)])
    assert got.shape == whole.shape and np.array_equal(got, whole)      # requests are independent: bit-identical
    for r in range(world):
        ms, extra, tok = np.load(tmp_path / ("red_%d.npy" % r))
        assert ms == 11.0 and extra == 5.0 and tok == w.n_tokens


def test_shard_requests_balances_and_covers():
    from paper_2604_02945_b200 import synth
    costs = np.array([5, 1, 1, 1, 8, 2, 2, 4], float)
    for world in (1, 2, 3, 8):
        sh = synth.shard_requests(costs, world)
        assert sh[0][0] == 0 and sh[-1][1] == len(costs)
        assert all(sh[i][1] == sh[i + 1][0] for i in range(world - 1))
    lo, hi = synth.shard_requests(costs, 2)[0]
    assert abs(costs[lo:hi].sum() - costs.sum() / 2) <= costs.max()
