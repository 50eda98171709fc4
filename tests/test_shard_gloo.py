"""The N > 1 path on CPU: two gloo ranks shard the events, run their part (here: the oracle stands in for the device
work, the sharding logic is the same) and all-gather the counters that define the global offsets."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_events, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import gen
    from gen import constants as C
    from oracle import ds_oracle as O
    from paper_2503_13092_b200 import shard
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        lo, hi = shard.event_range(rank, world, n_events)
        d = gen.generate(1, n_events=n_events)
        ho, so = d["hit_offsets"], d["seed_offsets"]
        hits = {k: v[ho[lo]:ho[hi]] for k, v in d["hits"].items()}
        seeds = {k: v[so[lo]:so[hi]] for k, v in d["seeds"].items()}
        mlp = O.Mlp(gen.mlp_weights(0))
        r = O.reconstruct(hits, ho[lo:hi + 1] - ho[lo], seeds, so[lo:hi + 1] - so[lo], C.GEOMETRY, C.PARAMS, mlp, n_threads=1)
        v = O.vertex(r, so[lo:hi + 1] - so[lo], C.GEOMETRY, C.PARAMS, n_threads=1)
        counts, offs = shard.gather_counts(hi - lo, int(r["found"].sum()), v["n"])
        tmax = shard.max_over_ranks(1.0 + rank)
        tsum = shard.sum_over_ranks(hi - lo)
        q.put((rank, lo, hi, counts, offs, tmax, tsum, int(r["found"].sum()), v["n"], (v["ia"] + so[lo]).tolist()))
    finally:
        dist.destroy_process_group()


def test_event_range_partitions():
    from paper_2503_13092_b200 import shard
    for n in (0, 1, 7, 10, 100000):
        for w in (1, 2, 3, 8):
            r = [shard.event_range(k, w, n) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n and all(a[1] == b[0] for a, b in zip(r, r[1:]))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1
    assert shard.block_range(3, 100) == (300, 400)
    assert shard.gather_counts(5, 4, 3) == ([[5, 4, 3]], [0, 0, 0]) and shard.max_over_ranks(2.5) == 2.5
    with pytest.raises(ValueError):
        shard.event_range(2, 2, 10)


def test_two_gloo_ranks_shard_events_and_gather_counts():
    import gen
    from gen import constants as C
    from oracle import ds_oracle as O
    n_events, world = 9, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_events, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # the union of the shards equals the single-process result
    d = gen.generate(1, n_events=n_events)
    mlp = O.Mlp(gen.mlp_weights(0))
    r = O.reconstruct(d["hits"], d["hit_offsets"], d["seeds"], d["seed_offsets"], C.GEOMETRY, C.PARAMS, mlp)
    v = O.vertex(r, d["seed_offsets"], C.GEOMETRY, C.PARAMS)
    (r0, r1) = res
    assert (r0[1], r0[2], r1[1], r1[2]) == (0, 5, 5, 9)
    assert r0[3] == r1[3] == [[5, r0[7], r0[8]], [4, r1[7], r1[8]]]
    assert r0[4] == [0, 0, 0] and r1[4] == [5, r0[7], r0[8]]
    assert r0[7] + r1[7] == int(r["found"].sum()) and r0[8] + r1[8] == v["n"]
    assert r0[9] + r1[9] == v["ia"].tolist()
    assert r0[5] == r1[5] == 2.0 and r0[6] == r1[6] == 9.0
