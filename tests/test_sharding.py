"""N > 1 path on CPU: two gloo ranks shard the event stream exactly as bench.py --gpus 2 does.
Checks the host logic (ranges, seeded shards, timing reductions) and that sharding needs no collective:
the oracle run per shard, concatenated, equals the oracle run on the whole batch."""
import hashlib
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2002_11529_b200.sharding import reduce_job, shard_event_range, split_events

N_PER_RANK = 5
CONFIG = 2


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _digest(*arrays):
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def _rank_main(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        import synth
        lo, hi = shard_event_range(rank, world, N_PER_RANK)
        geom, b, p = synth.make_workload(CONFIG, n_events=hi - lo, first_event=lo)
        h, t = oracle.run_batch(b, geom, p)
        # the timing protocol of bench.py: max of the times, sum of the events
        ms, ev = reduce_job(10.0 + 5.0 * rank, b.n_events)
        mine = dict(rank=rank, lo=lo, hi=hi, raw=_digest(b.raw), n_hits=h.n_hits, x=_digest(h.x_at_y0[:h.n_hits]),
                    ids=_digest(h.id[:h.n_hits]), n_trk=t.n_hits.tolist(), qop=_digest(t.qop), chi2=_digest(t.chi2),
                    local_idx=[(t.hit_idx[l]).tolist() for l in range(4)], ms=ms, ev=ev)
        gathered = [None] * world
        dist.all_gather_object(gathered, mine)          # test-only: the product path exchanges nothing
        if rank == 0:
            q.put(gathered)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_shards_equal_whole_batch():
    import oracle
    import synth
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, PORT, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    gathered = q.get()
    for pr in procs:
        pr.join(timeout=120)
        assert pr.exitcode == 0
    assert [g["rank"] for g in gathered] == [0, 1]
    assert [(g["lo"], g["hi"]) for g in gathered] == [(0, N_PER_RANK), (N_PER_RANK, 2 * N_PER_RANK)]
    for g in gathered:
        assert g["ms"] == 15.0 and g["ev"] == 2.0 * N_PER_RANK        # max over ranks, sum over ranks

    geom, whole, p = synth.make_workload(CONFIG, n_events=2 * N_PER_RANK)
    h, t = oracle.run_batch(whole, geom, p)
    ns = geom.n_sectors
    cut_raw = int(whole.bank_offsets[N_PER_RANK * ns])
    assert gathered[0]["raw"] == _digest(whole.raw[:cut_raw])
    assert gathered[1]["raw"] == _digest(whole.raw[cut_raw:])
    cut_h = int(h.hit_offsets[N_PER_RANK * geom.n_groups])
    cut_t = int(whole.velo_offsets[N_PER_RANK])
    assert gathered[0]["n_hits"] == cut_h and gathered[1]["n_hits"] == h.n_hits - cut_h
    assert gathered[0]["x"] == _digest(h.x_at_y0[:cut_h]) and gathered[1]["x"] == _digest(h.x_at_y0[cut_h:h.n_hits])
    assert gathered[0]["ids"] == _digest(h.id[:cut_h]) and gathered[1]["ids"] == _digest(h.id[cut_h:h.n_hits])
    assert gathered[0]["n_trk"] + gathered[1]["n_trk"] == t.n_hits.tolist()
    assert gathered[0]["qop"] == _digest(t.qop[:cut_t]) and gathered[1]["qop"] == _digest(t.qop[cut_t:])
    assert gathered[0]["chi2"] == _digest(t.chi2[:cut_t]) and gathered[1]["chi2"] == _digest(t.chi2[cut_t:])
    # hit indices are shard-local: rank 1's are offset by the hits of rank 0's events
    for l in range(4):
        r1 = np.asarray(gathered[1]["local_idx"][l])
        assert np.array_equal(np.where(r1 >= 0, r1 + cut_h, -1), t.hit_idx[l, cut_t:])
        assert np.array_equal(np.asarray(gathered[0]["local_idx"][l]), t.hit_idx[l, :cut_t])


PORT = _free_port()


def test_ranges_and_splits():
    assert shard_event_range(0, 4, 1000) == (0, 1000) and shard_event_range(3, 4, 1000) == (3000, 4000)
    with pytest.raises(ValueError):
        shard_event_range(4, 4, 10)
    for n in (0, 1, 7, 1000, 1001):
        for w in (1, 2, 3, 8):
            parts = split_events(n, w)
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1


def test_reduce_job_single_process():
    assert reduce_job(3.5, 1000) == (3.5, 1000.0)
