"""The N > 1 path of bench.py on CPU: two gloo ranks, each takes its own event range of the seeded stream
(paper_2407_12119_b200.sharding.rank_events), and the per-rank timings / counts are reduced to whole-job numbers
(whole_job) exactly as bench.py does it over NCCL.  Events are independent in every stage, so
there is no data-path collective to test (replicas only)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import datagen
from paper_2407_12119_b200.sharding import rank_events, whole_job


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, per_gpu, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = datagen.get_config("cfg1")
    first, n = rank_events(rank, world, per_gpu)
    b = datagen.generate_batch(cfg, n_events=n, first_event=first)
    # the rank's "timed region": rank 1 is the slow one; the whole-job time must be its time, the counts the sums
    ms = 10.0 + 5.0 * rank
    ms_all, (ev, hits) = whole_job(ms, [b.n_events, b.n_hits], dist)
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), xyz=b.xyz, plane=b.plane, off=b.event_offsets,
             ms=ms_all, ev=ev, hits=hits, first=first)
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_take_disjoint_event_ranges_and_reduce_like_bench(tmp_path):
    world, per_gpu = 2, 3
    mp.spawn(_worker, args=(world, _free_port(), per_gpu, str(tmp_path)), nprocs=world, join=True)
    cfg = datagen.get_config("cfg1")
    whole = datagen.generate_batch(cfg, n_events=world * per_gpu)          # the same stream in one process
    r = [np.load(tmp_path / f"r{k}.npz") for k in range(world)]
    lo = 0
    for k in range(world):
        assert int(r[k]["first"]) == k * per_gpu
        n_hits = int(r[k]["off"][-1])
        h0 = int(whole.event_offsets[k * per_gpu])
        assert np.array_equal(r[k]["xyz"], whole.xyz[h0:h0 + n_hits])      # rank k's events are events k*B .. k*B+B-1
        assert np.array_equal(r[k]["plane"], whole.plane[h0:h0 + n_hits])
        assert np.array_equal(r[k]["off"], whole.event_offsets[k * per_gpu:(k + 1) * per_gpu + 1] - h0)
        lo += n_hits
    assert lo == whole.n_hits                                              # disjoint and complete
    for k in range(world):                                                 # every rank holds the same whole-job numbers
        assert float(r[k]["ms"]) == 15.0                                   # max over ranks
        assert float(r[k]["ev"]) == world * per_gpu and float(r[k]["hits"]) == whole.n_hits


def test_rank_events_and_single_process_whole_job():
    assert rank_events(0, 1, 500) == (0, 500)
    assert [rank_events(k, 4, 7) for k in range(4)] == [(0, 7), (7, 7), (14, 7), (21, 7)]
    with pytest.raises(ValueError):
        rank_events(2, 2, 5)
    assert whole_job(3.5, [1, 2, 3]) == (3.5, [1.0, 2.0, 3.0])
    assert whole_job(3.5, []) == (3.5, [])
