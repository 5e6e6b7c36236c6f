"""The N > 1 path of bench.py on CPU: world_size 2, gloo.  The hot path shards over INDEPENDENT
systems (one seeded system per rank, no data-path collective); what the ranks
share is the max-over-ranks reduction of the timed totals and the whole-job aggregation."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from conftest import ROOT

if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench

    class Args:
        config, n = 4, 1536
    assert bench.dist_env() == (rank, rank, world)
    w = bench.make_workload(Args, rank)
    # every rank its own system of the same shape
    my_ms = [10.0 + 5.0 * rank, 20.0 - 3.0 * rank]
    tmax = bench.max_over_ranks(torch, dist, my_ms, "cpu")
    pairs = w.N * (w.N - 1.0)
    rate = bench.whole_job_rate(world, pairs, 7, tmax[0])
    # exchange a fingerprint of the state to prove the systems differ (test-only collective)
    fp = torch.tensor([float(w.N), float(w.x[:, 0].sum()), float(w.m.sum())], dtype=torch.float64)
    allfp = [torch.zeros_like(fp) for _ in range(world)]
    dist.all_gather(allfp, fp)
    np.save(os.path.join(out_dir, f"r{rank}.npy"),
            np.array([tmax[0], tmax[1], rate] + [float(v) for t in allfp for v in t.tolist()]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_independent_systems_and_max_time(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = (np.load(tmp_path / f"r{k}.npy") for k in range(world))
    assert np.array_equal(r0, r1)                       # both ranks agree on the reduction
    assert r0[0] == 15.0 and r0[1] == 20.0              # element-wise max over ranks
    n = 1536
    assert np.isclose(r0[2], 2 * n * (n - 1.0) * 7 / 15.0e-3)
    f0, f1 = r0[3:6], r0[6:9]
    assert f0[0] == f1[0] == n                          # same shape ...
    assert f0[1] != f1[1]                               # ... different (independently seeded) bodies
    assert np.isclose(f0[2], f1[2])                     # same total mass


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(torch, None, [1.5, 2.5], "cpu") == [1.5, 2.5]
    assert bench.whole_job_rate(1, 10.0, 4, 2.0) == 10.0 * 4 / 2.0e-3
