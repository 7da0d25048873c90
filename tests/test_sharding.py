"""The N > 1 path on CPU: two gloo ranks shard the event list, integrate their ranges with the
global event index in the Philox counter, gather, and take the max-over-ranks time.  The compute
stand-in on CPU is the oracle (tests may use it); the sharding and gathering code is the product's."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

import oracle
from paper_1407_7595_b200 import sharding
from paper_1407_7595_b200 import workloads as wl


def test_shard_ranges_partition_the_list():
    for n in (0, 1, 7, 64, 4096, 16385):
        for world in (1, 2, 3, 8):
            r = [sharding.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n_events, n_points, seed, out_path):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, w = sharding.init_process_group("gloo")
    assert (r, w) == (rank, world)
    proc = 1
    ev = wl.make_events(proc, n_events, seed=21)
    lo, hi = sharding.shard_range(n_events, rank, world)
    p = oracle.params_default(proc)
    pl, el = oracle.integrate(proc, p, ev[:, lo:hi], n_points, seed, event_offset=lo)
    full_p = sharding.gather_results(torch.from_numpy(pl), n_events)
    full_e = sharding.gather_results(torch.from_numpy(el), n_events)
    t = sharding.max_over_ranks(1.0 + rank)
    total = sharding.sum_over_ranks(hi - lo)
    if rank == 0:
        np.savez(out_path, p=full_p.numpy(), e=full_e.numpy(), t=t, total=total)
    torch.distributed.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_gloo_sharding_matches_unsharded(tmp_path):
    n_events, n_points, seed, world = 7, 500, 99, 2      # 7 events: unequal shards (4 + 3)
    out = str(tmp_path / "out.npz")
    mp.start_processes(_worker, args=(world, _free_port(), n_events, n_points, seed, out), nprocs=world,
                       join=True, start_method="spawn")
    got = np.load(out)
    ev = wl.make_events(1, n_events, seed=21)
    po, eo = oracle.integrate(1, oracle.params_default(1), ev, n_points, seed)
    assert np.array_equal(got["p"], po) and np.array_equal(got["e"], eo)      # bit for bit
    assert float(got["t"]) == 2.0 and float(got["total"]) == n_events
