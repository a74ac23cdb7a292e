"""N > 1 path on CPU: two `gloo` ranks.

The multi-GPU path has no collective inside the step: rank r simulates the global particle ids
r, r + world, ... (lpm_release pid_offset / pid_stride), bins its own particles, and the output grids are
summed with one all_reduce per grid.  What can go wrong is host logic: which ids a rank owns, how
many of them are born by a given step (the C ABI's lpm_schedule_born, usable without a GPU),
bench.py's weak-scaling workload construction, and the reduction.  Here each rank runs the fp64
oracle on its shard; the all-reduced result must equal the unsharded run.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        from oracle import oracle as orc
        import paper_0912_3223_b200 as lpm

        steps = 240
        w = bench.make_workload("c2", 2.0e-3, world, rank)          # 2000 particles per rank, 4000 in the ensemble
        w = w.replace(n_steps=steps, bin_every=120)
        r = w.release
        assert (r.pid_offset, r.pid_stride, r.n_particles) == (rank, world, 4000)

        # host-side schedule of the C ABI vs the oracle's injection, for this rank's ids
        o = orc.OracleSim(w)
        s_start, S = 0, 720
        born_prev = 0
        for n in range(steps):
            o.step(1)
            born = lpm.schedule_born(r.n_particles, rank, world, s_start, S, n)
            assert born == o.n, (rank, n, born, o.n)
            assert born - born_prev == o.injected(n)
            born_prev = born

        cnt = torch.from_numpy(o.counts().astype(np.int64))
        conc = torch.from_numpy(o.concentration().copy())
        led = torch.tensor(o.ledger(), dtype=torch.float64)
        n_local = torch.tensor([o.n], dtype=torch.int64)
        for t in (cnt, conc, led, n_local):
            dist.all_reduce(t)                                       # the one collective per output
        if rank == 0:
            np.savez(os.path.join(out_dir, "reduced.npz"), cnt=cnt.numpy(), conc=conc.numpy(), led=led.numpy(), n=n_local.numpy())
        pids = o.particles()["pid"]
        assert np.all(pids % world == rank)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_shards_reduce_to_the_unsharded_run(tmp_path):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    red = np.load(tmp_path / "reduced.npz")

    import bench
    from oracle import oracle as orc
    w = bench.make_workload("c2", 2.0e-3, world, 0).replace(n_steps=240, bin_every=120)
    w.release.pid_offset, w.release.pid_stride = 0, 1             # the whole ensemble in one process
    w = w.replace(capacity=w.release.n_particles)
    o = orc.OracleSim(w)
    o.step(240)
    assert int(red["n"][0]) == o.n == 1334                         # 4000 over 720 steps: ceil(240*4000/720) born
    np.testing.assert_array_equal(red["cnt"], o.counts().astype(np.int64))
    np.testing.assert_allclose(red["conc"], o.concentration(), rtol=1e-12, atol=0)
    np.testing.assert_allclose(red["led"], np.array(o.ledger()), rtol=1e-12, atol=0)
