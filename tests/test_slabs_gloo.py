"""Host logic of the y-slab decomposition (paper_2308_16597_b200/slabs.py) on CPU: the row
partition, the ownership rule (the paper's domain lists), and -- with two gloo
ranks -- the force combine as an all-reduce and the hand-over of a particle that crosses the cut.
The device side of the same protocol is tests/test_gpu_slabs.py."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_2308_16597_b200 import slabs


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_partition_covers_the_cavity_once_and_respects_the_halo():
    for ny, n, halo in ((4000, 8, 18), (1000, 3, 18), (257, 5, 20), (100, 1, 40)):
        r = slabs.partition_rows(ny, n, halo)
        assert len(r) == n and r[0][0] == 0 and r[-1][1] == ny
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        assert min(j1 - j0 for j0, j1 in r) >= halo
        assert max(j1 - j0 for j0, j1 in r) - min(j1 - j0 for j0, j1 in r) <= 1
    with pytest.raises(ValueError):
        slabs.partition_rows(100, 4, 30)
    assert slabs.halo_for_diameter(20.0) == 18 and slabs.halo_for_diameter(24.0) == 20
    assert slabs.halo_for_diameter(0.0) == 8


def test_every_centre_has_exactly_one_owner_and_the_cut_itself_goes_up():
    r = slabs.partition_rows(1000, 4, 18)            # cuts at 250, 500, 750
    y = np.array([0.3, 249.999999, 250.0, 250.000001, 499.5, 500.0, 999.4])
    assert slabs.owner_of(y, r).tolist() == [0, 0, 1, 1, 1, 2, 3]
    rng = np.random.default_rng(0)
    yy = rng.uniform(0.0, 1000.0, 100000)
    own = slabs.owner_of(yy, r)
    assert (own >= 0).all()
    for s, (j0, j1) in enumerate(r):
        assert ((yy[own == s] >= j0) & (yy[own == s] < j1)).all()


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ranges = slabs.partition_rows(400, world, 18)     # cut at row 200
    rng = np.random.default_rng(5)                    # same particles on every rank (replicated)
    n = 64
    y = rng.uniform(150.0, 250.0, n)
    y[0], y[1] = 199.9, 200.1                         # one just below, one just above the cut
    F_true = rng.standard_normal((3, n))              # what the owner's complete link sum gives
    res = []
    for step in range(3):
        own = slabs.owner_of(y, ranges)
        # this rank's bounce-back: the complete sum for particles it owns, an incomplete one (here:
        # garbage) for particles it only sees part of; k_slab_forces_out zeroes the latter
        partial = np.where(own[None, :] == rank, F_true, 12345.678 * (rank + 1))
        buf = np.where(own[None, :] == rank, partial, 0.0)
        t = torch.from_numpy(buf.copy())
        dist.all_reduce(t)                            # the force combine
        combined = t.numpy()
        # every rank integrates every particle from the same combined forces: identical states
        y = y - 0.15 + 1e-3 * combined[1]
        res.append((own.copy(), combined.copy(), y.copy()))
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_combine_forces_exactly_and_hand_a_particle_over():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    rng = np.random.default_rng(5)
    rng.uniform(150.0, 250.0, 64)
    F_true = rng.standard_normal((3, 64))
    for step in range(3):
        own0, c0, y0 = res[0][step]
        own1, c1, y1 = res[1][step]
        assert np.array_equal(own0, own1)                       # ownership follows from positions alone
        assert np.array_equal(c0, c1) and np.array_equal(y0, y1)  # replicated states stay identical, bitwise
        assert np.array_equal(c0, F_true)                       # the owner's sum, exactly (x + 0 = x)
    # particle 1 started at 200.1 in the upper slab and falls 0.15 per step: handed to the lower one
    assert res[0][0][0][1] == 1 and res[0][1][0][1] == 0
    # particle 0 stays below the cut; the totals are unchanged by the hand-over
    assert all(res[0][s][0][0] == 0 for s in range(3))
