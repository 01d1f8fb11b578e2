"""y-slab domain decomposition: host-side
orchestration of the slab calls of include/lbm.h.  No arithmetic of the method lives here: the
module only decides row ranges, calls the two halves of a step on every slab and moves the two
exchanges (force combine, halo rows) between them.

* `partition_rows`, `owner_of`: the row ranges of a decomposition and the slab that owns a particle
  (the one whose own rows hold its centre: the paper's domain list).
* `SlabGroup`: all slabs in ONE process (several slabs on one GPU in the tests; the GPUs of one
  node under one process): the library's own same-process exchanges.
* `SlabRank`: one slab per torch.distributed rank (torchrun, NCCL over NVLink): forces by
  all-reduce, halo rows by send / recv of packed buffers with the two neighbours.

BASELINE.json's north_star keeps the measured path on one GPU ("no sharding or collectives across
GPUs"); bench.py therefore runs replicas under torchrun unless `--slabs` is given.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

import numpy as np


def halo_for_diameter(d_max: float) -> int:
    """Ghost rows a decomposition needs for particles up to d_max (lbm_add_particles checks
    d/2 + 8: the particle, its link stencils and the refill stencils of its newborn nodes)."""
    return max(4, int(math.ceil(0.5 * d_max + 8.0)))


def partition_rows(ny: int, n_slabs: int, halo: int) -> List[Tuple[int, int]]:
    """Own row ranges [j0, j1) of n_slabs slabs of a cavity ny rows high: as even as integers
    allow, ascending, every slab at least `halo` rows high (a neighbour's ghost rows are filled
    from ONE slab)."""
    if n_slabs < 1 or ny < n_slabs * max(halo, 1):
        raise ValueError(f"cannot cut {ny} rows into {n_slabs} slabs of at least {halo} rows")
    cuts = [(ny * k) // n_slabs for k in range(n_slabs + 1)]
    return [(cuts[k], cuts[k + 1]) for k in range(n_slabs)]


def owner_of(y: np.ndarray, ranges: Sequence[Tuple[int, int]]) -> np.ndarray:
    """Index of the slab whose own rows hold each centre: j0 <= y < j1 (the rule
    k_slab_forces_out applies on the device).  Every centre inside the cavity has exactly one."""
    y = np.asarray(y, dtype=np.float64)
    own = np.full(y.shape, -1, dtype=np.int64)
    for s, (j0, j1) in enumerate(ranges):
        own[(y >= float(j0)) & (y < float(j1))] = s
    return own


def combine_owned(contributions: Sequence[np.ndarray]) -> np.ndarray:
    """What the force combine computes: the element-wise sum of the slabs' buffers in ascending
    slab order.  Each entry is non-zero in at most one of them, so the sum is that value exactly."""
    total = np.array(contributions[0], dtype=np.float64, copy=True)
    for c in contributions[1:]:
        total = total + np.asarray(c, dtype=np.float64)
    return total


def _slice_rows(T, rows):
    return None if T is None else np.ascontiguousarray(np.asarray(T)[rows[0]:rows[1], :])


class SlabGroup:
    """A cavity cut into y-slabs that all live in this process."""

    def __init__(self, w, n_slabs, halo=None, devices=None, fused_halo=True):
        """fused_halo: the lattice kernel pushes the rows next to a cut into the neighbour's ghost
        rows itself (lbm_slab_link_peers); False: copy-based lbm_slab_exchange_halos after the step."""
        from . import binding
        self.w = w
        d_max = float(np.max(w.particles["diam"])) if w.particles is not None else 0.0
        self.halo = int(halo) if halo is not None else halo_for_diameter(d_max)
        self.ranges = partition_rows(w.ny, n_slabs, self.halo)
        devices = list(devices) if devices is not None else ["cuda:0"] * n_slabs
        self.slabs = []
        for (j0, j1), dev in zip(self.ranges, devices):
            s = binding.Simulation(w.nx, w.ny, w.params, device=dev, slab=(j0, j1, self.halo))
            if w.T_init is not None:
                s.set_temperature(_slice_rows(w.T_init, s.rows_stored))
            if w.particles is not None:
                s.add_particles(**w.particles)       # every slab holds every particle
            self.slabs.append(s)
        self._L = binding.load_library()
        import ctypes as C
        self._arr = (C.c_void_p * n_slabs)(*[s._h for s in self.slabs])
        self._n = n_slabs
        self.fused_halo = bool(fused_halo)
        if self.fused_halo:
            self._chk(self._L.lbm_slab_link_peers(self._arr, self._n))

    def _chk(self, rc, who=0):
        self.slabs[who]._chk(rc)

    def step(self, nsteps=1):
        for _ in range(int(nsteps)):
            for s in self.slabs:
                s.slab_forces()
            self._chk(self._L.lbm_slab_combine_forces(self._arr, self._n))
            for s in self.slabs:
                s.slab_advance()
            if self.fused_halo:
                self._chk(self._L.lbm_slab_fence(self._arr, self._n))
            else:
                self._chk(self._L.lbm_slab_exchange_halos(self._arr, self._n))
        for s in self.slabs:
            s.slab_check()

    def fields(self, populations=False):
        parts = [s.fields(populations=populations) for s in self.slabs]
        out = {k: np.concatenate([p[k] for p in parts], axis=0) for k in ("rho", "ux", "uy", "T", "flag")}
        if populations:
            out["f"] = np.concatenate([p["f"] for p in parts], axis=1)
            out["g"] = np.concatenate([p["g"] for p in parts], axis=1)
        return out

    def particles(self, slab=0):
        return self.slabs[slab].particles()

    def close(self):
        for s in self.slabs:
            s.close()


class SlabRank:
    """This rank's slab of a cavity cut into world_size y-slabs (rank r owns the r-th range)."""

    def __init__(self, w, rank, world, device, halo=None):
        import torch
        from . import binding
        self.torch, self.rank, self.world = torch, rank, world
        d_max = float(np.max(w.particles["diam"])) if w.particles is not None else 0.0
        self.halo = int(halo) if halo is not None else halo_for_diameter(d_max)
        self.ranges = partition_rows(w.ny, world, self.halo)
        j0, j1 = self.ranges[rank]
        self.sim = binding.Simulation(w.nx, w.ny, w.params, device=device, slab=(j0, j1, self.halo))
        if w.T_init is not None:
            self.sim.set_temperature(_slice_rows(w.T_init, self.sim.rows_stored))
        if w.particles is not None:
            self.sim.add_particles(**w.particles)
        n = self.sim.slab_halo_doubles()
        mk = lambda: torch.empty(n, dtype=torch.float64, device=device)
        self.send = {0: mk() if rank > 0 else None, 1: mk() if rank < world - 1 else None}
        self.recv = {0: mk() if rank > 0 else None, 1: mk() if rank < world - 1 else None}
        self.has_particles = w.particles is not None

    def step(self, nsteps=1):
        import torch.distributed as dist
        sim = self.sim
        for _ in range(int(nsteps)):
            sim.slab_forces()
            if self.has_particles and self.world > 1:
                dist.all_reduce(sim.slab_force_tensor())   # one non-zero term per entry: exact
            sim.slab_advance()
            ops = []
            for side, peer in ((0, self.rank - 1), (1, self.rank + 1)):
                if self.send[side] is None:
                    continue
                sim.slab_pack(side, self.send[side])
                ops.append(dist.P2POp(dist.isend, self.send[side], peer))
                ops.append(dist.P2POp(dist.irecv, self.recv[side], peer))
            if ops:
                for r in dist.batch_isend_irecv(ops):
                    r.wait()
                for side in (0, 1):
                    if self.recv[side] is not None:
                        sim.slab_unpack(side, self.recv[side])
        sim.slab_check()

    def close(self):
        self.sim.close()
