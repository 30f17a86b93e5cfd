"""Slab decomposition of the Q6 workloads over several GPUs.

One process per GPU.  Rank r OWNS the atoms whose fractional c-coordinate lies in [r / W, (r + 1) / W) and HOLDS, beside them,
every atom within `reach` = 2 (rc + skin) of that slab (a and b span the x-y plane of the lower-triangular box, so the distance
to a slab face is |dz|).  The held atoms keep their GLOBAL coordinates and the GLOBAL box: every pair a rank sees is computed
with the very arithmetic of the undivided system, so the neighbour sets, per-atom q6 and forces of the owned atoms are those of
the whole system — the rest of the box is simply empty for that rank (`params.fill_fraction` sizes the tiles for it, `params.c_window_lo` says
where the occupied window starts, so that only its tiles are launched).

Per step and rank (all kernels; argument marshalling only here):
    metad_build_neighbors -> metad_eval_cv -> metad_cv_owned_sum          (Q6 CVs summed over the OWNED atoms)
    all-reduce of the ncv doubles over the ranks                          (the one exchange of the step; NCCL)
    metad_bias -> metad_apply_forces -> metad_deposit                     (same s on every rank: identical hills everywhere)
Why 2 (rc + skin): the force on an owned atom k needs the q6 records of its neighbours j (within rc of the slab), and those
need all of j's neighbours (within 2 rc of the slab).  Atoms deeper in the halo have incomplete shells; nothing reads them.

Scope: contexts whose CV dimensions are all Q6 CVs (the headline workloads c3, c4) — the only CVs with a per-atom value in
device memory to sum over the owned atoms.  Ownership is fixed when the object is made (BASELINE.json configs evaluate fixed
positions); an MD caller makes a new one when atoms have crossed a slab face or moved `skin` into the halo margin.
"""
from __future__ import annotations

import copy

import numpy as np


def slab_of(pos, box, world):
    """Owner rank of every atom: floor(W * fractional c-coordinate) (positions in the primary cell)."""
    cz = float(np.asarray(box, dtype=np.float64).reshape(3, 3)[2, 2])
    sc = np.asarray(pos, dtype=np.float64)[:, 2] / cz
    return np.minimum(np.maximum(np.floor(sc * world).astype(np.int64), 0), world - 1)


def slab_partition(pos, box, reach, world, rank):
    """(local, owned): `local` = ascending global indices of the atoms rank `rank` holds (its slab + everything within `reach`
    of it along z, periodic), `owned` = boolean mask over `local`.  Ascending order keeps the relative order of the atoms, and
    with it the in-cell order of the cell sort and the summation order of the forces, as in the undivided system."""
    pos = np.asarray(pos, dtype=np.float64)
    cz = float(np.asarray(box, dtype=np.float64).reshape(3, 3)[2, 2])
    if not (0 <= rank < world):
        raise ValueError("rank outside 0..world-1")
    owner = slab_of(pos, box, world)
    if world == 1:
        return np.arange(len(pos)), np.ones(len(pos), dtype=bool)
    z = pos[:, 2]
    lo, hi = rank * cz / world, (rank + 1) * cz / world
    # distance to the slab [lo, hi) along z over the periodic images z, z + cz, z - cz
    d = np.full(len(pos), np.inf)
    for shift in (0.0, cz, -cz):
        zz = z + shift
        d = np.minimum(d, np.maximum(np.maximum(lo - zz, zz - hi), 0.0))
    held = (d < reach) | (owner == rank)
    local = np.nonzero(held)[0]
    return local, owner[local] == rank


def fill_fraction(box, reach, world):
    """Fraction of the box volume a rank's atoms occupy: (slab + 2 reach) / c_z (a hair more), at most 1."""
    cz = float(np.asarray(box, dtype=np.float64).reshape(3, 3)[2, 2])
    return float(min(1.0, (cz / world + 2.0 * reach) / cz + 2e-9))


def c_window_lo(box, reach, world, rank):
    """Fractional c-coordinate at which the rank's window (slab + halo) starts, in [0, 1)."""
    cz = float(np.asarray(box, dtype=np.float64).reshape(3, 3)[2, 2])
    return float((rank / world - reach / cz - 1e-9) % 1.0)


def sub_workload(w, local):
    """The workload of one rank: the held atoms at their global coordinates in the global box.  The CV descriptors are kept as
    they are (scale = 1 / N of the WHOLE system), so the partial sums of the ranks add up to the global CV."""
    sub = copy.copy(w)
    sub.pos = np.ascontiguousarray(np.asarray(w.pos)[local])
    if getattr(w, "species", None) is not None:
        sub.species = np.asarray(w.species)[local]
    return sub


class SlabMetaD:
    """One rank of the decomposition: a MetaD context on the rank's atoms + the owned-atom mask on the device.

    step() = phase1() -> all-reduce -> phase2(); the two phases are public so that a test can run the ranks of a small world one
    after the other on ONE GPU and add the partial sums itself (no rank's kernels ever wait for another rank's)."""

    def __init__(self, w, world, rank, precision=None, skin=0.0, max_hills=None, **kw):
        import torch
        from .metad import MetaD
        self.world, self.rank = int(world), int(rank)
        self.reach = 2.0 * (w.rc + skin) * 1.001           # a hair more: ownership may be decided on other roundings of z
        self.local, owned = slab_partition(w.pos, w.box, self.reach, world, rank)
        self.owned_local = owned
        self.owned_global = self.local[owned]
        self.sub = sub_workload(w, self.local)
        self.md = MetaD(self.sub, precision=precision, skin=skin, max_hills=max_hills,
                        fill_fraction=fill_fraction(w.box, self.reach, world),
                        c_window_lo=c_window_lo(w.box, self.reach, world, rank), **kw)
        self.torch = torch
        with torch.cuda.stream(self.md.stream):
            self.d_owned = torch.tensor(owned.astype(np.uint8), device="cuda")
        self.md.synchronize()

    def phase1(self, pos):
        """Neighbours, CVs, and the Q6 CVs summed over the owned atoms: md.cv holds this rank's PARTIAL sums."""
        self.md.build_neighbors(pos)
        self.md.eval_cv()
        return self.md.cv_owned_sum(self.d_owned)

    def all_reduce(self):
        import torch.distributed as dist
        if self.world > 1:
            with self.torch.cuda.stream(self.md.stream):
                dist.all_reduce(self.md.cv, op=dist.ReduceOp.SUM)

    def phase2(self, F):
        """With the GLOBAL CVs in md.cv: V, dV/ds, forces of the held atoms added to F (rows of the owned atoms are complete,
        the halo rows are not and belong to other ranks), deposition."""
        self.md.bias()
        self.md.apply_forces(F)
        self.md.deposit()

    def step(self, pos, F):
        self.phase1(pos)
        self.all_reduce()
        self.phase2(F)
