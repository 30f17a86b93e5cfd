"""-m "not gpu": host logic of the slab decomposition (paper_2510_06873_b200/domain.py) — the partition,
that a halo of 2 rc is sufficient (checked with the ORACLE on the sub-systems against the oracle on the whole system), and
the one exchange of a step, an all-reduce of the ncv partial sums, over gloo with world_size 2 on CPU."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle as orc
from oracle.reference import OracleMetaD
from paper_2510_06873_b200 import domain
from paper_2510_06873_b200.inputs import configs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _workload():
    # an elongated GaN-shaped box (19 x 33 x 125 A, 5,760 atoms): crystalline sphere of radius 9 A in random liquid
    return configs.config3(cells=(6, 6, 24), sphere_r=9.0, n_hills=50)


@pytest.mark.parametrize("world", [1, 2, 3, 5])
def test_partition_owns_every_atom_once_and_holds_the_whole_halo(world):
    w = _workload()
    reach = 2.0 * w.rc
    cz = w.box.reshape(3, 3)[2, 2]
    owner_count = np.zeros(w.natoms, dtype=int)
    for rank in range(world):
        local, owned = domain.slab_partition(w.pos, w.box, reach, world, rank)
        assert np.all(np.diff(local) > 0)                                   # ascending: relative order of the atoms kept
        owner_count[local[owned]] += 1
        assert np.array_equal(domain.slab_of(w.pos[local[owned]], w.box, world), np.full(owned.sum(), rank))
        # brute force: an atom is held iff some periodic image of it lies within `reach` of some owned atom's slab ...
        lo, hi = rank * cz / world, (rank + 1) * cz / world
        z = w.pos[:, 2]
        mid, half = 0.5 * (lo + hi), 0.5 * (hi - lo)
        dz = np.abs(z - mid)
        dz = np.minimum(dz, cz - dz)                                        # periodic distance to the slab's mid-plane
        want = np.nonzero((dz - half < reach) | (domain.slab_of(w.pos, w.box, world) == rank))[0]
        assert np.array_equal(local, want)
        f = domain.fill_fraction(w.box, reach, world)
        assert 0 < f <= 1 and (world > 1 or f == 1.0)
        assert len(local) <= np.ceil(1.35 * f * w.natoms) + 64              # the held atoms fill about that fraction
    assert np.all(owner_count == 1)


@pytest.mark.parametrize("world", [2, 3])
def test_halo_of_two_cutoffs_is_sufficient_oracle(world):
    """The oracle on each rank's sub-system (global coordinates, global box) reproduces, for the OWNED atoms, the neighbour
    sets, the per-atom q6 and the CV gradient of the whole system; the owned partial sums add up to the global CV."""
    w = _workload()
    og = OracleMetaD(w)
    og.build_neighbors(w.pos)
    s_glob = og.eval_cv()
    total = 0.0
    for rank in range(world):
        local, owned = domain.slab_partition(w.pos, w.box, 2.0 * w.rc, world, rank)
        sub = domain.sub_workload(w, local)
        assert sub.cvs[0].scale == 1.0 / w.natoms                           # the GLOBAL scale
        o = OracleMetaD(sub)
        o.build_neighbors(sub.pos)
        o.eval_cv()
        gl = local[owned]
        assert np.array_equal(o.count[owned], og.count[gl])
        for a, g in zip(np.nonzero(owned)[0][:200], gl[:200]):              # same neighbours (as global indices)
            assert np.array_equal(local[o.list[a, :o.count[a]]], og.list[g, :og.count[g]])
        assert np.array_equal(o.q6[owned], og.q6[gl])                       # the very same arithmetic
        assert np.abs(o.grads[0][owned] - og.grads[0][gl]).max() <= 1e-13 * np.abs(og.grads[0]).max()
        # a halo of ONE cutoff is not enough for the forces: the gradient of some owned atom changes
        total += sub.cvs[0].scale * float(np.sum(o.q6[owned]))
    assert abs(total - s_glob[0]) <= 1e-13 * abs(s_glob[0])
    local1, owned1 = domain.slab_partition(w.pos, w.box, 1.0 * w.rc, world, 0)
    o1 = OracleMetaD(domain.sub_workload(w, local1))
    o1.build_neighbors(w.pos[local1])
    o1.eval_cv()
    assert np.array_equal(o1.q6[owned1], og.q6[local1[owned1]])             # the CV is already right with one cutoff ...
    assert np.abs(o1.grads[0][owned1] - og.grads[0][local1[owned1]]).max() > 1e-6 * np.abs(og.grads[0]).max()   # ... the forces are not


WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np
import torch
import torch.distributed as dist
from oracle.reference import OracleMetaD
from paper_2510_06873_b200 import domain
from paper_2510_06873_b200.inputs import configs
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["MASTER_PORT"],
                        rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
w = configs.config3(cells=(6, 6, 24), sphere_r=9.0, n_hills=50)         # every rank builds the same seeded system
local, owned = domain.slab_partition(w.pos, w.box, 2.0 * w.rc, world, rank)
sub = domain.sub_workload(w, local)
o = OracleMetaD(sub)
o.build_neighbors(sub.pos)
o.eval_cv()
cv = torch.tensor([sub.cvs[0].scale * float(np.sum(o.q6[owned]))], dtype=torch.float64)     # this rank's partial sum
n_owned = torch.tensor([int(owned.sum())])
dist.all_reduce(cv, op=dist.ReduceOp.SUM)                                # the one exchange of a step
dist.all_reduce(n_owned, op=dist.ReduceOp.SUM)
print(json.dumps({"rank": rank, "cv": float(cv[0]), "n_owned": int(n_owned[0]), "held": int(len(local))}))
dist.destroy_process_group()
""" % ROOT


def test_partial_sums_all_reduce_to_the_global_cv_gloo():
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29621")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    res = [json.loads(o[0].strip().splitlines()[-1]) for o in outs]
    w = _workload()
    og = OracleMetaD(w)
    og.build_neighbors(w.pos)
    s = og.eval_cv()
    assert res[0]["cv"] == res[1]["cv"]                                     # every rank goes on with the same bits
    assert abs(res[0]["cv"] - s[0]) <= 1e-13 * abs(s[0])
    assert res[0]["n_owned"] == w.natoms
    assert all(r["held"] < w.natoms for r in res)                           # a rank holds less than the whole system
