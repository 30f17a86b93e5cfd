"""-m gpu: the fp64 shared-memory tiled build (csrc/tiled64.cu: neighbour list fused with Q6 pass 1 in fp64 pair math) against
the oracle and against the generic fp64 kernels it replaces.  A context takes the tiled fp64 path when its neighbour-list CVs
are Q6 CVs only, max_neigh <= 32, no skin and the cell grid has >= 3 cells per direction; max_neigh = 33 keeps the same
workload on the generic kernels (k_build_list<double>, k_q6_pass1<double>), which is how both are compared here.  The captured
step graph tells the two apart: the tiled step has one kernel node less (no separate Q6 pass 1)."""
import copy

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import CVSpec, Workload, configs, wrap  # noqa: E402

from gpu_util import assert_stagewise, chained_run, positions_for, rel, sorted_rows_fast, stagewise  # noqa: E402


def _kernel_nodes(w, precision=64):
    import torch
    from paper_2510_06873_b200.metad import MetaD
    md = MetaD(w, precision=precision)
    dt = torch.float32 if precision == 32 else torch.float64
    with torch.cuda.stream(md.stream):
        dpos = torch.tensor(positions_for(w, precision), device="cuda", dtype=dt)
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=dt)
    md.synchronize()
    md.run(dpos, F, 1)
    md.synchronize()
    gi = md.graph_info()
    assert gi["nodes"] == gi["kernel"]
    md.close()
    return gi["kernel"]


@pytest.mark.parametrize("name", ["c3", "c4"])
def test_tiled_fp64_stagewise_against_the_oracle_and_the_generic_kernels(name):
    w = configs.small(name)
    assert w.max_neigh <= 32
    r = stagewise(w, precision=64)
    assert_stagewise(r, tol_cv=1e-12, tol_f=1e-11)            # fp64 pair math: far inside the north_star bars
    assert np.abs(r["q6"] - r["q6_ref"]).max() <= 1e-12
    wg = copy.deepcopy(w)
    wg.max_neigh = 33                                          # > 32: the generic fp64 kernels
    g = stagewise(wg, precision=64)
    assert_stagewise(g, tol_cv=1e-12, tol_f=1e-11)
    # the two CUDA paths against one another: same sets, sums in a different order
    assert np.array_equal(r["cnt"], g["cnt"])
    assert np.array_equal(sorted_rows_fast(r["cnt"], r["lst"]), sorted_rows_fast(g["cnt"], g["lst"][:, :r["lst"].shape[1]]))
    assert rel(r["s"], g["s"]) <= 1e-13
    assert np.abs(r["F"] - g["F"]).max() <= 1e-12 * np.abs(g["F"]).max()
    assert np.abs(r["q6"] - g["q6"]).max() <= 1e-13
    # and they ARE two paths: the tiled step has no separate Q6 pass 1
    assert _kernel_nodes(wg) == _kernel_nodes(w) + 1


@pytest.mark.parametrize("boxname", ["cubic3cells", "cubic4", "hex120", "hex60", "triclinic"])
def test_tiled_fp64_neighbor_sets_bit_exact_with_pairs_inside_the_recheck_band(boxname):
    """Planted partners at rc (1 +- eps) with eps from 2e-7 down to a few ulp: the fast fp64 test settles the far ones, the
    pairs within the 1e-9 band of rc^2 are re-decided with the canonical predicate of reading O, and every set equals the
    brute-force oracle's.  Boxes with exactly 3 cells per side reach every neighbouring cell through a periodic image."""
    import oracle
    import torch
    from paper_2510_06873_b200.metad import MetaD
    boxes = {
        "cubic3cells": (np.array([10.0, 0, 0, 0, 10.0, 0, 0, 0, 10.0]), 3.2),
        "cubic4": (np.array([14.5, 0, 0, 0, 13.0, 0, 0, 0, 16.1]), 3.2),
        "hex120": (np.array([24.0, 0, 0, -12.0, 12.0 * np.sqrt(3.0), 0, 0, 0, 19.0]), 4.0),
        "hex60": (np.array([24.0, 0, 0, 12.0, 12.0 * np.sqrt(3.0), 0, 0, 0, 19.0]), 4.0),
        "triclinic": (np.array([21.0, 0, 0, 5.0, 20.0, 0, -4.5, 7.0, 23.0]), 3.5),
    }
    box, rc = boxes[boxname]
    rng = np.random.default_rng(23)
    vol = box[0] * box[4] * box[8]
    n = max(int(10.0 / (4.19 * rc ** 3) * vol), 64)                  # about 10 neighbours per atom: max_neigh = 32 holds them
    pos = wrap(rng.random((n, 3)) @ box.reshape(3, 3), box)
    eps = [4e-7, 4e-10, 4e-13, 2e-15]
    for k in range(0, 2 * (n // 8), 2):
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        pos[k + 1] = pos[k] + u * rc * (1.0 + (rng.random() - 0.5) * eps[(k // 2) % len(eps)])
    pos = wrap(pos, box)
    w = Workload(name=boxname, pos=pos, box=box, rc=rc, max_neigh=32, cvs=[CVSpec(kind=1, r0=1.0, scale=1.0 / n)],
                 sigma=[0.1], n_hills=4, precision=64)
    cref, lref, mx = oracle.neighbors(pos, box, rc, 32, "brute")
    assert mx <= 32
    md = MetaD(w, precision=64)
    dpos = torch.tensor(pos, device="cuda")
    torch.cuda.synchronize()
    md.build_neighbors(dpos)
    cnt, lst = md.neighbors()
    assert md.status() == 0
    assert np.array_equal(cnt, cref)
    assert np.array_equal(sorted_rows_fast(cnt, lst), sorted_rows_fast(cref, lref))
    md.close()
    assert _kernel_nodes(w) == 8          # five sort kernels, k_tile_build64, hill sum (+ deposit), forces: the tiled path did run


def test_tiled_fp64_run_path_step_by_step():
    """metad_run on the tiled fp64 path (the last block of k_tile_build64 hands the CVs over, deposition in k_bias_sum), every
    step against the oracle fed with the CUDA path's own upstream values (reading S)."""
    w = configs.small("c4")
    w.stride = 2
    run = chained_run(w, precision=64, nsteps=7)
    assert run["states"][-1]["step"] == 7
    gi = run["md"].graph_info()
    assert gi["nodes"] == gi["kernel"] and gi["memcpy"] == 0


@pytest.mark.parametrize("rc_over_a,overflow", [(1.9, False), (2.3, True)])
def test_tiled_fp64_dense_blob_unstaged_tiles_and_overflow(rc_over_a, overflow):
    """A dense lattice blob in a thin gas: the tiles are sized for the AVERAGE density, so the tiles over the blob hold more
    halo atoms than the staging area (the unstaged path: positions from global memory) and more own atoms than threads
    (several rounds).  rc = 1.9 a: 26 neighbours, every set equals the oracle's.  rc = 2.3 a: 56 neighbours > max_neigh = 32:
    the sticky overflow bit is raised, the count is clamped and the entries kept are true neighbours."""
    import oracle
    import torch
    from paper_2510_06873_b200.metad import MetaD
    a = 2.0
    rc = rc_over_a * a
    box = np.array([60.0, 0, 0, 0, 60.0, 0, 0, 0, 60.0])
    rng = np.random.default_rng(11)
    gx, gy, gz = np.meshgrid(np.arange(18), np.arange(12), np.arange(12), indexing="ij")
    blob = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1) * a + np.array([11.3, 17.1, 20.7])
    blob = blob + 0.02 * rng.standard_normal(blob.shape)
    gas = rng.random((300, 3)) * 60.0
    gas = gas[np.all((gas < np.array([10.0, 16.0, 19.5])) | (gas > np.array([48.5, 42.5, 46.0])), axis=1)]   # clear of the blob
    pos = wrap(np.concatenate([blob, gas]), box)
    pos = pos[rng.permutation(len(pos))]
    n = len(pos)
    w = Workload(name="blob", pos=pos, box=box, rc=rc, max_neigh=32, cvs=[CVSpec(kind=1, r0=1.0, scale=1.0 / n)],
                 sigma=[0.1], n_hills=4, precision=64)
    cref, lref, mx = oracle.neighbors(pos, box, rc, 80, "cells")
    assert (mx > 32) == overflow
    md = MetaD(w, precision=64)
    dpos = torch.tensor(pos, device="cuda")
    torch.cuda.synchronize()
    md.build_neighbors(dpos)
    cnt, lst = md.neighbors()
    bits = md.status()
    assert np.array_equal(cnt, np.minimum(cref, 32))
    assert (bits & 1) == (1 if overflow else 0)                       # METAD_DEV_NEIGH_OVERFLOW
    ok = cref <= 32
    assert np.array_equal(sorted_rows_fast(cnt[ok], lst[ok]), sorted_rows_fast(cref[ok], lref[ok][:, :32]))
    for i in np.nonzero(~ok)[0][:200]:
        assert set(lst[i, :32]) <= set(lref[i, :cref[i]])
    md.close()
    wg = Workload(name="blob", pos=pos, box=box, rc=rc, max_neigh=33, cvs=w.cvs, sigma=[0.1], n_hills=4, precision=64)
    assert _kernel_nodes(w) == _kernel_nodes(wg) - 1                  # the tiled path did run


def test_tiled_fp64_device_resident_box_changing_every_step():
    """NEXT-3 on the tiled fp64 path: the box lives in device memory and is rescaled every step (metad_run_dev: one capture, no
    update); k_tile_build64 takes the lattice rows of its periodic images and of the recheck from the device geometry.  Every step
    against the oracle."""
    w = configs.small("c4")
    w.stride = 2
    frac = np.linalg.solve(w.box.reshape(3, 3).T, w.pos.T).T
    box0 = w.box.copy()
    scales = [1.0, 1.003, 0.99, 1.012, 1.02, 0.985, 1.0]
    r = chained_run(w, precision=64, nsteps=len(scales), device_box=True, box_slack=0.03,
                    box_of_step=lambda k: box0 * scales[k], pos_of_step=lambda k: frac @ (box0 * scales[k]).reshape(3, 3),
                    check_neighbors=True)
    gi = r["md"].graph_info()
    assert gi["captures"] == 1 and gi["updates"] == 0
    assert gi["nodes"] == gi["kernel"] == 9          # k_geom_update + five sort kernels + k_tile_build64 + hill sum + forces
    assert r["md"].status() == 0


@pytest.mark.parametrize("name", ["c3", "c4"])
def test_tiled_fp64_virial(name):
    """Bias virial of the Q6 CVs with the list and the records written by k_tile_build64 (k_q6_force<double, VIRIAL>) against the
    oracle's strain derivatives (reading AD) at the fp64 bar of tests/test_gpu_virial.py."""
    w = configs.small(name)
    r = stagewise(w, precision=64, want_virial=True)
    assert_stagewise(r, tol_cv=1e-12, tol_f=1e-11)
    W = r["md"].virial()
    W_ref = r["o"].virial(r["dV_ref"])
    assert np.abs(W_ref).max() > 0
    assert np.abs(W - W_ref).max() <= 1e-9 * np.abs(W_ref).max(), (W, W_ref)
    if name == "c3":
        assert abs(np.trace(W)) <= 1e-9 * np.abs(W).max()      # Q6 is scale-invariant: traceless virial
