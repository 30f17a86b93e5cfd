"""-m gpu: slab decomposition (paper_2510_06873_b200/domain.py, metad_cv_owned_sum) on ONE GPU: the ranks
of a small world run one after the other (no rank's kernels wait for another's), the test adds their partial CV sums in
place of the all-reduce, and the assembled result is compared with the oracle on the WHOLE system and with a single
context holding the whole system."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle.reference import OracleMetaD  # noqa: E402
from paper_2510_06873_b200 import domain  # noqa: E402
from paper_2510_06873_b200.inputs import configs, hill_walk, seeded_heights, wrap  # noqa: E402

from gpu_util import TOL_CV, TOL_F, positions_for, rel  # noqa: E402


def _workload(name):
    if name == "c3":            # 38 x 33 x 156 A, 17,280 atoms, Q6 mean
        return configs.config3(cells=(12, 12, 30), sphere_r=12.0, n_hills=60)
    w = configs.config4(cells=(12, 12, 30), sphere_r=12.0, n_hills=60, grid=(0, 0))       # Q6 mean + solid-like count
    w.cvs[1].q_thresh = 0.25
    return w


def _run_ranks(w, world, precision, pos, hills, skin=0.0, frames=None):
    """All ranks of the world, sequentially; returns per-step (s, V, dVds, F_global) and the rank objects."""
    import torch
    tdt = torch.float32 if precision == 32 else torch.float64
    ranks = [domain.SlabMetaD(w, world, r, precision=precision, skin=skin, max_hills=len(hills[1]) + 16) for r in range(world)]
    for rk in ranks:
        rk.md.set_hills(*hills)
    out = []
    for k in range(1 if frames is None else len(frames)):
        p = pos if frames is None else frames[k].astype(pos.dtype)
        dp, dF = [], []
        for rk in ranks:
            with torch.cuda.stream(rk.md.stream):
                dp.append(torch.tensor(p[rk.local], device="cuda", dtype=tdt))
                dF.append(torch.zeros((len(rk.local), 3), device="cuda", dtype=tdt))
            rk.md.synchronize()
        partial = []
        for rk, x in zip(ranks, dp):
            rk.phase1(x)
            rk.md.synchronize()
            partial.append(rk.md.cv.cpu().numpy().copy())
        total = np.sum(partial, axis=0)                        # stands in for the all-reduce (two or three fp64 terms)
        F = np.zeros((w.natoms, 3))
        V, dV = None, None
        for rk, f in zip(ranks, dF):
            with torch.cuda.stream(rk.md.stream):
                rk.md.cv.copy_(torch.tensor(total, dtype=torch.float64))
            rk.phase2(f)
            rk.md.synchronize()
            Vr, dVr = float(rk.md.V.cpu().numpy().ravel()[0]), rk.md.dVds.cpu().numpy().astype(np.float64)[:w.ncv].copy()
            if V is None:
                V, dV = Vr, dVr
            assert Vr == V and np.array_equal(dVr, dV)                            # every rank computes the same bias
            assert rk.md.status() == 0
            F[rk.owned_global] = f.cpu().numpy().astype(np.float64)[rk.owned_local]
        out.append((total, V, dV, F))
    h0 = ranks[0].md.get_hills()
    for rk in ranks[1:]:                                                          # identical hills on every rank
        h = rk.md.get_hills()
        assert np.array_equal(h[0], h0[0]) and np.array_equal(h[1], h0[1])
    return out, ranks


@pytest.mark.parametrize("name,precision,world", [("c3", 32, 2), ("c3", 32, 3), ("c3", 32, 5), ("c4", 32, 2), ("c3", 64, 2)])
def test_decomposed_step_matches_the_oracle_and_the_single_context(name, precision, world):
    import torch
    from paper_2510_06873_b200.metad import MetaD
    w = _workload(name)
    w.stride = 1
    pos = positions_for(w, precision)
    o = OracleMetaD(w)
    o.build_neighbors(pos.astype(np.float64))
    s_ref = o.eval_cv()
    hills = (hill_walk(4, s_ref, w.sigma, 40), seeded_heights(4, 40, w.w0))
    o.set_hills(*hills)
    (res,), ranks = _run_ranks(w, world, precision, pos, hills)
    s, V, dV, F = res
    assert sum(int(r.owned_local.sum()) for r in ranks) == w.natoms
    assert all(len(r.local) < w.natoms for r in ranks)                            # each rank holds a part only
    # --- against the oracle on the whole system (stage-wise on the CUDA path's own upstream values, reading S)
    assert rel(s, s_ref) <= TOL_CV
    V_ref, dV_ref = o.bias(s)
    assert abs(V - V_ref) <= TOL_CV * abs(V_ref) and np.abs(dV - dV_ref).max() <= TOL_CV * np.abs(dV_ref).max()
    F_ref = o.forces(dV)
    ulp = 2.0 ** -24 * np.abs(F_ref).max() if precision == 32 else 0.0
    assert np.abs(F_ref).max() > 0
    assert np.abs(F - F_ref).max() <= TOL_F * np.abs(F_ref).max() + ulp
    # --- against ONE context holding everything
    md = MetaD(w, precision=precision, max_hills=64)
    md.set_hills(*hills)
    tdt = torch.float32 if precision == 32 else torch.float64
    with torch.cuda.stream(md.stream):
        dp = torch.tensor(pos, device="cuda", dtype=tdt)
        dF = torch.zeros((w.natoms, 3), device="cuda", dtype=tdt)
    md.synchronize()
    md.build_neighbors(dp)
    md.eval_cv()
    md.synchronize()
    tight = 1e-7 if precision == 32 else 1e-12
    assert rel(s, md.cv.cpu().numpy()) <= tight                # the same per-atom q6, summed in another order
    with torch.cuda.stream(md.stream):
        md.cv.copy_(torch.tensor(s, dtype=torch.float64))      # the same s, hence the same dV/ds bits (dV/ds amplifies a
    md.bias()                                                  # difference in s by s / sigma: DESIGN.md reading S)
    md.apply_forces(dF)
    md.synchronize()
    assert np.array_equal(md.dVds.cpu().numpy()[:w.ncv], dV)
    F1 = dF.cpu().numpy().astype(np.float64)
    # fp64: the same arithmetic in another summation order.  fp32: the tile-local coordinates of a periodic image are rounded
    # once, relative to the tile's origin, and the two contexts tile the box differently — a difference of an fp32 ulp of a
    # coordinate (4e-6 A at 38 A), which the Y6m gradient amplifies to a few 1e-6 max|F|: the force bar itself is the bound
    assert np.abs(F - F1).max() <= (TOL_F if precision == 32 else 1e-11) * np.abs(F1).max()
    # the deposited hill: same centre bits on every rank, = the summed CV
    c, h = ranks[0].md.get_hills()
    assert len(h) == 41 and np.array_equal(c[-1], s)


def test_decomposed_steps_with_a_verlet_skin_and_moving_atoms():
    """Three steps of moving atoms with params.skin on every rank (the halo reaches 2 (rc + skin)); ownership stays as
    partitioned at step 0 — every step against the oracle on the whole system."""
    w = _workload("c3")
    w.stride = 2
    pos = positions_for(w, 32)
    rng = np.random.default_rng(12)
    frames, p = [], pos.astype(np.float64)
    for k in range(3):
        if k:
            p = wrap(p + rng.standard_normal(p.shape) * 0.012, w.box)
        frames.append(p.astype(np.float32))
    o = OracleMetaD(w)
    o.build_neighbors(frames[0].astype(np.float64))
    hills = (hill_walk(4, o.eval_cv(), w.sigma, 30), seeded_heights(4, 30, w.w0))
    res, ranks = _run_ranks(w, 2, 32, pos, hills, skin=0.3, frames=frames)
    of = OracleMetaD(w)
    of.set_hills(*hills)
    for k, (s, V, dV, F) in enumerate(res):
        of.build_neighbors(frames[k].astype(np.float64))
        s_ref = of.eval_cv()
        assert rel(s, s_ref) <= TOL_CV
        V_ref, dV_ref = of.bias(s)
        assert abs(V - V_ref) <= TOL_CV * abs(V_ref)
        F_ref = of.forces(dV)
        assert np.abs(F - F_ref).max() <= TOL_F * np.abs(F_ref).max() + 2.0 ** -24 * np.abs(F_ref).max()
        of.deposit(s, V)
    assert all(r.md.rebuilds() == 1 for r in ranks)


def test_owned_sum_rejects_contexts_without_per_atom_values():
    import torch
    from paper_2510_06873_b200 import metad
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = configs.small("c2")                                     # coordination number: no per-atom array to sum
    md = MetaD(w)
    with torch.cuda.stream(md.stream):
        dp = torch.tensor(w.pos, device="cuda")
        ow = torch.ones(w.natoms, device="cuda", dtype=torch.uint8)
    md.synchronize()
    md.build_neighbors(dp)
    md.eval_cv()
    with pytest.raises(MetadError) as e:
        md.cv_owned_sum(ow)
    assert e.value.code == metad.ERR_STATE


def test_an_atom_outside_the_window_of_the_rank_is_flagged():
    """Only the tiles of the rank's window [c_window_lo, c_window_lo + fill_fraction) are launched: an atom that has left it
    would silently get no neighbours, so the binning raises METAD_DEV_POS_RANGE."""
    import torch
    from paper_2510_06873_b200 import metad
    w = _workload("c3")
    rk = domain.SlabMetaD(w, 4, 1, precision=32, max_hills=8)
    p = w.pos[rk.local].astype(np.float32)
    with torch.cuda.stream(rk.md.stream):
        dp = torch.tensor(p, device="cuda")
    rk.md.synchronize()
    rk.phase1(dp)
    assert rk.md.status() == 0
    cz = w.box.reshape(3, 3)[2, 2]
    p[7, 2] = np.float32((p[7, 2] + 0.5 * cz) % cz)            # half a box away along c: outside the window of rank 1 of 4
    with torch.cuda.stream(rk.md.stream):
        dp.copy_(torch.tensor(p))
    rk.phase1(dp)
    assert rk.md.status() & metad.DEV_POS_RANGE
