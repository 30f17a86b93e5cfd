"""-m gpu: CUDA path (through the C ABI) against the oracle, element by element, on seeded inputs.
Tolerances are BASELINE.json north_star's: bit-exact neighbour sets, CV / V / dVds 1e-6 relative,
forces 1e-5 * max|F| absolute (stage-wise, reading S)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import CVSpec, Workload, configs, hill_walk, wrap  # noqa: E402

from gpu_util import (TOL_CV, TOL_F, assert_stagewise, chained_run, force_bound, make_hills, positions_for, rel,  # noqa: E402
                      sorted_rows_fast, stagewise)


def _small(name):
    if name == "c0":
        return configs.config0()
    if name == "c0'":
        return configs.config0(shifted=True)
    return configs.small(name)


@pytest.mark.parametrize("name", ["c0", "c0'", "c1", "c2", "c3", "c4"])
def test_stagewise_parity_small(name):
    w = _small(name)
    r = stagewise(w)
    assert_stagewise(r)
    if "q6" in r:
        tol = 2e-6 if w.precision == 32 else 1e-12
        assert np.abs(r["q6"] - r["q6_ref"]).max() <= tol


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("n,m", [(6, 10), (5, 9)])
def test_grouped_coordination_general_exponents(precision, n, m):
    """m != 2n takes the general branch of the switching function (reading A) on the generic (grouped, warp-per-atom) kernels;
    in fp32 pair math it has to stay accurate for pairs near r0, where (1 - x^n) / (1 - x^m) is 0 / 0."""
    w = _small("c2")
    w.cvs[0].n, w.cvs[0].m = n, m
    r = stagewise(w, precision=precision)
    assert_stagewise(r)
    assert np.abs(r["F_ref"]).max() > 0


def test_c3_fp32_pair_math_meets_the_same_tolerances():
    w = _small("c3")
    r = stagewise(w, precision=32)
    assert_stagewise(r)
    assert np.abs(r["q6"] - r["q6_ref"]).max() <= 2e-6


@pytest.mark.parametrize("prec,kind", [(64, 0), (32, 0), (32, 1)])      # (32, Q6) takes the shared-memory tiled path
@pytest.mark.parametrize("boxname", ["cubic3cells", "cubic3dense", "two_cells", "hex120", "hex60", "triclinic"])
def test_neighbor_sets_bit_exact_on_awkward_boxes(boxname, prec, kind):
    import oracle
    import torch
    from paper_2510_06873_b200.metad import MetaD
    boxes = {
        "cubic3cells": (np.array([10.0, 0, 0, 0, 10.0, 0, 0, 0, 10.0]), 3.2),
        # exactly 3 x 3 x 3 cells with more than 1,024 atoms: the cell-list kernels (not the brute-force one-launch build),
        # every neighbouring cell reached through a wrap in some direction (per-run lattice shifts of the fp64 build)
        "cubic3dense": (np.array([12.6, 0, 0, 0, 12.6, 0, 0, 0, 12.6]), 3.9, 0.55),
        "two_cells": (np.array([9.0, 0, 0, 0, 11.0, 0, 0, 0, 30.0]), 4.4),      # 2 x 2 x 6 cells
        "hex120": (np.array([24.0, 0, 0, -12.0, 12.0 * np.sqrt(3.0), 0, 0, 0, 19.0]), 4.0),
        "hex60": (np.array([24.0, 0, 0, 12.0, 12.0 * np.sqrt(3.0), 0, 0, 0, 19.0]), 4.0),
        "triclinic": (np.array([21.0, 0, 0, 5.0, 20.0, 0, -4.5, 7.0, 23.0]), 3.5),
    }
    box, rc = boxes[boxname][:2]
    density = boxes[boxname][2] if len(boxes[boxname]) > 2 else 0.15
    rng = np.random.default_rng(17)
    vol = box[0] * box[4] * box[8]
    n = max(int(density * vol), 64)
    pos = wrap(rng.random((n, 3)) @ box.reshape(3, 3), box)
    # plant borderline pairs: partner at distance rc*(1 +- tiny) so that the fp32 guard band is exercised
    for k in range(0, 2 * (n // 8), 2):
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        pos[k + 1] = pos[k] + u * rc * (1.0 + (rng.random() - 0.5) * 4e-7)
    pos = wrap(pos, box)
    w = Workload(name=boxname, pos=pos, box=box, rc=rc, max_neigh=200, cvs=[CVSpec(kind=kind, r0=1.0, scale=1.0)],
                 sigma=[0.1], n_hills=4, precision=prec)
    p = positions_for(w, prec)
    cref, lref, mx = oracle.neighbors(p.astype(np.float64), box, rc, 200, "brute")
    assert mx <= 200
    md = MetaD(w, precision=prec)
    dpos = torch.tensor(p, device="cuda")
    torch.cuda.synchronize()
    md.build_neighbors(dpos)
    cnt, lst = md.neighbors()
    assert md.status() == 0
    assert np.array_equal(cnt, cref)
    assert np.array_equal(sorted_rows_fast(cnt, lst), sorted_rows_fast(cref, lref))


def test_deposition_replay_matches_oracle_heights():
    """Reading K pin on the GPU side: replaying a scripted centre path through metad_bias +
    metad_deposit reproduces the oracle's well-tempered heights to 1e-9 relative."""
    import torch
    from oracle.reference import replay_heights
    from paper_2510_06873_b200.metad import MetaD
    w = _small("c1")
    w.stride = 1
    H = 300
    centers = hill_walk(3, [8.0, 0.9], w.sigma, H, step_frac=0.3)
    href = replay_heights(centers, w.sigma, w.w0, w.kT, w.bias_factor)
    md = MetaD(w, max_hills=H + 4)
    with torch.cuda.stream(md.stream):
        dc = torch.tensor(centers, device="cuda")
    md.synchronize()
    for k in range(H):
        md.bias(cv=dc[k])
        md.deposit(cv=dc[k])
    c, h = md.get_hills()
    assert len(h) == H and np.array_equal(c, centers)
    assert rel(h, href) <= 1e-9
    assert md.state()["step"] == H


def test_graph_run_end_to_end_and_determinism():
    """metad_run (CUDA graph, deposition every `stride` steps) against the oracle's step loop (gpu_util.chained_run: every
    step stage-wise on the library's own values + the free-running loop with the derived force bound, reading S), and
    bit-identical results when the whole loop is repeated in one call (reading P)."""
    import torch
    from paper_2510_06873_b200.metad import MetaD
    w = _small("c3")
    w.stride = 2
    nsteps = 7
    ref = chained_run(w, nsteps=nsteps)
    results = []
    for rep in range(2):
        md = MetaD(w, max_hills=64)
        md.set_hills(*ref["hills0"])
        with torch.cuda.stream(md.stream):
            dpos = torch.tensor(w.pos, device="cuda")
            F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float64)
        md.synchronize()
        md.run(dpos, F, nsteps)
        st = md.state()
        c, h = md.get_hills()
        results.append((F.cpu().numpy(), st, c, h))
        assert md.status() == 0
    F, st, c, h = results[0]
    assert st["step"] == nsteps and st["nhills"] == 40 + nsteps // 2
    # one call of n steps == n calls of one step (same graph): hills and state bit for bit, forces up to the order of the
    # per-step additions into F
    last = ref["states"][-1]
    assert np.array_equal(st["cv"], last["cv"]) and st["V"] == last["V"]
    assert np.array_equal(h, ref["md"].get_hills()[1])
    assert np.abs(F - ref["F"]).max() <= 1e-13 * np.abs(F).max()
    # determinism
    assert np.array_equal(results[0][0], results[1][0])
    assert np.array_equal(results[0][3], results[1][3])
    assert results[0][1]["V"] == results[1][1]["V"]


def test_ten_fixed_position_steps_are_bit_identical_config0():
    """BASELINE.json configs[0]: evaluate V, dV/ds and forces for 10 steps with fixed positions."""
    import torch
    from paper_2510_06873_b200.metad import MetaD
    w = configs.config0(shifted=True)
    md = MetaD(w)
    md.set_hills(w.hill_centers, w.hill_heights)
    dpos = torch.tensor(w.pos, device="cuda")
    torch.cuda.synchronize()
    outs = []
    for _ in range(10):
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float64)
        torch.cuda.synchronize()
        md.run(dpos, F, 1)
        st = md.state()
        outs.append((st["cv"].copy(), st["V"], st["dVds"].copy(), F.cpu().numpy()))
    for k in range(1, 10):
        assert np.array_equal(outs[k][0], outs[0][0]) and outs[k][1] == outs[0][1]
        assert np.array_equal(outs[k][2], outs[0][2]) and np.array_equal(outs[k][3], outs[0][3])
    assert md.state()["nhills"] == 200          # stride 0: nothing deposited


def test_grid_bias_matches_oracle_grid():
    """Reading M: the grid path is compared with the ORACLE'S grid path (same nodes, same interpolant)."""
    import torch
    from oracle.reference import OracleMetaD
    from paper_2510_06873_b200.metad import MetaD
    w = _small("c4")
    pos = positions_for(w, 32)
    o = OracleMetaD(w)
    o.build_neighbors(pos.astype(np.float64))
    s_ref = o.eval_cv(want_grad=False)
    sig = np.asarray(w.sigma)
    centers, heights = make_hills(w, s_ref)
    lo, hi = s_ref - 40 * sig, s_ref + 40 * sig
    o.enable_grid(w.grid_n, lo, hi)
    o.set_hills(centers, heights)
    md = MetaD(w, precision=32, grid=(w.grid_n, lo, hi), max_hills=len(heights) + 8)
    md.set_hills(centers, heights)
    tab = md.grid_table()
    scale = np.abs(o.grid["table"]).reshape(4, -1).max(1)[:, None, None]
    assert np.abs(tab - o.grid["table"]).max() / 1.0 <= 1e-9 * scale.max()
    assert (np.abs(tab - o.grid["table"]) / scale).max() <= 1e-10
    rng = np.random.default_rng(0)
    for k in range(20):
        s = s_ref + (rng.random(2) - 0.5) * 20 * sig
        V_ref, dV_ref = o.bias(s)
        with torch.cuda.stream(md.stream):
            ds = torch.tensor(s, device="cuda")
        V, dV = md.bias(cv=ds)
        md.synchronize()
        assert rel(V.cpu().numpy(), V_ref) <= TOL_CV
        assert np.abs(dV.cpu().numpy() - dV_ref).max() <= TOL_CV * np.abs(dV_ref).max() + 1e-300
    assert md.status() == 0
    # outside the table: exact sum + sticky bit
    s = s_ref + np.array([50.0, 0.0]) * sig
    with torch.cuda.stream(md.stream):
        ds = torch.tensor(s, device="cuda")
    V, dV = md.bias(cv=ds)
    md.synchronize()
    V_ref, dV_ref = o.bias(s, use_grid=False)
    assert rel(V.cpu().numpy(), V_ref) <= TOL_CV
    assert md.status() & 4
    # deposition adds the new hill to the table
    w2 = _small("c4")
    w2.stride = 1
    o2 = OracleMetaD(w2)
    o2.enable_grid(w2.grid_n, lo, hi)
    o2.set_hills(centers, heights)
    md2 = MetaD(w2, precision=32, grid=(w2.grid_n, lo, hi), max_hills=len(heights) + 8)
    md2.set_hills(centers, heights)
    s = s_ref + np.array([0.4, -0.7]) * sig
    V0, _ = o2.bias(s)
    o2.deposit(s, V0)
    with torch.cuda.stream(md2.stream):
        ds = torch.tensor(s, device="cuda")
    md2.bias(cv=ds)
    md2.deposit(cv=ds)
    tab2 = md2.grid_table()
    assert (np.abs(tab2 - o2.grid["table"]) / scale).max() <= 1e-10
    c, h = md2.get_hills()
    assert rel(h[-1], o2.heights[-1]) <= 1e-9


def test_step_host_round_trip():
    import torch
    from paper_2510_06873_b200.metad import MetaD
    w = _small("c2")
    r = stagewise(w)
    md = MetaD(w, max_hills=len(r["heights"]) + 8)
    md.set_hills(r["centers"], r["heights"])
    pos_h = torch.tensor(w.pos).pin_memory()
    F_h = torch.ones((w.natoms, 3), dtype=torch.float64).pin_memory()
    cv, V = md.step_host(pos_h, F_h)
    assert rel(cv, r["s_ref"]) <= TOL_CV
    dV_ref = r["o"].bias(r["s_ref"], use_grid=False)[1]
    Fb = r["o"].forces(dV_ref)
    # the two sides used their own dV/ds: derived end-to-end bound (reading S), no slack factor
    assert np.abs(F_h.numpy() - 1.0 - Fb).max() <= force_bound(Fb, md.state()["dVds"], dV_ref, r["o"].grads) + 1e-15


def test_step_host_with_the_library_page_locked_buffers():
    """metad_host_alloc / metad_host_free through the binding: same numbers as with any other host pointer."""
    import gc
    from paper_2510_06873_b200.metad import MetaD, MetadError, load, pinned_array
    import ctypes
    w = _small("c2")
    r = stagewise(w)
    md = MetaD(w, max_hills=len(r["heights"]) + 8)
    md.set_hills(r["centers"], r["heights"])
    pos_h = pinned_array(w.pos.shape, np.float64)
    pos_h[...] = w.pos
    F_h = pinned_array((w.natoms, 3), np.float64)
    F_h[...] = 1.0
    cv, V = md.step_host(pos_h, F_h)
    assert rel(cv, r["s_ref"]) <= TOL_CV
    dV_ref = r["o"].bias(r["s_ref"], use_grid=False)[1]
    Fb = r["o"].forces(dV_ref)
    assert np.abs(F_h - 1.0 - Fb).max() <= force_bound(Fb, md.state()["dVds"], dV_ref, r["o"].grads) + 1e-15
    del pos_h, F_h
    gc.collect()
    p = ctypes.c_void_p()
    assert load().metad_host_alloc(ctypes.byref(p), 0) != 0          # zero size is an argument error
    assert load().metad_host_alloc(None, 16) != 0
    assert load().metad_host_free(None) == 0


def test_errors_and_sticky_bits():
    import torch
    from paper_2510_06873_b200 import metad
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = configs.config0()
    md = MetaD(w)
    dpos = torch.tensor(w.pos, device="cuda")
    torch.cuda.synchronize()
    with pytest.raises(MetadError) as e:
        md.build_neighbors(dpos, rc=10.0)                     # rc == half the box
    assert e.value.code == metad.ERR_BOX
    with pytest.raises(MetadError) as e:
        md.build_neighbors(dpos, box=np.array([20.0, 1, 0, 0, 20, 0, 0, 0, 20]))
    assert e.value.code == metad.ERR_BOX
    md2 = MetaD(w)
    with pytest.raises(MetadError) as e:
        md2.eval_cv()                                         # no neighbour list yet
    assert e.value.code == metad.ERR_STATE
    # neighbour overflow: capacity 16 < ~56 neighbours -> sticky bit, counts clipped
    w.max_neigh = 16
    md3 = MetaD(w)
    md3.build_neighbors(dpos)
    cnt, lst = md3.neighbors()
    assert md3.status() & metad.DEV_NEIGH_OVERFLOW and cnt.max() == 16
    # hill overflow
    w4 = configs.config0()
    w4.stride = 1
    md4 = MetaD(w4, max_hills=3)
    F = torch.zeros((w4.natoms, 3), device="cuda", dtype=torch.float64)
    torch.cuda.synchronize()
    md4.run(dpos, F, 5)
    assert md4.status() & metad.DEV_HILL_OVERFLOW and md4.state()["nhills"] == 3
    # a position outside the primary cell, and a NaN position: POS_RANGE sticky bit, no crash
    for bad in (np.array([25.0, 1.0, 1.0]), np.array([np.nan, 1.0, 1.0])):
        p = w4.pos.copy(); p[7] = bad
        md6 = MetaD(configs.config0())
        md6.build_neighbors(torch.tensor(p, device="cuda"))
        assert md6.status() & metad.DEV_POS_RANGE
    # empty hill set: V = 0, forces untouched
    md5 = MetaD(configs.config0())
    md5.run(dpos, F.zero_(), 1)
    st = md5.state()
    assert st["V"] == 0.0 and float(F.abs().max().cpu()) == 0.0


def test_positions_that_round_onto_the_far_box_face_fp32_tiled():
    """Regression (found at 4.096 M atoms): a coordinate in [0, L) can round to fractional 1.0 in fp32.  Such atoms are
    clamped into the boundary cell; neighbour sets must still be bit-exact on the tiled path."""
    import oracle
    import torch
    from paper_2510_06873_b200.metad import MetaD
    w = _small("c3")
    B = w.box.reshape(3, 3)
    rng = np.random.default_rng(3)
    pos = w.pos.copy()
    idx = rng.choice(w.natoms, 60, replace=False)
    frac = np.linalg.solve(B.T, pos[idx].T).T
    for k, i in enumerate(idx):
        frac[k, k % 3] = 1.0 - 1e-10          # wrapped in fp64, == 1.0 (or just above) after fp32 rounding
    pos[idx] = frac @ B
    p32 = pos.astype(np.float32)
    cref, lref, mx = oracle.neighbors(p32.astype(np.float64), w.box, w.rc, w.max_neigh, "brute")
    assert mx <= w.max_neigh
    md = MetaD(w, precision=32)
    dpos = torch.tensor(p32, device="cuda")
    torch.cuda.synchronize()
    md.build_neighbors(dpos)
    cnt, lst = md.neighbors()
    assert md.status() == 0
    assert np.array_equal(cnt, cref)
    assert np.array_equal(sorted_rows_fast(cnt, lst), sorted_rows_fast(cref, lref))
    md.eval_cv()
    md.synchronize()
    q_ref = oracle.q6_atoms(p32.astype(np.float64), w.box, cref, lref)
    assert np.abs(md.q6() - q_ref).max() <= 5e-6


@pytest.mark.parametrize("precision", [64, 32])
def test_isolated_atoms_and_empty_cells(precision):
    """Degenerate cases of the Q6 path: atoms with no neighbour at all (q6 = 0, zero gradient, reading E), atoms with a single
    neighbour (q6 = 1), and a box that is mostly vacuum (empty cells, empty tiles) — generic fp64 and tiled fp32 paths."""
    from paper_2510_06873_b200.inputs import CV_Q6_MEAN
    rng = np.random.default_rng(21)
    L = 64.0
    box = np.array([L, 0, 0, 0, L, 0, 0, 0, L], dtype=np.float64)
    blob = 8.0 + rng.random((1500, 3)) * 18.0                       # dense-ish droplet in one corner: ~0.26 atoms / A^3 -> thin it
    keep = [0]
    for i in range(1, len(blob)):                                    # minimum separation 2.0 A
        if np.min(np.linalg.norm(blob[keep] - blob[i], axis=1)) > 2.0:
            keep.append(i)
    blob = blob[keep]
    lone = np.array([[50.0, 50.0, 50.0], [40.0, 10.0, 55.0], [5.0, 60.0, 33.0]])          # no neighbour within rc
    pair = np.array([[52.0, 20.0, 20.0], [52.0, 20.0, 22.5]])                              # one neighbour each
    pos = np.concatenate([blob, lone, pair])
    w = Workload(name="iso", pos=pos, box=box, rc=3.6, max_neigh=32,
                 cvs=[CVSpec(kind=CV_Q6_MEAN, scale=1.0 / len(pos))], sigma=[0.01], n_hills=50, precision=precision)
    r = stagewise(w, precision=precision)
    assert_stagewise(r)
    nb = len(blob)
    assert np.all(r["cnt"][nb:nb + 3] == 0) and np.all(r["cnt"][nb + 3:] == 1)
    assert np.all(r["q6"][nb:nb + 3] == 0.0) and np.allclose(r["q6"][nb + 3:], 1.0, atol=2e-6)
    assert np.all(r["F"][nb:nb + 3] == 0.0) and np.all(np.isfinite(r["F"]))


def test_fp32_borderline_pairs_across_the_faces_of_a_large_box():
    """The fp64 recheck band of the generic fp32 build is derived from the box (neighbor.cu: make_pbox): in a 640 A cell the raw
    difference of two fp32 coordinates on opposite faces is rounded at ulp(640) = 6e-5 A, far more than the 1e-5 rc^2 band
    resolves for rc = 3.2 A.  Planted pairs at rc (1 +- 2e-7) straddling every face must come out exactly as the fp64
    definition decides (reading O), on the generic (max_neigh > 32) and on the tiled path."""
    import oracle
    import torch
    from paper_2510_06873_b200.metad import MetaD
    Lb, rc = 640.0, 3.2
    box = np.array([Lb, 0, 0, 0, Lb, 0, 0, 0, Lb])
    rng = np.random.default_rng(23)
    n = 24000
    pos = rng.random((n, 3)) * Lb
    npl = 4000
    for k in range(0, 2 * npl, 2):
        face = (k // 2) % 3
        pos[k, face] = rng.random() * 0.5 * rc                                   # next to the low face
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        u[face] = -abs(u[face]) - 0.2                                            # partner across that face
        u /= np.linalg.norm(u)
        pos[k + 1] = pos[k] + u * rc * (1.0 + (rng.random() - 0.5) * 4e-7)
    pos = wrap(pos, box)
    for maxn, kind in ((40, 0), (32, 1)):                                        # generic coordination build, tiled Q6 build
        w = Workload(name="bigbox", pos=pos, box=box, rc=rc, max_neigh=maxn, cvs=[CVSpec(kind=kind, r0=1.0, scale=1.0)],
                     sigma=[0.1], n_hills=4, precision=32)
        p = positions_for(w, 32)
        cref, lref, mx = oracle.neighbors(p.astype(np.float64), box, rc, maxn, "cells")
        assert mx <= maxn and cref.sum() > npl
        md = MetaD(w, precision=32)
        dpos = torch.tensor(p, device="cuda")
        torch.cuda.synchronize()
        md.build_neighbors(dpos)
        cnt, lst = md.neighbors()
        assert md.status() == 0
        assert np.array_equal(cnt, cref)
        assert np.array_equal(sorted_rows_fast(cnt, lst), sorted_rows_fast(cref, lref))


@pytest.mark.parametrize("precision", [64, 32])
def test_several_list_cvs_in_one_context(precision):
    """Two coordination numbers with different groups, exponents and r0, an ungrouped one, and a nearest-distance CV in ONE
    context (each list CV owns two bits of the per-atom group flags): every CV, V, dV/ds, the forces and the bias virial against
    the oracle, stage-wise."""
    from paper_2510_06873_b200.inputs import CV_COORD, CV_MINDIST
    w = _small("c2")
    cv = w.cvs[0]
    A, B = np.asarray(cv.group_a), np.asarray(cv.group_b)
    w.cvs = [CVSpec(kind=CV_COORD, r0=1.2, n=6, m=12, scale=1.0, group_a=A, group_b=B),
             CVSpec(kind=CV_COORD, r0=1.6, n=8, m=16, scale=1.0 / len(B), group_a=B[::2], group_b=B[1::2]),
             CVSpec(kind=CV_MINDIST, group_a=A[11:12], group_b=B),
             CVSpec(kind=CV_COORD, r0=2.0, n=6, m=10, scale=1.0 / w.natoms)]
    w.sigma = [0.5, 0.05, 0.05, 0.02]
    w.n_hills = 120
    r = stagewise(w, precision=precision, want_virial=True)
    assert_stagewise(r)
    assert np.all(np.abs(r["dV_ref"]) > 0)
    W, W_ref = r["md"].virial(), r["o"].virial(r["dV_ref"])
    assert np.abs(W - W_ref).max() <= (1e-9 if precision == 64 else 1e-5) * np.abs(W_ref).max()
    # and through the run path with a skin (every list CV filters the kept list on its own)
    w.stride = 2
    frames = [wrap(w.pos + np.random.default_rng(3 + k).standard_normal(w.pos.shape) * 0.01 * k, w.box) for k in range(5)]
    w.max_neigh = 96
    rr = chained_run(w, precision=precision, nsteps=5, skin=0.3, check_neighbors=True, pos_of_step=lambda k: frames[k])
    assert rr["md"].rebuilds() < 5
